// philox.cuh -- Philox4x32-10 counter-based generator (Salmon, Moraes, Dror, Shaw, SC'11) and the
// Box-Muller normals of the PILE (Eq. 16) and QTB white-noise
// streams.  Stream contract:
//   key = (seed_lo, seed_hi); counter = (atom, mode | tag<<24, step_lo, step_hi);
//   u_k = (w_k + 0.5) 2^-32;  z_x, z_y = sqrt(-2 ln u_0) (cos, sin)(2 pi u_1);  z_z = sqrt(-2 ln u_2) cos(2 pi u_3).
// The trigonometric argument 2 u is exact in fp64, so cospi/sinpi need no range reduction.
#pragma once
#include <stdint.h>

__device__ __forceinline__ void qhp_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                  uint32_t k0, uint32_t k1, uint32_t w[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

__device__ __forceinline__ double qhp_u01(uint32_t w) {
  return ((double)w + 0.5) * (1.0 / 4294967296.0);
}

// ---- Box-Muller pieces written for their actual arguments (round 2: one Philox + Box-Muller call cost 413
//      instructions with the general-purpose libdevice log / sqrt / sincospi, 36 % of the fused integrator pass and
//      46 % of the noise kernel).  u = (w + 1/2) 2^-32 = t 2^-33 with t = 2 w + 1 an odd 33-bit integer: no zero, no
//      denormal, no special value, and the trigonometric argument 2 u is an exact binary fraction.  Each piece is
//      accurate to ~1 ulp (Taylor series with truncation below 2^-54 relative; tests/test_gpu_primitives.py bounds
//      the normals against the oracle's libm values). ----
// sqrt(-2 ln u)
__device__ __forceinline__ double qhp_bm_radius(uint32_t w) {
  const unsigned long long t = 2ull * w + 1ull;
  const int lz = __clzll((long long)t);                       // 31 .. 63
  int e = 30 - lz;                                            // floor(log2 t) - 33, in [-33, -1]
  const unsigned long long mant = (t << (lz + 1)) >> 12;      // the 52 bits behind the leading one
  double m = __longlong_as_double((long long)(0x3ff0000000000000ull | mant));   // [1, 2)
  if (m > 1.4142135623730951) { m *= 0.5; e += 1; }           // [sqrt(1/2), sqrt(2)]
  const double f = m - 1.0, d = 2.0 + f;                      // exact
  // s = f / d by a seeded reciprocal (d in [1.7, 2.42])
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  y = fma(fma(-d, y, 1.0), y, y);
  y = fma(fma(-d, y, 1.0), y, y);
  double sq = f * y;
  sq = fma(fma(-d, sq, f), y, sq);
  // ln m = 2 atanh(sq) = 2 sq (1 + z/3 + z^2/5 + ...), z = sq^2 <= 0.0295: 12 terms leave 0.0295^12 / 25 < 2e-20
  const double z = sq * sq;
  double p = 1.0 / 25.0;
  p = fma(p, z, 1.0 / 23.0); p = fma(p, z, 1.0 / 21.0); p = fma(p, z, 1.0 / 19.0); p = fma(p, z, 1.0 / 17.0);
  p = fma(p, z, 1.0 / 15.0); p = fma(p, z, 1.0 / 13.0); p = fma(p, z, 1.0 / 11.0); p = fma(p, z, 1.0 / 9.0);
  p = fma(p, z, 1.0 / 7.0); p = fma(p, z, 1.0 / 5.0); p = fma(p, z, 1.0 / 3.0);
  const double lnm = fma(sq * z, p, sq);                      // atanh(sq) = ln(m) / 2
  // x = -2 ln u = e (-2 ln 2) - 4 atanh(sq), -2 ln 2 = hi + lo split so that e * hi is exact
  const double ed = (double)e;
  const double x = fma(-4.0, lnm, ed * -3.8164298585411754e-10) + ed * -1.3862943607382476;   // e * hi is exact (hi: 32 significant bits)
  // sqrt(x), x in (2.3e-10, 46]: seeded reciprocal square root + one correction of the product
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double h = fma(-x * r, r, 1.0);
  r = fma(r * h, fma(0.375, h, 0.5), r);                      // 1/sqrt(x) to ~1 ulp
  double sr = x * r;
  sr = fma(fma(-sr, sr, x), 0.5 * r, sr);
  return sr;
}

// cos(pi a) and sin(pi a) for a = 2 u = t 2^-32 in (0, 2): quadrant and remainder by integer arithmetic (exact),
// Taylor polynomials on |r| <= 1/4
__device__ __forceinline__ void qhp_bm_sincos(uint32_t w, double *sn, double *cs) {
  const long long t = 2ll * (long long)w + 1ll;
  const int q = (int)((t + (1ll << 30)) >> 31);               // round(2 a), 0 .. 4
  const int di = (int)(t - ((long long)q << 31));             // |di| <= 2^30
  const double r = (double)di * (1.0 / 4294967296.0);         // a - q/2, exact
  const double z = r * r;
  double S = -2.1915353447830215827e-5;
  S = fma(S, z, 4.6630280576761256442e-4); S = fma(S, z, -7.3704309457143507773e-3); S = fma(S, z, 8.2145886611128228799e-2);
  S = fma(S, z, -5.9926452932079207689e-1); S = fma(S, z, 2.5501640398773454439); S = fma(S, z, -5.1677127800499700292);
  S = fma(S, z, 3.1415926535897932385);
  S *= r;
  double Cc = 4.3030695870329470073e-6;
  Cc = fma(Cc, z, -1.0463810492484570712e-4); Cc = fma(Cc, z, 1.9295743094039230479e-3); Cc = fma(Cc, z, -2.5806891390014060013e-2);
  Cc = fma(Cc, z, 2.3533063035889320454e-1); Cc = fma(Cc, z, -1.3352627688545894959); Cc = fma(Cc, z, 4.0587121264167682182);
  Cc = fma(Cc, z, -4.9348022005446793094);
  Cc = fma(Cc, z, 1.0);
  // angle = pi (q/2 + r)
  const double s0 = (q & 1) ? Cc : S, c0 = (q & 1) ? S : Cc;
  *sn = (q & 2) ? -s0 : s0;
  *cs = ((q + 1) & 2) ? -c0 : c0;
}

// One Cartesian component c (0,1,2) of the normals of (atom, mode, tag, step).
__device__ __forceinline__ double qhp_normal_comp(uint64_t seed, uint32_t atom, uint32_t mode,
                                                  uint32_t tag, uint64_t step, int c) {
  uint32_t w[4];
  qhp_philox4x32_10(atom, mode | (tag << 24), (uint32_t)step, (uint32_t)(step >> 32),
                    (uint32_t)seed, (uint32_t)(seed >> 32), w);
  const uint32_t wa = (c == 2) ? w[2] : w[0];
  const uint32_t wb = (c == 2) ? w[3] : w[1];
  double sn, cs;
  qhp_bm_sincos(wb, &sn, &cs);
  return qhp_bm_radius(wa) * ((c == 1) ? sn : cs);
}

// All three components.
__device__ __forceinline__ void qhp_normals3(uint64_t seed, uint32_t atom, uint32_t mode,
                                             uint32_t tag, uint64_t step, double z[3]) {
  uint32_t w[4];
  qhp_philox4x32_10(atom, mode | (tag << 24), (uint32_t)step, (uint32_t)(step >> 32),
                    (uint32_t)seed, (uint32_t)(seed >> 32), w);
  const double r0 = qhp_bm_radius(w[0]), r1 = qhp_bm_radius(w[2]);
  double sn, cs, sn1, cs1;
  qhp_bm_sincos(w[1], &sn, &cs);
  qhp_bm_sincos(w[3], &sn1, &cs1);
  z[0] = r0 * cs;
  z[1] = r0 * sn;
  z[2] = r1 * cs1;
}
