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

// One Cartesian component c (0,1,2) of the normals of (atom, mode, tag, step).
__device__ __forceinline__ double qhp_normal_comp(uint64_t seed, uint32_t atom, uint32_t mode,
                                                  uint32_t tag, uint64_t step, int c) {
  uint32_t w[4];
  qhp_philox4x32_10(atom, mode | (tag << 24), (uint32_t)step, (uint32_t)(step >> 32),
                    (uint32_t)seed, (uint32_t)(seed >> 32), w);
  const uint32_t wa = (c == 2) ? w[2] : w[0];
  const uint32_t wb = (c == 2) ? w[3] : w[1];
  const double r = sqrt(-2.0 * log(qhp_u01(wa)));
  // sin(2 pi u) = cos(pi (2u - 1/2)); 2u - 1/2 is exact
  const double arg = 2.0 * qhp_u01(wb) - ((c == 1) ? 0.5 : 0.0);
  return r * cospi(arg);
}

// All three components.
__device__ __forceinline__ void qhp_normals3(uint64_t seed, uint32_t atom, uint32_t mode,
                                             uint32_t tag, uint64_t step, double z[3]) {
  uint32_t w[4];
  qhp_philox4x32_10(atom, mode | (tag << 24), (uint32_t)step, (uint32_t)(step >> 32),
                    (uint32_t)seed, (uint32_t)(seed >> 32), w);
  const double r0 = sqrt(-2.0 * log(qhp_u01(w[0])));
  const double r1 = sqrt(-2.0 * log(qhp_u01(w[2])));
  double sn, cs;
  sincospi(2.0 * qhp_u01(w[1]), &sn, &cs);
  z[0] = r0 * cs;
  z[1] = r0 * sn;
  z[2] = r1 * cospi(2.0 * qhp_u01(w[3]));
}
