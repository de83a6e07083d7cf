// pair_staged.cu -- bead-batched short-range pair forces V_s on the contracted beads, shared-memory
// staged version ("the most time-consuming operation";
// contraction PAPER.md:174-182 Eq. 20; lists on the centroids shared by all beads).
//
// Why: a warp-per-atom walk over a Verlet list gathers one 32-byte position per candidate pair;
// through L1 that costs one wavefront per lane (32 distinct lines per load instruction) and was
// the limiter of the first kernel (k_pair, pair.cu), not the FP64 pipe.  Here one CTA owns one
// (cell, contracted bead): it stages the positions of the cell's 27-cell neighbourhood once in
// shared memory, in coordinates relative to the cell centre (so the minimum image is applied per
// staged atom, not per pair), and the neighbour table holds 16-bit indices into that staged array.
//
// Per atom i (one warp); a list entry = staged index | atom type << 13:
//   check   32 list entries at a time: packed-half distance test on an 8-byte fp16 copy (conservative margin,
//           it only rejects pairs that are certainly outside r_c), ballot compaction of the
//           survivors into a per-warp queue; the record of the next step is requested one step ahead;
//   eval    whenever the queue holds >= 32 survivors: all 32 lanes evaluate one pair each in fp64
//           (exact r^2 < r_c^2 test, LJ + damped-shifted-force Coulomb); no lane idles on the
//           cutoff, which cost 41 % of the lanes before.
// Shared memory is addressed through 32-bit shared addresses (inline PTX ld/st.shared): no generic
// pointers, no 64-bit address arithmetic in the inner loops.
// The DSF radial function needs no erfc/exp: with w = (alpha r)^2,
//   erfc(x) + (2x/sqrt(pi)) e^{-x^2} = 1 - x^3 S(w),   erfc(x)/x = 1/x - E(w),
// S and E entire in w, so F/r = qq (1/r^3 - alpha^3 S(w) - fshift/r) with 1/r from one rsqrt and
// alpha^3 S a degree-15 polynomial in u = 2 r^2/r_c^2 - 1 whose coefficients (fitted at create time
// from the Taylor series of S, qhp_pair_setup) sit in the kernel's constant bank.
// Full list (each ordered pair evaluated from its own side): no atomics, fixed summation order.
#include <math.h>
#include <cuda_fp16.h>

#include "qhp_internal.cuh"

#ifndef STG_THREADS
#define STG_THREADS 768           // largest CTA (24 warps, <= 85 registers); the host launches fewer warps when shared memory is short
#endif
#define STG_MAX_WARPS (STG_THREADS / 32)
#define STG_BLOCK 256             // list entries per row block (8 per lane)
#define STG_QUEUE (STG_BLOCK + 32)   // <= 31 left over + 256
#define STG_IDX_BITS 13           // list entry = staged index | atom type << 13 (QHP_MAX_TYPES = 8)
#define STG_IDX_MASK 0x1fffu

struct StagedArgs {
  int N, Pc, nt, split, cap;     // cap - 1 = dummy staged atom (infinitely far): target of the row padding
  int bead0;                     // first contracted bead of this launch (grid.y beads from here: bead slices, qhp_set_comm)
  int nc[3];
  double box[3], inv_box[3], cell_edge[3];
  const double *pos4;            // [Pc][N] (x, y, z, type bits), slot order
  double *Fs;                    // [Pc][N][3]
  const uint16_t *nbr16;         // [N][stride] entries (blocked, see below), rows padded to a multiple of 32 with the dummy
  const int32_t *nbr_count, *cell_start;
  long long stride;
  const double *pair_tab;        // [nt*nt][4] = qq, 4 eps, sigma^2, LJ shift
  double qs[QHP_MAX_TYPES];      // sqrt(Coulomb constant) * charge per type: qq = qs_i * qs_j
  unsigned lj_mask[QHP_MAX_TYPES]; // bit tj: types (ti, tj) have a Lennard-Jones term
  double rc, rc2, u_scale, fshift, erfc_rc;
  unsigned rc2h;                 // fp16 pre-test threshold (r_c^2 + error bound, rounded up), both halves of a half2
  double cS[QHP_NPOLY], cE[QHP_NPOLY];
  double *part;                  // ENERGY: per-CTA partial sums of U_s
  unsigned long long *count;     // ENERGY: in-cutoff pair-bead counter
  long long *counters;           // [7] = staged-region overflow flag
};

// 1/sqrt(s): hardware seed (upper-word approximation, ~2^-20) + one third-order step -> ~1 ulp
__device__ __forceinline__ double rsqrt_seeded(double s) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
  const double e = fma(-s * y, y, 1.0);
  return fma(y * e, fma(0.375, e, 0.5), y);
}

// even/odd split Horner (two independent chains)
__device__ __forceinline__ double poly_eval(const double *c, double u) {
  static_assert(QHP_NPOLY % 2 == 0, "even/odd split");
  const double v = u * u;
  double a = c[QHP_NPOLY - 2], b = c[QHP_NPOLY - 1];
#pragma unroll
  for (int k = QHP_NPOLY - 4; k >= 0; k -= 2) { a = fma(a, v, c[k]); b = fma(b, v, c[k + 1]); }
  return fma(b, u, a);
}

// shared-memory accesses through 32-bit shared addresses (no generic pointers, no 64-bit address arithmetic)
__device__ __forceinline__ uint2 lds_u2(uint32_t a) { uint2 v; asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v; }
__device__ __forceinline__ double2 lds_d2(uint32_t a) { double2 v; asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a)); return v; }
__device__ __forceinline__ double lds_d(uint32_t a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds_u(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts_u(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }

// fp16 pre-test record of a staged atom: (x, y) and (z, 0) as two half2 words, round to nearest
__device__ __forceinline__ uint2 half_record(double x, double y, double z) {
  const __half2 xy = __floats2half2_rn((float)x, (float)y), zw = __floats2half2_rn((float)z, 0.f);
  return make_uint2(*reinterpret_cast<const unsigned *>(&xy), *reinterpret_cast<const unsigned *>(&zw));
}
// packed-half squared distance of two records against the threshold (qhp_pair_staged_forces derives the error bound
// that makes this test conservative: it never rejects a pair whose fp64 r^2 is below r_c^2)
__device__ __forceinline__ bool half_test(uint2 ci, uint2 cj, unsigned thr) {
  const __half2 dxy = __hsub2(*reinterpret_cast<const __half2 *>(&ci.x), *reinterpret_cast<const __half2 *>(&cj.x));
  const __half2 dzw = __hsub2(*reinterpret_cast<const __half2 *>(&ci.y), *reinterpret_cast<const __half2 *>(&cj.y));
  const __half2 s = __hfma2(dzw, dzw, __hmul2(dxy, dxy));              // (dx^2 + dz^2, dy^2)
  return __hlt(__hadd(__low2half(s), __high2half(s)), __low2half(*reinterpret_cast<const __half2 *>(&thr)));
}

// Row layout of the 16-bit table (written by k_list_build16, cells.cu): the entry of rank `pos` in a
// row sits at (pos / 256) * 256 + (pos % 32) * 8 + (pos % 256) / 32, i.e. one 16-byte load per lane
// brings entries pos = 256 m + 32 j + lane, j = 0..7; a row is padded with the dummy index up to a
// multiple of 32 entries, so a check step never needs a per-lane tail predicate.
// Shared memory: XY[cap] (x, y) and Z[cap] fp64, cell-centred; F32: C[cap] 8-byte fp16 copy (x, y | z, 0)
// for the packed-half pre-test.  !F32 (neighbourhoods too large for 32 B per atom): 24 B per atom, fp64 pre-test.
template <bool ENERGY, bool F32>
__global__ void __launch_bounds__(STG_THREADS, 1) k_pair_staged(const StagedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2 *XY = reinterpret_cast<double2 *>(smem_raw);
  double *Z = reinterpret_cast<double *>(XY + a.cap);
  uint2 *C = reinterpret_cast<uint2 *>(Z + a.cap);
  double *tab = F32 ? reinterpret_cast<double *>(C + a.cap) : reinterpret_cast<double *>(Z + a.cap);
  double *qtab = tab + QHP_MAX_TYPES * QHP_MAX_TYPES * 4;             // sqrt(Coulomb constant) * charge per type
  uint32_t *queue = reinterpret_cast<uint32_t *>(qtab + QHP_MAX_TYPES);
  __shared__ int off[28], cbeg[27], next_atom;
  __shared__ double su[STG_MAX_WARPS];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x;
  const int cell = blockIdx.x / a.split, part = blockIdx.x % a.split, bead = a.bead0 + blockIdx.y;
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);

  for (int k = tid; k < a.nt * a.nt * 4; k += nthr) {      // (qq, 4 eps, sigma^2, shift) -> (24 eps, sigma^2, qq, shift)
    const int f = k & 3;
    tab[(k & ~3) + (f == 0 ? 2 : (f == 1 ? 0 : (f == 2 ? 1 : 3)))] = (f == 1 ? 6.0 : 1.0) * a.pair_tab[k];
  }
  if (tid < a.nt) qtab[tid] = a.qs[tid];
  if (tid < 27) {
    // same stencil order as the list build (cells.cu k_list_build16)
    const int ox = tid / 9, oy = (tid / 3) % 3, oz = tid % 3;
    const int qx = (cx - 1 + ox + a.nc[0]) % a.nc[0], qy = (cy - 1 + oy + a.nc[1]) % a.nc[1],
              qz = (cz - 1 + oz + a.nc[2]) % a.nc[2];
    const int c2 = (qx * a.nc[1] + qy) * a.nc[2] + qz;
    cbeg[tid] = a.cell_start[c2];
    off[tid + 1] = a.cell_start[c2 + 1] - a.cell_start[c2];
  }
  __syncthreads();
  if (tid == 0) {
    next_atom = 0;
    off[0] = 0;
    for (int s = 0; s < 27; ++s) off[s + 1] += off[s];
  }
  __syncthreads();
  const int total = off[27];
  if (off[14] == off[13]) return;            // empty home cell
  if (total > a.cap - 1) {                   // cannot happen after the host-side capacity check
    if (tid == 0) a.counters[7] = 1;
    return;
  }
  // ---- stage the neighbourhood in coordinates relative to the cell centre ------------------------
  const double4 *pos = reinterpret_cast<const double4 *>(a.pos4) + (long long)bead * a.N;
  {
    const double ctr[3] = {(cx + 0.5) * a.cell_edge[0], (cy + 0.5) * a.cell_edge[1], (cz + 0.5) * a.cell_edge[2]};
    const double MAGIC = 6755399441055744.0;             // 1.5 * 2^52: (t + MAGIC) - MAGIC = rint(t) for |t| < 2^51
    constexpr int UN = 4;                                // independent loads in flight per thread
    for (int g0 = tid; g0 < total; g0 += UN * nthr) {
      double4 p[UN];
      int s = 0;
#pragma unroll
      for (int u = 0; u < UN; ++u) {
        const int g = g0 + u * nthr;
        if (g < total) {
          while (g >= off[s + 1]) ++s;
          p[u] = pos[cbeg[s] + g - off[s]];
        }
      }
#pragma unroll
      for (int u = 0; u < UN; ++u) {
        const int g = g0 + u * nthr;
        if (g < total) {
          double lx = p[u].x - ctr[0], ly = p[u].y - ctr[1], lz = p[u].z - ctr[2];
          lx = fma(-a.box[0], (lx * a.inv_box[0] + MAGIC) - MAGIC, lx);
          ly = fma(-a.box[1], (ly * a.inv_box[1] + MAGIC) - MAGIC, ly);
          lz = fma(-a.box[2], (lz * a.inv_box[2] + MAGIC) - MAGIC, lz);
          XY[g] = make_double2(lx, ly); Z[g] = lz;
          if (F32) C[g] = half_record(lx, ly, lz);
        }
      }
    }
    if (tid == 0) {                                      // the dummy: every pre-test against it fails
      XY[a.cap - 1] = make_double2(1e9, 1e9); Z[a.cap - 1] = 1e9;
      if (F32) C[a.cap - 1] = half_record(1e9, 1e9, 1e9);     // +inf: inf - x = inf, inf - inf = NaN, neither is < the threshold
    }
  }
  __syncthreads();

  const int h0 = off[13], nh = off[14] - off[13], slot0 = cbeg[13];
  const uint32_t sXY = (uint32_t)__cvta_generic_to_shared(XY), sZ = (uint32_t)__cvta_generic_to_shared(Z),
                 sC = (uint32_t)__cvta_generic_to_shared(C), sTab = (uint32_t)__cvta_generic_to_shared(tab), sQt = (uint32_t)__cvta_generic_to_shared(qtab),
                 sQ = (uint32_t)__cvta_generic_to_shared(queue) + warp * (STG_QUEUE * 4);
  unsigned lt;
  asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt));   // volatile: kept in a register (ptxas re-derives (1 << lane) - 1 per use)
  double U = 0.0;
  unsigned long long hits = 0;

  // Atoms of the home cell are handed to the warps dynamically (the CTAs of one cell take the atoms
  // ii = part, part + split, ...); each atom is summed by one warp in a fixed order, so the result
  // does not depend on which warp took it.
  for (;;) {
    int t = 0;
    if (lane == 0) t = atomicAdd(&next_atom, 1);
    const int ii = part + a.split * __shfl_sync(0xffffffffu, t, 0);
    if (ii >= nh) break;
    const uint32_t ei = (uint32_t)(h0 + ii);
    const long long slot = slot0 + ii;
    const int n = a.nbr_count[slot];
    const uint16_t *rowp = a.nbr16 + slot * a.stride;
    const int nblk = (n + STG_BLOCK - 1) / STG_BLOCK;
    uint4 cur = make_uint4(0u, 0u, 0u, 0u);
    if (nblk > 0) cur = *reinterpret_cast<const uint4 *>(rowp + 8 * lane);
    const double2 xyi = lds_d2(sXY + ei * 16);
    const double zi = lds_d(sZ + ei * 8);
    uint2 ci = make_uint2(0u, 0u);
    if (F32) ci = lds_u2(sC + ei * 8);
    const int ti = (int)__double_as_longlong(pos[slot].w);
    const uint32_t sTi = sTab + (uint32_t)(ti * a.nt) * 32u;
    const double qi = lds_d(sQt + ti * 8);
    const unsigned lj_mask = a.lj_mask[ti];
    const bool lj_row = lj_mask != 0u;
    double Fx = 0.0, Fy = 0.0, Fz = 0.0;
    uint32_t qa = sQ;                                    // byte address of the queue end

    // one pair per lane, fp64: LJ + damped-shifted-force Coulomb (oracle O3); the fp64 test decides
    auto eval = [&](uint32_t entry, bool active) {
      const uint32_t sj = entry & STG_IDX_MASK, tj = entry >> STG_IDX_BITS;
      const double2 xyj = lds_d2(sXY + sj * 16);
      const double zj = lds_d(sZ + sj * 8);
      const double qq = qi * lds_d(sQt + tj * 8);
      const double dx = xyi.x - xyj.x, dy = xyi.y - xyj.y, dz = zi - zj;
      const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
      const bool in = active && r2 < a.rc2;
      const double y = rsqrt_seeded(r2), y2 = y * y;
      const double u = fma(r2, a.u_scale, -1.0);
      double fr = qq * fma(y, y2 - a.fshift, -poly_eval(a.cS, u));
      double s6 = 0.0, eps24 = 0.0;
      if (lj_row && __any_sync(0xffffffffu, (lj_mask >> tj) & 1u)) {   // LJ partners are rare (O-O only in water)
        const double2 lj = lds_d2(sTi + tj * 32);        // 24 eps, sigma^2
        eps24 = lj.x;
        const double s2 = lj.y * y2;
        s6 = s2 * s2 * s2;
        fr = fma(eps24 * y2, fma(s6 + s6, s6, -s6), fr);
      }
      fr = in ? fr : 0.0;
      Fx = fma(fr, dx, Fx); Fy = fma(fr, dy, Fy); Fz = fma(fr, dz, Fz);
      if (ENERGY) {
        const double r = r2 * y;
        const double up = qq * (y - poly_eval(a.cE, u) - a.erfc_rc + a.fshift * (r - a.rc)) +
                          (1.0 / 6.0) * eps24 * (s6 * s6 - s6) - lds_d(sTi + tj * 32 + 24);
        U += in ? up : 0.0;
        hits += in ? 1ull : 0ull;
      }
    };

    for (int m = 0; m < nblk; ++m) {
      uint4 nxt = cur;
      if (m + 1 < nblk) nxt = *reinterpret_cast<const uint4 *>(rowp + STG_BLOCK * (m + 1) + 8 * lane);
      const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
      auto entry = [&](int j) { return (j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu); };
      const int nst = min(8, (n - STG_BLOCK * m + 31) >> 5);
      // ---- check: pre-test of 32 entries per step, survivors compacted into the queue; the staged record
      //      of the next step is requested before this step's compaction store ------------------------------
      uint2 cj = make_uint2(0u, 0u);
      double2 xyj = make_double2(0.0, 0.0);
      double zj = 0.0;
      if (F32) cj = lds_u2(sC + (entry(0) & STG_IDX_MASK) * 8);
      else { xyj = lds_d2(sXY + (entry(0) & STG_IDX_MASK) * 16); zj = lds_d(sZ + (entry(0) & STG_IDX_MASK) * 8); }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (j >= nst) break;
        const uint32_t e = entry(j);
        bool hit;
        if (F32) {
          hit = half_test(ci, cj, a.rc2h);
          if (j < 7) cj = lds_u2(sC + (entry(j + 1) & STG_IDX_MASK) * 8);
        } else {
          const double dx = xyi.x - xyj.x, dy = xyi.y - xyj.y, dz = zi - zj;
          hit = fma(dz, dz, fma(dy, dy, dx * dx)) < a.rc2;
          if (j < 7) { xyj = lds_d2(sXY + (entry(j + 1) & STG_IDX_MASK) * 16); zj = lds_d(sZ + (entry(j + 1) & STG_IDX_MASK) * 8); }
        }
        unsigned mask;
        asm volatile("{ .reg .pred p; setp.ne.u32 p, %1, 0; vote.sync.ballot.b32 %0, p, 0xffffffff; }" : "=r"(mask) : "r"((unsigned)hit));
        if (hit) sts_u(qa + __popc(mask & lt) * 4, e);
        qa += __popc(mask) * 4;
      }
      __syncwarp();
      // ---- eval: full warps of survivors ---------------------------------------------------------------
      while (qa >= sQ + 128) {
        qa -= 128;
        eval(lds_u(qa + lane * 4), true);
      }
      __syncwarp();
      cur = nxt;
    }
    if (qa > sQ) {
      const bool act = sQ + lane * 4 < qa;
      eval(act ? lds_u(sQ + lane * 4) : ei, act);
      __syncwarp();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      Fx += __shfl_xor_sync(0xffffffffu, Fx, o);
      Fy += __shfl_xor_sync(0xffffffffu, Fy, o);
      Fz += __shfl_xor_sync(0xffffffffu, Fz, o);
    }
    if (lane == 0) {
      double *o = a.Fs + ((long long)bead * a.N + slot) * 3;
      o[0] = Fx; o[1] = Fy; o[2] = Fz;
    }
  }
  if (ENERGY) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      U += __shfl_xor_sync(0xffffffffu, U, o);
      hits += __shfl_xor_sync(0xffffffffu, hits, o);
    }
    if (lane == 0) { su[warp] = U; atomicAdd(a.count, hits); }
    __syncthreads();
    if (tid == 0) {
      double s = 0.0;
      for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += su[k];
      a.part[(long long)blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
// S(w) = (4/sqrt(pi)) sum_k (-1)^k w^k / (k! (2k+3)),  E(w) = (2/sqrt(pi)) sum_k (-1)^k w^k / (k! (2k+1)):
// Taylor series of (1 - erfc(x) - (2x/sqrt(pi)) e^{-x^2}) / x^3 and erf(x)/x in w = x^2 (long double;
// the terms stay below e^w <= ~400 for w <= 6, so the alternating sum loses < 3 digits of 19).
static long double series_SE(long double w, int which) {
  const long double c = (which == 0 ? 4.0L : 2.0L) / sqrtl(acosl(-1.0L));
  long double term = 1.0L, sum = 0.0L;
  for (int k = 0; k < 200; ++k) {
    const long double t = term / (which == 0 ? (2 * k + 3) : (2 * k + 1));
    sum += t;
    if (fabsl(t) < 1e-24L * fabsl(sum) && k > 4) break;
    term *= -w / (long double)(k + 1);
  }
  return c * sum;
}

// degree-(QHP_NPOLY-1) Chebyshev interpolant of scale * f(w), w = (u + 1) wmax / 2, as monomials in u
static long double fit_poly(int which, long double wmax, long double scale, double *out) {
  const int n = QHP_NPOLY;
  const long double pi = acosl(-1.0L);
  long double fn[QHP_NPOLY], c[QHP_NPOLY];
  for (int j = 0; j < n; ++j) fn[j] = scale * series_SE((cosl(pi * (j + 0.5L) / n) + 1.0L) * 0.5L * wmax, which);
  for (int k = 0; k < n; ++k) {
    long double s = 0.0L;
    for (int j = 0; j < n; ++j) s += fn[j] * cosl(pi * k * (j + 0.5L) / n);
    c[k] = 2.0L * s / n;
  }
  c[0] *= 0.5L;
  // Chebyshev -> monomial: T_0 = 1, T_1 = u, T_{k+1} = 2 u T_k - T_{k-1}
  long double mono[QHP_NPOLY] = {0}, t0[QHP_NPOLY] = {0}, t1[QHP_NPOLY] = {0}, t2[QHP_NPOLY];
  t0[0] = 1.0L; t1[1] = 1.0L;
  for (int k = 0; k < n; ++k) {
    const long double *tk = (k == 0) ? t0 : t1;
    for (int m = 0; m < n; ++m) mono[m] += c[k] * tk[m];
    if (k >= 1) {
      for (int m = 0; m < n; ++m) t2[m] = (m ? 2.0L * t1[m - 1] : 0.0L) - t0[m];
      for (int m = 0; m < n; ++m) { t0[m] = t1[m]; t1[m] = t2[m]; }
    }
  }
  for (int m = 0; m < n; ++m) out[m] = (double)mono[m];
  // worst relative error of the fp64 Horner evaluation on a fine grid
  long double worst = 0.0L;
  for (int g = 0; g <= 400; ++g) {
    const double u = -1.0 + 2.0 * g / 400.0;
    double v = 0.0;
    for (int m = n - 1; m >= 0; --m) v = fma(v, u, out[m]);
    const long double ex = scale * series_SE(((long double)u + 1.0L) * 0.5L * wmax, which);
    const long double err = fabsl(((long double)v - ex) / ex);
    if (err > worst) worst = err;
  }
  return worst;
}

static size_t staged_atom_bytes(bool f32) { return 3 * sizeof(double) + (f32 ? sizeof(uint2) : 0); }
static size_t staged_smem_bytes(int cap, int warps, bool f32) {
  return (size_t)cap * staged_atom_bytes(f32) + 16 + sizeof(double) * (QHP_MAX_TYPES * QHP_MAX_TYPES * 4 + QHP_MAX_TYPES) +
         sizeof(uint32_t) * (size_t)warps * STG_QUEUE;
}

// decide whether the staged kernel can serve this system and fit the polynomial tables
int qhp_pair_setup(qhp_system *s) {
  s->staged_ok = false;
  if (s->nc[0] < 4 || s->nc[1] < 4 || s->nc[2] < 4) return QHP_OK;    // cell-centre coordinates need >= 4 cells
  if (s->N / s->ncell < 8) return QHP_OK;                             // sparse boxes: one CTA per cell does not pay
  const long double al = s->alpha, rc = s->r_cut, wmax = al * al * rc * rc;
  if (wmax > 6.0L) return QHP_OK;                                     // polynomial degree fixed: generic kernel instead
  const long double eS = fit_poly(0, wmax, al * al * al, s->polyS);
  const long double eE = fit_poly(1, wmax, al, s->polyE);
  if (!(eS < 2e-14L && eE < 2e-14L)) return QHP_OK;
  int max_smem = 0;
  QHP_CUDA_OK(s, cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, s->device));
  s->staged_smem_max = max_smem - 1024;                                // room for the static shared variables
  if (s->staged_smem_max < 64 * 1024) return QHP_OK;
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_staged<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->staged_smem_max));
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_staged<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->staged_smem_max));
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_staged<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->staged_smem_max));
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_staged<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->staged_smem_max));
  // CTAs per (cell, bead): aim at >= 6 waves of one CTA per SM, keep >= one atom per warp
  int sms = 148;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device);
  long long ctas = (long long)s->ncell * s->Pc;
  int split = (int)((6LL * sms + ctas - 1) / ctas);
  const int per_cell = s->N / s->ncell + 1;
  while (split > 1 && per_cell / split < STG_MAX_WARPS) --split;
  if (split < 1) split = 1;
  if (split > 8) split = 8;
  s->staged_split = split;
  s->staged_ok = true;
  return QHP_OK;
}

int qhp_pair_staged_partials(const qhp_system *s) { return s->ncell * 8 * s->Pc; }

// Largest CTA (in warps) whose queues leave room for `region` staged atoms (+ 1/16 for drift between
// list builds); sets staged_warps / staged_cap.  False: the neighbourhood does not fit at all.
bool qhp_pair_staged_fit(qhp_system *s, long long region) {
  static const int tries[] = {STG_MAX_WARPS, 24, 16};
  const long long need = region + region / 16 + 32 + 1;               // + the dummy at cap - 1
  // first choice: the fp16 pre-test copy with the largest CTA; then the same CTA sizes without the copy
  for (int f32 = 1; f32 >= 0; --f32)
    for (int w : tries) {
      if (w > STG_MAX_WARPS) continue;
      const long long room = (long long)s->staged_smem_max - (long long)staged_smem_bytes(0, w, f32 != 0);
      long long cap = room / (long long)staged_atom_bytes(f32 != 0);
      if (cap > (1 << STG_IDX_BITS)) cap = 1 << STG_IDX_BITS;           // 13-bit staged indices in the list entries
      cap &= ~3LL;                                                     // keeps the arrays behind the positions aligned
      if (cap >= need) { s->staged_warps = w; s->staged_cap = (int)cap; s->staged_f32 = f32 != 0; return true; }
      if (f32 && w == STG_MAX_WARPS) break;                            // a smaller CTA is worse than dropping the copy
    }
  return false;
}

int qhp_pair_staged_forces(qhp_system *s, bool energy, double *part, unsigned long long *count, int bead0, int nbeads) {
  StagedArgs a{};
  a.bead0 = bead0;
  a.N = s->N; a.Pc = s->Pc; a.nt = s->nt; a.split = s->staged_split; a.cap = s->staged_cap;
  for (int d = 0; d < 3; ++d) {
    a.nc[d] = s->nc[d]; a.box[d] = s->box[d]; a.inv_box[d] = s->inv_box[d];
    a.cell_edge[d] = s->box[d] / s->nc[d];
  }
  a.pos4 = s->pos4; a.Fs = s->Fs; a.nbr16 = s->nbr16; a.nbr_count = s->nbr_count; a.cell_start = s->cell_start;
  a.stride = s->nbr_stride; a.pair_tab = s->pair_tab;
  const double rc = s->r_cut, al = s->alpha;
  a.rc = rc; a.rc2 = rc * rc; a.u_scale = 2.0 / (rc * rc);
  a.erfc_rc = erfc(al * rc) / rc;
  a.fshift = erfc(al * rc) / (rc * rc) + 2.0 * al / sqrt(QHP_PI) * exp(-al * al * rc * rc) / rc;
  {
    // fp16 pre-test threshold = r_c^2 + a bound on the error of the packed-half r^2, rounded UP to a half.
    // Staged coordinates reach 1.5 cell edges + skin: rounding them to half moves each by <= ulp(cmax)/2; the half
    // difference of two records adds <= ulp(r_c + 1)/2; so each component of d is off by e_d, r^2 by
    // <= 2 sqrt(3) r_c' e_d + 3 e_d^2 (r_c' = r_c + 1 covers the margin itself); the product, the fma, the sum and the
    // rounding of the threshold add <= 4 half-ulps at r_c^2 + margin.  The float -> half double rounding of the
    // staging adds 2^-13 relative to the half-ulp (the 1.01).  Pairs certainly outside r_c are the only ones rejected.
    auto ulp16 = [](double v) { int e; frexp(v, &e); return ldexp(1.0, e - 11); };   // spacing of halves just below 2^e >= v
    double cmax = 0.0;
    for (int d = 0; d < 3; ++d) cmax = fmax(cmax, 1.5 * a.cell_edge[d] + s->skin + 1.0);
    const double e_d = 1.01 * (ulp16(cmax) + 0.5 * ulp16(rc + 1.0));
    double thr = rc * rc + 2.0 * sqrt(3.0) * (rc + 1.0) * e_d + 3.0 * e_d * e_d;
    thr += 2.0 * ulp16(thr + 4.0);
    __half h = __double2half(thr);                                      // round to nearest, then step up if it fell below
    if (__half2float(h) < thr) {
      unsigned short b = *reinterpret_cast<unsigned short *>(&h);
      ++b;
      h = *reinterpret_cast<__half *>(&b);
    }
    const unsigned short hb = *reinterpret_cast<unsigned short *>(&h);
    a.rc2h = (unsigned)hb | ((unsigned)hb << 16);
    s->staged_thr = (double)__half2float(h);
  }
  for (int k = 0; k < QHP_NPOLY; ++k) { a.cS[k] = s->polyS[k]; a.cE[k] = s->polyE[k]; }
  for (int t = 0; t < s->nt; ++t) {
    a.qs[t] = sqrt(QHP_COUL) * s->charge[t];
    a.lj_mask[t] = 0u;
    for (int u = 0; u < s->nt; ++u)
      if (s->lj_eps[t] > 0 && s->lj_eps[u] > 0) a.lj_mask[t] |= 1u << u;
  }
  a.part = part; a.count = count; a.counters = (long long *)s->counters;
  const dim3 grid((unsigned)(s->ncell * s->staged_split), (unsigned)nbeads);
  const size_t smem = staged_smem_bytes(s->staged_cap, s->staged_warps, s->staged_f32);
  const int threads = 32 * s->staged_warps;
  if (s->staged_f32) {
    if (energy) k_pair_staged<true, true><<<grid, threads, smem, s->stream>>>(a);
    else k_pair_staged<false, true><<<grid, threads, smem, s->stream>>>(a);
  } else {
    if (energy) k_pair_staged<true, false><<<grid, threads, smem, s->stream>>>(a);
    else k_pair_staged<false, false><<<grid, threads, smem, s->stream>>>(a);
  }
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}
