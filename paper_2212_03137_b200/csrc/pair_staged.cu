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
//
// Kernels of this file:
//   k_pair_staged<ENERGY, F32>   the design above (pre-test + compaction + evaluation on the centroid table every step):
//                                energy variant of every staged system, force path when the pruned rows are off / do not fit;
//   k_prune_check, k_prune       per contracted bead, a second table with the entries within r_c + prune_skin of the bead's
//                                own positions, renewed on the device when the bead has moved prune_skin / 2 or the centroid
//                                table was rebuilt (see the comment above k_prune_check);
//   k_pair_dense<COUNT>          evaluation of those pruned rows without pre-test: the force path of C3 / C4.
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
  // k_pair_dense: rows of the table it walks ([bead][N][stride] pruned rows, or the shared table with bead strides 0)
  long long list_bead_stride;    // entries between the tables of two beads
  long long count_bead_stride;   // row counts between two beads
  int dcap;                      // staged atoms of the dense kernel (dummy at dcap - 1)
  long long *pruned_at;          // [Pc] or NULL: written with the rebuild count by CTA (0, bead)
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
  if (tid < 32) {                             // prefix over the 27 stencil cells by one warp
    if (tid == 0) next_atom = 0;
    int v = tid < 27 ? off[tid + 1] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (tid >= o) v += u; }
    if (tid < 27) off[tid + 1] = v;
    if (tid == 0) off[0] = 0;
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
    // one warp per stencil cell at a time: coalesced 32-byte records, no search for the cell of a staged index
    constexpr int UN = 3;                                // independent loads in flight per lane
    for (int s = warp; s < 27; s += nthr >> 5) {
      const int o = off[s], n = off[s + 1] - o;
      const double4 *src = pos + cbeg[s];
      for (int k0 = lane; k0 < n; k0 += UN * 32) {
        double4 p[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u)
          if (k0 + 32 * u < n) p[u] = src[k0 + 32 * u];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
          const int k = k0 + 32 * u;
          if (k < n) {
            double lx = p[u].x - ctr[0], ly = p[u].y - ctr[1], lz = p[u].z - ctr[2];
            lx = fma(-a.box[0], (lx * a.inv_box[0] + MAGIC) - MAGIC, lx);
            ly = fma(-a.box[1], (ly * a.inv_box[1] + MAGIC) - MAGIC, ly);
            lz = fma(-a.box[2], (lz * a.inv_box[2] + MAGIC) - MAGIC, lz);
            XY[o + k] = make_double2(lx, ly); Z[o + k] = lz;
            if (F32) C[o + k] = half_record(lx, ly, lz);
          }
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
// k_pair_dense: evaluation without pre-test.  Same CTA-per-(cell, bead) staging, but only the fp64 records
// (24 B per staged atom: two CTAs per SM) and no queue: every entry of the row is evaluated, the exact fp64
// r^2 < r_c^2 test masks the result.  Pays when the rows are dense (the pruned per-bead rows: >= 85 % of the
// entries inside r_c).  COUNT (parity hook qhp_pair_prune_stats only) also counts the pairs that pass the fp64 test.
// ---------------------------------------------------------------------------------------------
#ifndef DNS_THREADS
#define DNS_THREADS 448          // 14 warps x 2 CTAs per SM at 72 registers (512: 64 registers, spills)
#endif
#ifndef DNS_CTAS
#define DNS_CTAS 2
#endif
template <bool COUNT>
__global__ void __launch_bounds__(DNS_THREADS, DNS_CTAS) k_pair_dense(const StagedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2 *XY = reinterpret_cast<double2 *>(smem_raw);
  double *Z = reinterpret_cast<double *>(XY + a.dcap);
  double *tab = reinterpret_cast<double *>(Z + a.dcap);
  double *qtab = tab + a.nt * a.nt * 4;                     // tables sized by the number of types: room for staged atoms
  __shared__ int off[28], cbeg[27];

  const int tid = threadIdx.x, lane = tid & 31, nthr = blockDim.x;
  const int cell = blockIdx.x / a.split, part = blockIdx.x % a.split, bead = a.bead0 + blockIdx.y;
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);
  // the rows of this bead were made current by the k_prune launch in front of this one: record their rebuild count
  if (a.pruned_at && blockIdx.x == 0 && tid == 0) a.pruned_at[bead] = a.counters[0];

  for (int k = tid; k < a.nt * a.nt * 4; k += nthr) {      // (qq, 4 eps, sigma^2, shift) -> (24 eps, sigma^2, qq, shift)
    const int f = k & 3;
    tab[(k & ~3) + (f == 0 ? 2 : (f == 1 ? 0 : (f == 2 ? 1 : 3)))] = (f == 1 ? 6.0 : 1.0) * a.pair_tab[k];
  }
  if (tid < a.nt) qtab[tid] = a.qs[tid];
  if (tid < 27) {
    const int ox = tid / 9, oy = (tid / 3) % 3, oz = tid % 3;
    const int qx = (cx - 1 + ox + a.nc[0]) % a.nc[0], qy = (cy - 1 + oy + a.nc[1]) % a.nc[1],
              qz = (cz - 1 + oz + a.nc[2]) % a.nc[2];
    const int c2 = (qx * a.nc[1] + qy) * a.nc[2] + qz;
    cbeg[tid] = a.cell_start[c2];
    off[tid + 1] = a.cell_start[c2 + 1] - a.cell_start[c2];
  }
  __syncthreads();
  if (tid < 32) {                             // prefix over the 27 stencil cells by one warp
    int v = tid < 27 ? off[tid + 1] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (tid >= o) v += u; }
    if (tid < 27) off[tid + 1] = v;
    if (tid == 0) off[0] = 0;
  }
  __syncthreads();
  const int total = off[27];
  if (off[14] == off[13]) return;
  if (total > a.dcap - 1) {
    if (tid == 0) a.counters[7] = 1;
    return;
  }
  const double4 *pos = reinterpret_cast<const double4 *>(a.pos4) + (long long)bead * a.N;
  const int h0 = off[13], nh = off[14] - off[13], slot0 = cbeg[13];
  const uint16_t *table = a.nbr16 + (long long)bead * a.list_bead_stride;
  const int32_t *counts = a.nbr_count + (long long)bead * a.count_bead_stride;
  // Rows are dealt to the warps round-robin (rows of one cell have near-equal lengths); the next row's count, type
  // and first block are requested before the current row is evaluated (the first one before the staging), so a row
  // never starts on a global-load wait.
  // (the broadcast tells the compiler that the row loop is warp-uniform: polynomial coefficients stay in uniform registers)
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0), istep = a.split * (nthr >> 5);
  int ii = part + a.split * warp;
  int n_nx = 0, ti_nx = 0;
  uint4 cur = make_uint4(0u, 0u, 0u, 0u);                  // the block being evaluated; its successor (same row or next row) in flight
  if (ii < nh) {
    n_nx = counts[slot0 + ii];
    ti_nx = (int)__double_as_longlong(pos[slot0 + ii].w);
    cur = *reinterpret_cast<const uint4 *>(table + (long long)(slot0 + ii) * a.stride + 8 * lane);
  }
  {
    const double ctr[3] = {(cx + 0.5) * a.cell_edge[0], (cy + 0.5) * a.cell_edge[1], (cz + 0.5) * a.cell_edge[2]};
    const double MAGIC = 6755399441055744.0;
    // one warp per stencil cell at a time: coalesced 32-byte records, no search for the cell of a staged index
    constexpr int UN = 3;                                // independent loads in flight per lane
    for (int s = tid >> 5; s < 27; s += nthr >> 5) {
      const int o = off[s], n = off[s + 1] - o;
      const double4 *src = pos + cbeg[s];
      for (int k0 = lane; k0 < n; k0 += UN * 32) {
        double4 p[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u)
          if (k0 + 32 * u < n) p[u] = src[k0 + 32 * u];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
          const int k = k0 + 32 * u;
          if (k < n) {
            double lx = p[u].x - ctr[0], ly = p[u].y - ctr[1], lz = p[u].z - ctr[2];
            lx = fma(-a.box[0], (lx * a.inv_box[0] + MAGIC) - MAGIC, lx);
            ly = fma(-a.box[1], (ly * a.inv_box[1] + MAGIC) - MAGIC, ly);
            lz = fma(-a.box[2], (lz * a.inv_box[2] + MAGIC) - MAGIC, lz);
            XY[o + k] = make_double2(lx, ly); Z[o + k] = lz;
          }
        }
      }
    }
    if (tid == 0) { XY[a.dcap - 1] = make_double2(1e9, 1e9); Z[a.dcap - 1] = 1e9; }
  }
  __syncthreads();

  const uint32_t sXY = (uint32_t)__cvta_generic_to_shared(XY), sZ = (uint32_t)__cvta_generic_to_shared(Z),
                 sTab = (uint32_t)__cvta_generic_to_shared(tab), sQt = (uint32_t)__cvta_generic_to_shared(qtab);
  unsigned long long hits = 0;
  // per-row pointers advance by fixed strides (kept in registers: the compiler otherwise rebuilds each address from
  // the kernel parameters in every row, ~60 instructions of 64-bit arithmetic)
  const uint16_t *rowp = table + (long long)(slot0 + ii) * a.stride + 8 * lane;
  const int32_t *cntp = counts + slot0 + ii;
  const double *typp = reinterpret_cast<const double *>(pos + slot0 + ii) + 3;
  const long long row_step = (long long)istep * a.stride;
  asm volatile("" : "+l"(rowp), "+l"(cntp), "+l"(typp));

  for (; ii < nh; ii += istep, rowp += row_step, cntp += istep, typp += 4 * istep) {
    const uint32_t ei = (uint32_t)(h0 + ii);
    const long long slot = slot0 + ii;
    const int n = n_nx, ti = ti_nx;
    const int nblk = max(1, (n + STG_BLOCK - 1) / STG_BLOCK);
    const bool more = ii + istep < nh;
    if (more) {
      n_nx = cntp[istep];
      ti_nx = (int)__double_as_longlong(typp[4 * istep]);
    }
    const double2 xyi = lds_d2(sXY + ei * 16);
    const double zi = lds_d(sZ + ei * 8);
    const uint32_t sTi = sTab + (uint32_t)(ti * a.nt) * 32u;
    const double qi = lds_d(sQt + ti * 8);
    const unsigned lj_mask = a.lj_mask[ti];
    const bool lj_row = lj_mask != 0u;
    double Fx = 0.0, Fy = 0.0, Fz = 0.0;

    // The staged records of an entry are requested one evaluation ahead (a warp issues in order: without this every
    // evaluation starts on the latency of its own gathers).  Entries behind the row's last step are not initialised:
    // the index is clamped to the dummy.
    const uint32_t dummyi = (uint32_t)(a.dcap - 1);
    double2 xyn = make_double2(0.0, 0.0);
    double zn = 0.0;
    auto fetch = [&](uint32_t entry) {
      const uint32_t sj = min(entry & STG_IDX_MASK, dummyi);
      xyn = lds_d2(sXY + sj * 16); zn = lds_d(sZ + sj * 8);
    };
    auto eval = [&](uint32_t entry, uint32_t next) {
      const uint32_t tj = entry >> STG_IDX_BITS;
      const double2 xyj = xyn;
      const double zj = zn;
      fetch(next);
      const double qq = qi * lds_d(sQt + tj * 8);
      const double dx = xyi.x - xyj.x, dy = xyi.y - xyj.y, dz = zi - zj;
      const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
      const bool in = r2 < a.rc2;
      const double y = rsqrt_seeded(r2), y2 = y * y;
      const double u = fma(r2, a.u_scale, -1.0);
      double fr = qq * fma(y, y2 - a.fshift, -poly_eval(a.cS, u));
      if (lj_row && __any_sync(0xffffffffu, (lj_mask >> tj) & 1u)) {
        const double2 lj = lds_d2(sTi + tj * 32);        // 24 eps, sigma^2
        const double s2 = lj.y * y2;
        const double s6 = s2 * s2 * s2;
        fr = fma(lj.x * y2, fma(s6 + s6, s6, -s6), fr);
      }
      fr = in ? fr : 0.0;
      Fx = fma(fr, dx, Fx); Fy = fma(fr, dy, Fy); Fz = fma(fr, dz, Fz);
      if (COUNT) hits += in ? 1ull : 0ull;
    };

    for (int m = 0; m < nblk; ++m) {
      uint4 nxt = cur;
      if (m + 1 < nblk) nxt = *reinterpret_cast<const uint4 *>(rowp + STG_BLOCK * (m + 1));
      else if (more) nxt = *reinterpret_cast<const uint4 *>(rowp + row_step);   // first block of the next row
      const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
      const int nst = min(8, (n - STG_BLOCK * m + 31) >> 5);
      fetch(w[0] & 0xffffu);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (j >= nst) break;
        const int jn = j < 7 ? j + 1 : 7;                  // (the last step of a block re-requests its own record: harmless)
        eval((j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu), (jn & 1) ? (w[jn >> 1] >> 16) : (w[jn >> 1] & 0xffffu));
      }
      cur = nxt;
    }
    // (Fx, Fy, Fz) over the 32 lanes in 6 exchanges instead of 15: the halves of the warp first swap what the other
    // one keeps (lower: x, y; upper: z), then quarters split x | y, then a plain butterfly; fixed order -> reproducible
    {
      const bool up = lane & 16, q = lane & 8;
      const double r1 = __shfl_xor_sync(0xffffffffu, up ? Fx : Fz, 16);
      const double r2 = __shfl_xor_sync(0xffffffffu, up ? Fy : 0.0, 16);
      const double A = (up ? Fz : Fx) + r1, B = up ? 0.0 : Fy + r2;
      double V = (q ? B : A) + __shfl_xor_sync(0xffffffffu, q ? A : B, 8);
      V += __shfl_xor_sync(0xffffffffu, V, 4);
      V += __shfl_xor_sync(0xffffffffu, V, 2);
      V += __shfl_xor_sync(0xffffffffu, V, 1);
      if ((lane & 7) == 0 && lane < 24) a.Fs[((long long)bead * a.N + slot) * 3 + (lane >> 3)] = V;
    }
  }
  if (COUNT) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, o);
    if (lane == 0) atomicAdd(a.count, hits);
  }
}

// ---------------------------------------------------------------------------------------------
// Pruned per-bead rows for k_pair_dense.  The centroid table (skin 2 A, shared by all beads, the list the
// oracle is compared with) holds ~1.8x the pairs inside r_c.  k_prune copies, per contracted bead, the entries
// within r_c + prune_skin of the bead's CURRENT positions into a second table (same blocked 16-bit row format,
// dummy = dcap - 1) and records those positions (pref4).  The pruned rows of a bead stay complete while no atom
// of that bead has moved by more than prune_skin / 2 since (k_prune_check, every step) and the centroid table has
// not been rebuilt (pruned_at[bead] == rebuild count): both are tested on the device, no host round trip.
// The prune test is the packed-half pre-test (conservative: it keeps every pair inside its radius).
// ---------------------------------------------------------------------------------------------
#define PRUNE_CHECK_CTAS 296
#ifndef PRUNE_THREADS
#define PRUNE_THREADS 512
#endif
#define PRUNE_WARPS (PRUNE_THREADS / 32)
#define PRUNE_QUEUE (2 * STG_BLOCK)      // circular: < 256 entries waiting + 256 new ones per warp (a power of two)

struct PruneArgs {
  int N, Pc, nt, cap, bead0;     // cap = dcap of the dense kernel (dummy at cap - 1)
  int ccap, src_dummy;           // records staged here (>= both staged arrays); dummy index of the centroid rows
  int nc[3];
  double box[3], inv_box[3], cell_edge[3];
  const double *pos4;            // [Pc][N][4] current contracted beads, slot order
  double *pref4;                 // [Pc][N][4] positions the pruned rows were made from
  const uint16_t *nbr16;         // centroid table [N][stride]
  const int32_t *nbr_count, *cell_start;
  uint16_t *nbr16p;              // [Pc][N][stride] pruned rows
  int32_t *nbr_count_p;          // [Pc][N]
  long long stride;
  double *part;                  // [Pc][PRUNE_CHECK_CTAS] per-CTA maxima of |pos - pref|^2
  long long *pruned_at;          // [Pc] rebuild count the pruned rows of the bead belong to (-1: none)
  int *work;                     // [Pc] next cell of k_prune (zeroed by k_prune_check every step)
  long long *nprune;             // [Pc] number of prunes of the bead so far (statistics)
  const long long *counters;     // [0] = rebuild count
  double move2;                  // (prune_skin / 2)^2
  unsigned thr_h;                // packed-half threshold for r_c + prune_skin
};

// every step: per-bead maximum of the squared displacement since the last prune (fixed order, no atomics)
__global__ void __launch_bounds__(256) k_prune_check(const PruneArgs a) {
  __shared__ double red[8];
  const int bead = a.bead0 + blockIdx.y;
  const double4 *p = reinterpret_cast<const double4 *>(a.pos4) + (long long)bead * a.N;
  const double4 *r = reinterpret_cast<const double4 *>(a.pref4) + (long long)bead * a.N;
  double m = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < a.N; i += gridDim.x * blockDim.x) {
    const double4 u = p[i], v = r[i];
    const double dx = u.x - v.x, dy = u.y - v.y, dz = u.z - v.z;
    const double d2 = fma(dz, dz, fma(dy, dy, dx * dx));
    m = (d2 > m || d2 != d2) ? d2 : m;                   // a NaN sticks: the comparison in k_prune then fails towards "prune"
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double t = __shfl_xor_sync(0xffffffffu, m, o);
    m = (t > m || t != t) ? t : m;
  }
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = (red[w] > m || red[w] != red[w]) ? red[w] : m;
    a.part[(long long)bead * PRUNE_CHECK_CTAS + blockIdx.x] = m;
    if (blockIdx.x == 0) a.work[bead] = 0;
  }
}

// the rows of bead `bead` must be pruned again (uniform over the grid: read-only inputs of this launch); all threads
// of the CTA call it
__device__ __forceinline__ bool prune_due(const PruneArgs &a, int bead) {
  const int t = threadIdx.x;
  int f = (t == 0) && (a.pruned_at[bead] != a.counters[0]);
  if (t < PRUNE_CHECK_CTAS) f |= !(a.part[(long long)bead * PRUNE_CHECK_CTAS + t] < a.move2);   // NaN: prune
  return __syncthreads_or(f) != 0;
}

__global__ void __launch_bounds__(PRUNE_THREADS, 2) k_prune(const PruneArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint2 *C = reinterpret_cast<uint2 *>(smem_raw);
  uint32_t *queue = reinterpret_cast<uint32_t *>(C + a.ccap);
  __shared__ int off[28], cbeg[27];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x;
  const int bead = a.bead0 + blockIdx.y;
  if (!prune_due(a, bead)) return;
  if (blockIdx.x == 0 && tid == 0) a.nprune[bead] += 1;
  // a small grid (the launch returns at once on most steps) takes the cells from a work counter
  __shared__ int cell_s;
  for (;;) {
  __syncthreads();                                         // the previous cell's shared arrays are no longer read
  if (tid == 0) cell_s = atomicAdd(&a.work[bead], 1);
  __syncthreads();
  const int cell = cell_s;
  if (cell >= a.nc[0] * a.nc[1] * a.nc[2]) break;
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);
  if (tid < 27) {
    const int ox = tid / 9, oy = (tid / 3) % 3, oz = tid % 3;
    const int qx = (cx - 1 + ox + a.nc[0]) % a.nc[0], qy = (cy - 1 + oy + a.nc[1]) % a.nc[1],
              qz = (cz - 1 + oz + a.nc[2]) % a.nc[2];
    const int c2 = (qx * a.nc[1] + qy) * a.nc[2] + qz;
    cbeg[tid] = a.cell_start[c2];
    off[tid + 1] = a.cell_start[c2 + 1] - a.cell_start[c2];
  }
  __syncthreads();
  if (tid < 32) {                             // prefix over the 27 stencil cells by one warp
    int v = tid < 27 ? off[tid + 1] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (tid >= o) v += u; }
    if (tid < 27) off[tid + 1] = v;
    if (tid == 0) off[0] = 0;
  }
  __syncthreads();
  const int total = off[27];
  if (off[14] == off[13] || total > a.cap - 1) continue;   // the dense kernel reports the overflow
  const double4 *pos = reinterpret_cast<const double4 *>(a.pos4) + (long long)bead * a.N;
  {
    const double ctr[3] = {(cx + 0.5) * a.cell_edge[0], (cy + 0.5) * a.cell_edge[1], (cz + 0.5) * a.cell_edge[2]};
    const double MAGIC = 6755399441055744.0;
    // one warp per stencil cell at a time (as in k_pair_dense); the home cell's positions become the reference of the
    // displacement check
    constexpr int UN = 3;
    for (int s = tid >> 5; s < 27; s += nthr >> 5) {
      const int o = off[s], n = off[s + 1] - o;
      const double4 *src = pos + cbeg[s];
      double4 *ref = reinterpret_cast<double4 *>(a.pref4) + (long long)bead * a.N + cbeg[s];
      for (int k0 = lane; k0 < n; k0 += UN * 32) {
        double4 p[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u)
          if (k0 + 32 * u < n) p[u] = src[k0 + 32 * u];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
          const int k = k0 + 32 * u;
          if (k < n) {
            double lx = p[u].x - ctr[0], ly = p[u].y - ctr[1], lz = p[u].z - ctr[2];
            lx = fma(-a.box[0], (lx * a.inv_box[0] + MAGIC) - MAGIC, lx);
            ly = fma(-a.box[1], (ly * a.inv_box[1] + MAGIC) - MAGIC, ly);
            lz = fma(-a.box[2], (lz * a.inv_box[2] + MAGIC) - MAGIC, lz);
            C[o + k] = half_record(lx, ly, lz);
            if (s == 13) ref[k] = p[u];
          }
        }
      }
    }
  }
  if (tid == 0) C[a.src_dummy] = half_record(1e9, 1e9, 1e9);   // the padding of the centroid rows: no test against it passes
  __syncthreads();
  const int h0 = off[13], nh = off[14] - off[13], slot0 = cbeg[13];
  const uint32_t sC = (uint32_t)__cvta_generic_to_shared(C),
                 sQ = (uint32_t)__cvta_generic_to_shared(queue) + warp * (PRUNE_QUEUE * 4);
  unsigned lt;
  asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt));
  const uint32_t dummy = (uint32_t)(a.cap - 1);
  // Rows are dealt to the warps round-robin; the next block of entries (of this row or of the warp's next row) and the
  // next row's count are requested one block ahead.  Survivors go into a circular queue of 512 slots per warp
  // (tail = entries of the row so far, head = entries written out, a multiple of 256).
  const int nw = nthr >> 5, wrp = __shfl_sync(0xffffffffu, warp, 0);
  int ii = wrp, n_nx = 0;
  uint4 cur = make_uint4(0u, 0u, 0u, 0u);
  if (ii < nh) {
    n_nx = a.nbr_count[slot0 + ii];
    cur = *reinterpret_cast<const uint4 *>(a.nbr16 + (long long)(slot0 + ii) * a.stride + 8 * lane);
  }
  for (; ii < nh; ii += nw) {
    const long long slot = slot0 + ii;
    const int n = n_nx;
    const uint16_t *rowp = a.nbr16 + slot * a.stride;
    uint16_t *outp = a.nbr16p + ((long long)bead * a.N + slot) * a.stride;
    const int nblk = max(1, (n + STG_BLOCK - 1) / STG_BLOCK);
    const bool more = ii + nw < nh;
    if (more) n_nx = a.nbr_count[slot + nw];
    const uint2 ci = lds_u2(sC + (uint32_t)(h0 + ii) * 8);
    uint32_t tail = 0, head = 0;
    // one 256-entry block of the pruned row from queue slots head .. head + 255 (lane l: entries 32 j + l, j = 0..7)
    auto flush = [&]() {
      uint32_t e[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) e[j] = lds_u(sQ + ((head + 32 * j + lane) & (PRUNE_QUEUE - 1)) * 4);
      *reinterpret_cast<uint4 *>(outp + head + 8 * lane) =
          make_uint4(e[0] | (e[1] << 16), e[2] | (e[3] << 16), e[4] | (e[5] << 16), e[6] | (e[7] << 16));
    };
    for (int m = 0; m < nblk; ++m) {
      uint4 nxt = cur;
      if (m + 1 < nblk) nxt = *reinterpret_cast<const uint4 *>(rowp + STG_BLOCK * (m + 1) + 8 * lane);
      else if (more) nxt = *reinterpret_cast<const uint4 *>(rowp + (long long)nw * a.stride + 8 * lane);   // first block of the next row
      const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
      auto entry = [&](int j) { return (j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu); };
      const int nst = min(8, (n - STG_BLOCK * m + 31) >> 5);
      uint2 cj = lds_u2(sC + (entry(0) & STG_IDX_MASK) * 8);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (j >= nst) break;
        const uint32_t e = entry(j);
        const bool hit = half_test(ci, cj, a.thr_h);
        if (j < 7) cj = lds_u2(sC + (entry(j + 1) & STG_IDX_MASK) * 8);
        unsigned mask;
        asm volatile("{ .reg .pred p; setp.ne.u32 p, %1, 0; vote.sync.ballot.b32 %0, p, 0xffffffff; }" : "=r"(mask) : "r"((unsigned)hit));
        if (hit) sts_u(sQ + ((tail + __popc(mask & lt)) & (PRUNE_QUEUE - 1)) * 4, e);
        tail += __popc(mask);
      }
      __syncwarp();
      if (tail - head >= STG_BLOCK) {
        flush();
        head += STG_BLOCK;
        __syncwarp();
      }
      cur = nxt;
    }
    if (tail > head) {                                     // < 256 entries left
      const uint32_t pad = (tail + 31u) & ~31u;
      if (tail + lane < pad) sts_u(sQ + ((tail + lane) & (PRUNE_QUEUE - 1)) * 4, dummy);   // complete the last 32-entry step
      __syncwarp();
      flush();                                             // entries behind `pad` are never read (row count)
      __syncwarp();
    }
    if (lane == 0) a.nbr_count_p[(long long)bead * a.N + slot] = (int)tail;
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

// fp16 pre-test threshold for radius r: r^2 + a bound on the error of the packed-half r^2, rounded UP to a half,
// both halves of a half2.  Staged coordinates reach 1.5 cell edges + skin: rounding them to half moves each by
// <= ulp(cmax)/2; the half difference of two records adds <= ulp(r + 1)/2; so each component of d is off by e_d,
// r^2 by <= 2 sqrt(3) r' e_d + 3 e_d^2 (r' = r + 1 covers the margin itself); the product, the fma, the sum and
// the rounding of the threshold add <= 4 half-ulps at r^2 + margin.  The float -> half double rounding of the
// staging adds 2^-13 relative to the half-ulp (the 1.01).  Only pairs certainly outside r are rejected.
static unsigned half_threshold(const qhp_system *s, double r, double *thr_out) {
  auto ulp16 = [](double v) { int e; frexp(v, &e); return ldexp(1.0, e - 11); };   // spacing of halves just below 2^e >= v
  double cmax = 0.0;
  for (int d = 0; d < 3; ++d) cmax = fmax(cmax, 1.5 * s->box[d] / s->nc[d] + s->skin + 1.0);
  const double e_d = 1.01 * (ulp16(cmax) + 0.5 * ulp16(r + 1.0));
  double thr = r * r + 2.0 * sqrt(3.0) * (r + 1.0) * e_d + 3.0 * e_d * e_d;
  thr += 2.0 * ulp16(thr + 4.0);
  __half h = __double2half(thr);                                        // round to nearest, then step up if it fell below
  if (__half2float(h) < thr) {
    unsigned short b = *reinterpret_cast<unsigned short *>(&h);
    ++b;
    h = *reinterpret_cast<__half *>(&b);
  }
  const unsigned short hb = *reinterpret_cast<unsigned short *>(&h);
  if (thr_out) *thr_out = (double)__half2float(h);
  return (unsigned)hb | ((unsigned)hb << 16);
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

static size_t dense_tab_bytes(const qhp_system *s) { return sizeof(double) * ((size_t)s->nt * s->nt * 4 + (size_t)s->nt + 1); }

void qhp_pair_dense_free(qhp_system *s) {
  if (s->nbr16p) cudaFree(s->nbr16p);
  if (s->nbr_count_p) cudaFree(s->nbr_count_p);
  if (s->pref4) cudaFree(s->pref4);
  if (s->prune_part) cudaFree(s->prune_part);
  if (s->pruned_at) cudaFree(s->pruned_at);
  if (s->prune_work) cudaFree(s->prune_work);
  s->nbr16p = nullptr; s->nbr_count_p = nullptr; s->pref4 = nullptr; s->prune_part = nullptr; s->pruned_at = nullptr; s->prune_work = nullptr;
  s->nbr16p_stride = 0;
}

// Called at every synchronising list build (after the table and its stride are final): the pruned-row path serves
// the system when the staged kernel does, prune_skin > 0, and the densest neighbourhood leaves room for TWO
// k_pair_dense CTAs per SM (24 B per staged atom); allocates the per-bead tables and marks them stale.
int qhp_pair_dense_prepare(qhp_system *s, long long region) {
  s->dense = false;
  if (!s->staged || !s->staged_f32 || !(s->prune_skin > 0.0) || s->prune_skin >= s->skin) return QHP_OK;
  int sm_bytes = 0;
  QHP_CUDA_OK(s, cudaDeviceGetAttribute(&sm_bytes, cudaDevAttrMaxSharedMemoryPerMultiprocessor, s->device));
  const long long dyn = (long long)sm_bytes / DNS_CTAS - 1024 - 256;   // per-CTA reserve + the static shared variables
  long long cap = (dyn - (long long)dense_tab_bytes(s)) / 24;
  if (cap > (1 << STG_IDX_BITS)) cap = 1 << STG_IDX_BITS;
  cap &= ~3LL;
  if (cap < region + region / 32 + 32 + 1) return QHP_OK;               // one CTA per SM: the pre-test kernel is the better one
  s->dense_cap = (int)cap;
  const size_t PcN = (size_t)s->Pc * (size_t)s->N;
  if (!s->nbr16p || s->nbr16p_stride != s->nbr_stride) {
    qhp_pair_dense_free(s);
    cudaError_t e = cudaMalloc(&s->nbr16p, sizeof(uint16_t) * PcN * (size_t)s->nbr_stride);
    if (e == cudaSuccess) e = cudaMalloc(&s->nbr_count_p, sizeof(int32_t) * PcN);
    if (e == cudaSuccess) e = cudaMalloc(&s->pref4, sizeof(double) * 4 * PcN);
    if (e == cudaSuccess) e = cudaMalloc(&s->prune_part, sizeof(double) * (size_t)s->Pc * PRUNE_CHECK_CTAS);
    if (e == cudaSuccess) e = cudaMalloc(&s->pruned_at, sizeof(long long) * 2 * (size_t)s->Pc);      // + [Pc] prune counts
    if (e == cudaSuccess) e = cudaMalloc(&s->prune_work, sizeof(int) * (size_t)s->Pc);
    if (e != cudaSuccess) {
      cudaGetLastError();
      qhp_pair_dense_free(s);                                          // not fatal: the pre-test kernel serves the system
      return QHP_OK;
    }
    s->nbr16p_stride = s->nbr_stride;
    QHP_CUDA_OK(s, cudaMemsetAsync(s->pref4, 0, sizeof(double) * 4 * PcN, s->stream));
    QHP_CUDA_OK(s, cudaMemsetAsync(s->prune_part, 0, sizeof(double) * (size_t)s->Pc * PRUNE_CHECK_CTAS, s->stream));
    QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_dense<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    QHP_CUDA_OK(s, cudaFuncSetAttribute(k_pair_dense<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    QHP_CUDA_OK(s, cudaFuncSetAttribute(k_prune, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));   // <= 8192 records + queues
  }
  QHP_CUDA_OK(s, cudaMemsetAsync(s->pruned_at, 0xff, sizeof(long long) * (size_t)s->Pc, s->stream));   // -1: stale
  QHP_CUDA_OK(s, cudaMemsetAsync(s->pruned_at + s->Pc, 0, sizeof(long long) * (size_t)s->Pc, s->stream));
  s->dense = true;
  return QHP_OK;
}

// check (every step) -> prune (returns at once unless due) -> evaluation of the pruned rows
static int pair_dense_forces(qhp_system *s, StagedArgs &a, int bead0, int nbeads, bool count = false) {
  PruneArgs p{};
  p.N = s->N; p.Pc = s->Pc; p.nt = s->nt; p.cap = s->dense_cap; p.bead0 = bead0;
  for (int d = 0; d < 3; ++d) {
    p.nc[d] = s->nc[d]; p.box[d] = s->box[d]; p.inv_box[d] = s->inv_box[d]; p.cell_edge[d] = s->box[d] / s->nc[d];
  }
  p.pos4 = s->pos4; p.pref4 = s->pref4; p.nbr16 = s->nbr16; p.nbr_count = s->nbr_count; p.cell_start = s->cell_start;
  p.nbr16p = s->nbr16p; p.nbr_count_p = s->nbr_count_p; p.stride = s->nbr_stride;
  p.part = s->prune_part; p.pruned_at = s->pruned_at; p.work = s->prune_work; p.nprune = s->pruned_at + s->Pc; p.counters = (const long long *)s->counters;
  p.move2 = 0.25 * s->prune_skin * s->prune_skin;
  p.thr_h = half_threshold(s, s->r_cut + s->prune_skin, nullptr);
  {
    qhp_prof_scope ps(s, 5);
    k_prune_check<<<dim3(PRUNE_CHECK_CTAS, (unsigned)nbeads), 256, 0, s->stream>>>(p);
  }
  QHP_LAUNCH_OK(s);
  p.src_dummy = s->staged_cap - 1;                      // the centroid rows are padded with the dummy of k_pair_staged
  p.ccap = s->staged_cap > s->dense_cap ? s->staged_cap : s->dense_cap;
  const size_t psm = (size_t)p.ccap * sizeof(uint2) + sizeof(uint32_t) * PRUNE_WARPS * PRUNE_QUEUE;
  {
    qhp_prof_scope ps(s, 6);
    k_prune<<<dim3((unsigned)(s->ncell < PRUNE_CHECK_CTAS ? s->ncell : PRUNE_CHECK_CTAS), (unsigned)nbeads), PRUNE_THREADS, psm, s->stream>>>(p);
  }
  QHP_LAUNCH_OK(s);
  a.dcap = s->dense_cap;
  a.nbr16 = s->nbr16p; a.nbr_count = s->nbr_count_p;
  a.list_bead_stride = (long long)s->N * s->nbr_stride; a.count_bead_stride = s->N;
  a.pruned_at = s->pruned_at;
  const size_t sm = (size_t)s->dense_cap * 24 + dense_tab_bytes(s);
  const dim3 grid((unsigned)(s->ncell * s->staged_split), (unsigned)nbeads);
  {
    qhp_prof_scope ps(s, 7);
    if (count) k_pair_dense<true><<<grid, DNS_THREADS, sm, s->stream>>>(a);
    else k_pair_dense<false><<<grid, DNS_THREADS, sm, s->stream>>>(a);
  }
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

static int staged_args(qhp_system *s, StagedArgs &a, double *part, unsigned long long *count, int bead0) {
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
  a.rc2h = half_threshold(s, rc, &s->staged_thr);
  for (int k = 0; k < QHP_NPOLY; ++k) { a.cS[k] = s->polyS[k]; a.cE[k] = s->polyE[k]; }
  for (int t = 0; t < s->nt; ++t) {
    a.qs[t] = sqrt(QHP_COUL) * s->charge[t];
    a.lj_mask[t] = 0u;
    for (int u = 0; u < s->nt; ++u)
      if (s->lj_eps[t] > 0 && s->lj_eps[u] > 0) a.lj_mask[t] |= 1u << u;
  }
  a.part = part; a.count = count; a.counters = (long long *)s->counters;
  return QHP_OK;
}

int qhp_pair_staged_forces(qhp_system *s, bool energy, double *part, unsigned long long *count, int bead0, int nbeads) {
  StagedArgs a{};
  const int rc0 = staged_args(s, a, part, count, bead0);
  if (rc0) return rc0;
  const dim3 grid((unsigned)(s->ncell * s->staged_split), (unsigned)nbeads);
  if (!energy && s->dense) return pair_dense_forces(s, a, bead0, nbeads);
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

__global__ void k_sum_counts(const int32_t *__restrict__ c, long long n, unsigned long long *out) {
  unsigned long long v = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) v += (unsigned long long)c[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0 && v) atomicAdd(out, v);
}

// parity hook (include/qhp.h qhp_pair_prune_stats): the pruned rows are made current for the present state (exactly what
// a step does), V_s is evaluated through them with the counting variant of the kernel
int qhp_pair_prune_stats_impl(qhp_system *s, int64_t *out_host) {
  out_host[0] = s->staged && s->dense ? 1 : 0;
  out_host[1] = out_host[2] = out_host[3] = 0;
  if (!out_host[0]) return QHP_OK;
  unsigned long long *cnt = (unsigned long long *)&s->counters[3];
  QHP_CUDA_OK(s, cudaMemsetAsync(cnt, 0, sizeof(int64_t), s->stream));
  StagedArgs a{};
  int rc = staged_args(s, a, nullptr, cnt, 0);
  if (rc) return rc;
  rc = pair_dense_forces(s, a, 0, s->Pc, true);
  if (rc) return rc;
  long long hits = 0, entries = 0;
  std::vector<long long> np(s->Pc);
  QHP_CUDA_OK(s, cudaMemcpyAsync(&hits, cnt, sizeof(long long), cudaMemcpyDeviceToHost, s->stream));
  QHP_CUDA_OK(s, cudaMemsetAsync(cnt, 0, sizeof(int64_t), s->stream));
  k_sum_counts<<<296, 256, 0, s->stream>>>(s->nbr_count_p, (long long)s->Pc * s->N, cnt);
  QHP_LAUNCH_OK(s);
  QHP_CUDA_OK(s, cudaMemcpyAsync(&entries, cnt, sizeof(long long), cudaMemcpyDeviceToHost, s->stream));
  QHP_CUDA_OK(s, cudaMemcpyAsync(np.data(), s->pruned_at + s->Pc, sizeof(long long) * s->Pc, cudaMemcpyDeviceToHost, s->stream));
  QHP_CUDA_OK(s, cudaStreamSynchronize(s->stream));
  out_host[1] = 0;
  for (long long v : np) out_host[1] += v;
  out_host[2] = entries;
  out_host[3] = hits;
  return QHP_OK;
}
