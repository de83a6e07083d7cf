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
// Per atom i (one warp):
//   check   32 list entries at a time: fp32 distance test on a float4 copy (conservative margin,
//           it only rejects pairs that are certainly outside r_c), ballot compaction of the
//           survivors into a per-warp queue;
//   eval    whenever the queue holds >= 32 survivors: all 32 lanes evaluate one pair each in fp64
//           (exact r^2 < r_c^2 test, LJ + damped-shifted-force Coulomb); no lane idles on the
//           cutoff, which cost 41 % of the lanes before.
// The DSF radial function needs no erfc/exp: with w = (alpha r)^2,
//   erfc(x) + (2x/sqrt(pi)) e^{-x^2} = 1 - x^3 S(w),   erfc(x)/x = 1/x - E(w),
// S and E entire in w, so F/r = qq (1/r^3 - alpha^3 S(w) - fshift/r) with 1/r from one rsqrt and
// alpha^3 S a degree-15 polynomial in u = 2 r^2/r_c^2 - 1 whose coefficients (fitted at create time
// from the Taylor series of S, qhp_pair_setup) sit in the kernel's constant bank.
// Full list (each ordered pair evaluated from its own side): no atomics, fixed summation order.
#include <math.h>

#include "qhp_internal.cuh"

#ifndef STG_THREADS
#define STG_THREADS 896           // largest CTA (28 warps, 68 registers); the host launches fewer warps when shared memory is short
#endif
#define STG_MAX_WARPS (STG_THREADS / 32)
#define STG_BLOCK 256             // list entries per row block (8 per lane)
#define STG_QUEUE (STG_BLOCK + 32)

struct StagedArgs {
  int N, Pc, nt, split, cap;
  int nc[3];
  double box[3], inv_box[3], cell_edge[3];
  const double *pos4;            // [Pc][N] (x, y, z, type bits), slot order
  double *Fs;                    // [Pc][N][3]
  const uint16_t *nbr16;         // [N][stride] indices into the staged array of the row's cell (blocked, see below)
  const int32_t *nbr_count, *cell_start;
  long long stride;
  const double *pair_tab;        // [nt*nt][4] = qq, 4 eps, sigma^2, LJ shift
  double rc, rc2, u_scale, fshift, erfc_rc;
  float rc2f;
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

// Row layout of the 16-bit table (written by k_list_build16, cells.cu): the entry of rank `pos` in a
// row sits at (pos / 256) * 256 + (pos % 32) * 8 + (pos % 256) / 32, i.e. one 16-byte load per lane
// brings entries pos = 256 m + 32 j + lane, j = 0..7; rows are padded with index 0 up to a multiple
// of 256 entries.
// F32: with the float4 copy for the fp32 pre-test (40 B per staged atom).  !F32: neighbourhoods too
// large for that stage fp64 positions + an int type only (28 B per atom) and pre-test in fp64.
template <bool ENERGY, bool F32>
__global__ void __launch_bounds__(STG_THREADS, 1) k_pair_staged(const StagedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *sp = reinterpret_cast<double *>(smem_raw);                  // [cap][3] fp64, cell-centred
  float4 *sf = reinterpret_cast<float4 *>(sp + 3 * (size_t)a.cap);    // F32: [cap] fp32 copy + type bits
  int *st = reinterpret_cast<int *>(sp + 3 * (size_t)a.cap);          // !F32: [cap] types
  double *tab = F32 ? reinterpret_cast<double *>(sf + a.cap) : reinterpret_cast<double *>(st + a.cap);
  uint32_t *queue = reinterpret_cast<uint32_t *>(tab + QHP_MAX_TYPES * QHP_MAX_TYPES * 4);
  __shared__ int off[28], cbeg[27], next_atom;
  __shared__ double su[STG_MAX_WARPS];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x;
  const int cell = blockIdx.x / a.split, part = blockIdx.x % a.split, bead = blockIdx.y;
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);

  for (int k = tid; k < a.nt * a.nt * 4; k += nthr) tab[k] = a.pair_tab[k];
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
  if (total > a.cap) {                       // cannot happen after the host-side capacity check
    if (tid == 0) a.counters[7] = 1;
    return;
  }
  // ---- stage the neighbourhood in coordinates relative to the cell centre ------------------------
  const double ctr[3] = {(cx + 0.5) * a.cell_edge[0], (cy + 0.5) * a.cell_edge[1], (cz + 0.5) * a.cell_edge[2]};
  const double4 *pos = reinterpret_cast<const double4 *>(a.pos4) + (long long)bead * a.N;
  for (int g = tid, s = 0; g < total; g += nthr) {
    while (g >= off[s + 1]) ++s;
    const double4 p = pos[cbeg[s] + g - off[s]];
    double lx = p.x - ctr[0], ly = p.y - ctr[1], lz = p.z - ctr[2];
    lx = fma(-a.box[0], rint(lx * a.inv_box[0]), lx);
    ly = fma(-a.box[1], rint(ly * a.inv_box[1]), ly);
    lz = fma(-a.box[2], rint(lz * a.inv_box[2]), lz);
    sp[3 * g] = lx; sp[3 * g + 1] = ly; sp[3 * g + 2] = lz;
    if (F32) sf[g] = make_float4((float)lx, (float)ly, (float)lz, __int_as_float((int)__double_as_longlong(p.w)));
    else st[g] = (int)__double_as_longlong(p.w);
  }
  __syncthreads();

  const int h0 = off[13], nh = off[14] - off[13], slot0 = cbeg[13];
  uint32_t *ql = queue + warp * STG_QUEUE + lane;          // this lane's view of the warp's queue
  unsigned lt = (1u << lane) - 1u;
  asm volatile("" : "+l"(ql), "+r"(lt));                   // keep both in registers (ptxas would recompute them per use)
  double U = 0.0;
  unsigned long long hits = 0;

  // Atoms of the home cell are handed to the warps dynamically (the CTAs of one cell take the atoms
  // ii = part, part + split, ...); each atom is summed by one warp in a fixed order, so the result
  // does not depend on which warp took it.  The next row block -- of this row or of the next atom's
  // row -- is in flight while the current one is processed.
  auto grab = [&]() {
    int t = 0;
    if (lane == 0) t = atomicAdd(&next_atom, 1);
    return part + a.split * __shfl_sync(0xffffffffu, t, 0);
  };
  auto load_block = [&](int ii, int m) {
    return *reinterpret_cast<const uint4 *>(a.nbr16 + (slot0 + ii) * a.stride + STG_BLOCK * m + 8 * lane);
  };

  int ii = grab();
  int n = (ii < nh) ? a.nbr_count[slot0 + ii] : 0;
  uint4 cur = make_uint4(0u, 0u, 0u, 0u), nxt = cur;
  if (ii < nh && n > 0) cur = load_block(ii, 0);
  int ii_n = grab();
  int n_n = (ii_n < nh) ? a.nbr_count[slot0 + ii_n] : 0;

  while (ii < nh) {
    const int ei = h0 + ii;
    const long long slot = slot0 + ii;
    const float4 fi = F32 ? sf[ei] : make_float4(0.f, 0.f, 0.f, 0.f);
    const double xi = sp[3 * ei], yi = sp[3 * ei + 1], zi = sp[3 * ei + 2];
    const double *tab_i = tab + (F32 ? __float_as_int(fi.w) : st[ei]) * a.nt * 4;
    double Fx = 0.0, Fy = 0.0, Fz = 0.0;
    int qn = 0;

    // one pair per lane, fp64: LJ + damped-shifted-force Coulomb (oracle O3)
    auto eval = [&](uint32_t entry, bool active) {
      const double *pj = sp + 3 * (entry & 0xffffu);
      const double *pt = tab_i + 4 * (entry >> 16);
      const double dx = xi - pj[0], dy = yi - pj[1], dz = zi - pj[2];
      const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
      const bool in = active && r2 < a.rc2;          // the fp64 test decides
      const double r2s = in ? r2 : a.rc2;
      const double qq = pt[0], eps4 = pt[1];
      const double y = rsqrt_seeded(r2s), y2 = y * y, y3 = y2 * y;
      const double u = fma(r2s, a.u_scale, -1.0);
      double fr = qq * fma(-a.fshift, y, y3 - poly_eval(a.cS, u));
      double s6 = 0.0;
      if (__any_sync(0xffffffffu, eps4 != 0.0)) {
        const double s2 = pt[2] * y2;
        s6 = s2 * s2 * s2;
        fr = fma(6.0 * eps4 * y2, fma(2.0 * s6, s6, -s6), fr);
      }
      fr = in ? fr : 0.0;
      Fx = fma(fr, dx, Fx); Fy = fma(fr, dy, Fy); Fz = fma(fr, dz, Fz);
      if (ENERGY) {
        const double r = r2s * y;
        const double up = qq * (y - poly_eval(a.cE, u) - a.erfc_rc + a.fshift * (r - a.rc)) + eps4 * (s6 * s6 - s6) - pt[3];
        U += in ? up : 0.0;
        hits += in ? 1ull : 0ull;
      }
    };

    for (int m = 0; STG_BLOCK * m < n; ++m) {
      if (STG_BLOCK * (m + 1) < n) nxt = load_block(ii, m + 1);
      else if (ii_n < nh && n_n > 0) nxt = load_block(ii_n, 0);
      // ---- check: fp32 pre-test of 8 x 32 entries, survivors compacted into the queue ----------------
      const int left = n - STG_BLOCK * m - lane;           // entry j of this lane is real iff 32 j < left
      const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (32 * j >= n - STG_BLOCK * m) break;            // warp-uniform: the row ends before this step
        const uint32_t e = (j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu);
        bool hit;
        uint32_t tj;
        if (F32) {
          const float4 pj = sf[e];
          const float dxf = fi.x - pj.x, dyf = fi.y - pj.y, dzf = fi.z - pj.z;
          const float r2f = fmaf(dzf, dzf, fmaf(dyf, dyf, dxf * dxf));
          hit = (32 * j < left) && r2f < a.rc2f;
          tj = (uint32_t)__float_as_int(pj.w);
        } else {
          const double *pj = sp + 3 * e;
          const double dx = xi - pj[0], dy = yi - pj[1], dz = zi - pj[2];
          hit = (32 * j < left) && fma(dz, dz, fma(dy, dy, dx * dx)) < a.rc2;
          tj = (uint32_t)st[e];
        }
        const unsigned mask = __ballot_sync(0xffffffffu, hit);
        if (hit) ql[qn + __popc(mask & lt) - lane] = e | (tj << 16);
        qn += __popc(mask);
      }
      __syncwarp();
      // ---- eval: full warps of survivors ---------------------------------------------------------------
      while (qn >= 32) {
        qn -= 32;
        eval(ql[qn], true);
      }
      __syncwarp();
      cur = nxt;
    }
    if (qn > 0) {
      const bool act = lane < qn;
      eval(act ? ql[0] : (uint32_t)ei, act);
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
    if (n == 0 && ii_n < nh && n_n > 0) cur = load_block(ii_n, 0);   // nothing was prefetched for an empty row
    ii = ii_n; n = n_n;
    ii_n = grab();
    n_n = (ii_n < nh) ? a.nbr_count[slot0 + ii_n] : 0;
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

static size_t staged_atom_bytes(bool f32) { return 3 * sizeof(double) + (f32 ? sizeof(float4) : sizeof(int)); }
static size_t staged_smem_bytes(int cap, int warps, bool f32) {
  return (size_t)cap * staged_atom_bytes(f32) + 16 + sizeof(double) * QHP_MAX_TYPES * QHP_MAX_TYPES * 4 +
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
  const long long need = region + region / 16 + 32;
  // first choice: the fp32 pre-test copy with the largest CTA; then the same CTA sizes without the copy
  for (int f32 = 1; f32 >= 0; --f32)
    for (int w : tries) {
      if (w > STG_MAX_WARPS) continue;
      const long long room = (long long)s->staged_smem_max - (long long)staged_smem_bytes(0, w, f32 != 0);
      long long cap = room / (long long)staged_atom_bytes(f32 != 0);
      if (cap > 65534) cap = 65534;                                    // 16-bit list entries
      cap &= ~3LL;                                                     // keeps the arrays behind the positions aligned
      if (cap >= need) { s->staged_warps = w; s->staged_cap = (int)cap; s->staged_f32 = f32 != 0; return true; }
      if (f32 && w == STG_MAX_WARPS) break;                            // a smaller CTA is worse than dropping the copy
    }
  return false;
}

int qhp_pair_staged_forces(qhp_system *s, bool energy, double *part, unsigned long long *count) {
  StagedArgs a{};
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
    // fp32 pre-test margin: 4x a bound on the fp32 error of r^2 (two roundings of coordinates up to
    // 1.5 cell edges + skin, one of each difference, three of the sum of squares)
    double cmax = 0.0;
    for (int d = 0; d < 3; ++d) cmax = fmax(cmax, 1.5 * a.cell_edge[d] + s->skin + 1.0);
    const double err = 2.0 * sqrt(3.0) * rc * (cmax * ldexp(1.0, -23) + rc * ldexp(1.0, -24)) + 4.0 * ldexp(1.0, -24) * rc * rc;
    a.rc2f = (float)(rc * rc + 4.0 * err) * (1.0f + 1.2e-7f);
  }
  for (int k = 0; k < QHP_NPOLY; ++k) { a.cS[k] = s->polyS[k]; a.cE[k] = s->polyE[k]; }
  a.part = part; a.count = count; a.counters = (long long *)s->counters;
  const dim3 grid((unsigned)(s->ncell * s->staged_split), (unsigned)s->Pc);
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
