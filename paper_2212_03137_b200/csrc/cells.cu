// cells.cu -- neighbour objects on the centroids (lists are
// "computed with respect to centroid positions" and shared by all beads).
//
// Canonical integer objects (bit-exact contract with the oracle):
//   nc[d]      = max(1, floor(L_d / r_list)),  r_list = r_cut + skin
//   cell_of[a] : s = c*(1/L); s -= floor(s); q = min((int)(s*nc), nc-1); cell = (qx*ncy + qy)*ncz + qz
//   order[]    = atoms stably sorted by cell (ties by atom index); cell_start[] = prefix sums
//   pair set   = {(i,j): mol_i != mol_j, d2 < r_list^2}, dx = fma(-L, rint(dx*(1/L)), dx),
//                d2 = fma(dz,dz, fma(dy,dy, dx*dx))
// All floating-point steps that decide an integer use explicit _rn intrinsics so that nvcc's FMA
// contraction cannot change them.
//
// The list is a fixed-stride table nbr[slot][k] in SLOT space (slot = position in `order`), built by
// one warp per slot scanning the 27-cell stencil with ballot compaction (deterministic order).
// Every kernel of the rebuild chain returns at once unless the integrator's list-validity statistic
// max |xc - cref|^2 reached (skin/2)^2, so the chain can be enqueued every step without a host sync.
#include <cooperative_groups.h>

#include "qhp_internal.cuh"
#include "contract.cuh"

struct CellArgs {
  int N, nc[3], ncell;
  double box[3], inv_box[3], rl2;
  float boxf[3], inv_boxf[3], edgef[3], rl2_lo, rl2_hi;   // fp32 pre-test: d2f < lo surely inside, >= hi surely outside
  const unsigned long long *flag;
  double thresh2;
};

__device__ __forceinline__ bool cells_skip(const CellArgs &a) {
  return a.flag && __longlong_as_double((long long)*a.flag) < a.thresh2;
}

// Order INSIDE a cell (internal slot order only; the canonical `order` of the parity hook breaks ties by atom index):
// 9-bit Morton code of the atom's position within its cell (8 x 8 x 8 sub-cells), then atom index.  Atoms that are
// neighbours in space become neighbours in slot order, so the staged records a warp of the pair kernel gathers for
// one atom come in runs of consecutive 16-byte records instead of scattered ones (shared-memory bank conflicts).
__device__ __forceinline__ int cell_subkey(double fx, double fy, double fz) {   // fractions in [0, 1)
  const int a = min((int)(fx * 8.0), 7), b = min((int)(fy * 8.0), 7), c = min((int)(fz * 8.0), 7);
  int k = 0;
#pragma unroll
  for (int bit = 0; bit < 3; ++bit) k |= (((a >> bit) & 1) << (3 * bit + 2)) | (((b >> bit) & 1) << (3 * bit + 1)) | (((c >> bit) & 1) << (3 * bit));
  return k;
}

__global__ void k_cells_assign(const CellArgs a, const double *__restrict__ Q0, int32_t *cell_of, int32_t *cell_count, int32_t *cell_key) {
  if (cells_skip(a)) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.N) return;
  int q[3];
  double fr[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double s = __dmul_rn(Q0[3LL * i + d], a.inv_box[d]);
    s = __dsub_rn(s, floor(s));
    const double sn = __dmul_rn(s, (double)a.nc[d]);
    int v = (int)sn;
    if (v > a.nc[d] - 1) v = a.nc[d] - 1;
    q[d] = v;
    fr[d] = fmin(fmax(sn - v, 0.0), 0.999999);
  }
  const int cell = (q[0] * a.nc[1] + q[1]) * a.nc[2] + q[2];
  cell_of[i] = cell;
  cell_key[i] = cell_subkey(fr[0], fr[1], fr[2]);
  atomicAdd(&cell_count[cell], 1);
}

// single-CTA exclusive scan of n ints -> out[0..n]; optionally copies to out2 and zeroes `in`
__global__ void k_scan_excl(const CellArgs a, int32_t *in, int32_t *out, int32_t *out2, int n, int zero_in) {
  if (cells_skip(a)) return;
  __shared__ int32_t part[1024];
  const int t = threadIdx.x, nt = blockDim.x;
  const int len = (n + nt - 1) / nt;
  const int b = min(n, t * len), e = min(n, b + len);
  int32_t s = 0;
  for (int k = b; k < e; ++k) s += in[k];
  part[t] = s;
  __syncthreads();
  // Hillis-Steele inclusive scan over the per-thread sums
  for (int o = 1; o < nt; o <<= 1) {
    int32_t v = (t >= o) ? part[t - o] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int32_t run = part[t] - s;
  for (int k = b; k < e; ++k) {
    const int32_t v = in[k];
    out[k] = run;
    if (out2) out2[k] = run;
    if (zero_in) in[k] = 0;
    run += v;
  }
  if (t == nt - 1) { out[n] = part[t]; if (out2) out2[n] = part[t]; }
}

__global__ void k_cells_fill(const CellArgs a, const int32_t *__restrict__ cell_of, int32_t *cursor, int32_t *tmp) {
  if (cells_skip(a)) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.N) return;
  tmp[atomicAdd(&cursor[cell_of[i]], 1)] = i;
}

// stable order inside each cell: slot = cell_start + #{members with a smaller atom index}
// key == NULL: the canonical order (ties by atom index; parity hook), rank may be NULL then
__global__ void k_cells_rank(const CellArgs a, const int32_t *__restrict__ cell_of, const int32_t *__restrict__ cell_start,
                             const int32_t *__restrict__ tmp, const int32_t *__restrict__ key, int32_t *order, int32_t *rank) {
  if (cells_skip(a)) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.N) return;
  const int c = cell_of[i], b = cell_start[c], e = cell_start[c + 1];
  const int ki = key ? key[i] : 0;
  int cnt = 0;
  for (int k = b; k < e; ++k) {
    const int j = tmp[k], kj = key ? key[j] : 0;
    cnt += (kj < ki) || (kj == ki && j < i);
  }
  order[b + cnt] = i;
  if (rank) rank[i] = b + cnt;
}

// Is slot k a list neighbour of the slot whose centroid is ci / fi?  The decision is the canonical
// fp64 one (O4); an fp32 pre-test on wrapped single-precision copies settles every pair that is not
// within the fp32 error of r_list, so only a thin shell pays for the fp64 arithmetic.
__device__ __forceinline__ bool list_hit_exact(const CellArgs &a, const double *__restrict__ cent4, const double4 &ci, int k) {
  const double4 cj = reinterpret_cast<const double4 *>(cent4)[k];
  double dx = __dsub_rn(ci.x, cj.x), dy = __dsub_rn(ci.y, cj.y), dz = __dsub_rn(ci.z, cj.z);
  dx = __fma_rn(-a.box[0], rint(__dmul_rn(dx, a.inv_box[0])), dx);
  dy = __fma_rn(-a.box[1], rint(__dmul_rn(dy, a.inv_box[1])), dy);
  dz = __fma_rn(-a.box[2], rint(__dmul_rn(dz, a.inv_box[2])), dz);
  return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx))) < a.rl2;
}
__device__ __forceinline__ bool list_hit(const CellArgs &a, const double *__restrict__ cent4, const float4 *__restrict__ centf,
                                         const double4 &ci, const float4 &fi, int k) {
  const float4 fj = centf[k];
  if (((__float_as_int(fj.w) ^ __float_as_int(fi.w)) & 0x0fffffff) == 0) return false;   // same molecule (bits 28-30: type)
  float fx = fi.x - fj.x, fy = fi.y - fj.y, fz = fi.z - fj.z;
  fx = fmaf(-a.boxf[0], rintf(fx * a.inv_boxf[0]), fx);
  fy = fmaf(-a.boxf[1], rintf(fy * a.inv_boxf[1]), fy);
  fz = fmaf(-a.boxf[2], rintf(fz * a.inv_boxf[2]), fz);
  const float d2f = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
  if (d2f < a.rl2_lo) return true;
  if (d2f >= a.rl2_hi) return false;
  return list_hit_exact(a, cent4, ci, k);
}

// one warp per slot (row i of the table); nbr == NULL: count only
__device__ __forceinline__ void list_row32(const CellArgs &a, const double *__restrict__ cent4, const int32_t *__restrict__ cell_of,
                                           const int32_t *__restrict__ order, const int32_t *__restrict__ cell_start, int32_t *nbr,
                                           int32_t *nbr_count, long long stride, long long *counters, long long i, int lane) {
  const float4 *centf = reinterpret_cast<const float4 *>(cent4 + 4LL * a.N);   // fp32 copies live behind cent4
  const double4 ci = reinterpret_cast<const double4 *>(cent4)[i];
  const float4 fi = centf[i];
  const int cell = cell_of[order[i]];
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);
  const int nox = min(a.nc[0], 3), noy = min(a.nc[1], 3), noz = min(a.nc[2], 3);
  const int sx = a.nc[0] >= 3 ? -1 : 0, sy = a.nc[1] >= 3 ? -1 : 0, sz = a.nc[2] >= 3 ? -1 : 0;
  const unsigned lt = (1u << lane) - 1u;
  int cnt = 0;
  for (int ox = 0; ox < nox; ++ox)
    for (int oy = 0; oy < noy; ++oy)
      for (int oz = 0; oz < noz; ++oz) {
        const int qx = (cx + sx + ox + a.nc[0]) % a.nc[0], qy = (cy + sy + oy + a.nc[1]) % a.nc[1],
                  qz = (cz + sz + oz + a.nc[2]) % a.nc[2];
        const int c2 = (qx * a.nc[1] + qy) * a.nc[2] + qz;
        const int b = cell_start[c2], e = cell_start[c2 + 1];
        for (int k0 = b; k0 < e; k0 += 32) {
          const int k = k0 + lane;
          bool hit = false;
          if (k < e && k != i) hit = list_hit(a, cent4, centf, ci, fi, k);
          const unsigned mask = __ballot_sync(0xffffffffu, hit);
          if (hit && nbr) {
            const int pos = cnt + __popc(mask & lt);
            if (pos < stride) nbr[i * stride + pos] = k;
          }
          cnt += __popc(mask);
        }
      }
  if (lane == 0) {
    if (nbr) {
      nbr_count[i] = (int)min((long long)cnt, stride);
      if (cnt > stride) counters[1] = 1;
    } else {
      nbr_count[i] = cnt;
    }
    atomicMax((unsigned long long *)&counters[2], (unsigned long long)cnt);
  }
}

__global__ void __launch_bounds__(256) k_list_build(const CellArgs a, const double *__restrict__ cent4,
                                                    const int32_t *__restrict__ cell_of, const int32_t *__restrict__ order,
                                                    const int32_t *__restrict__ cell_start, int32_t *nbr,
                                                    int32_t *nbr_count, long long stride, long long *counters) {
  if (cells_skip(a)) return;
  const int lane = threadIdx.x & 31;
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= a.N) return;
  if (i == 0 && lane == 0 && nbr) counters[0] += 1;
  list_row32(a, cent4, cell_of, order, cell_start, nbr, nbr_count, stride, counters, i, lane);
}

// Same pair set, written as 16-bit indices into the staged array of the row's cell (pair_staged.cu):
// index = (number of atoms in the stencil cells before this one, in the stencil order below) + (k - b).
// Requires nc >= 4 in every dimension (27 distinct stencil cells).
template <bool FILL>
__device__ __forceinline__ void list_row16(const CellArgs &a, const double *__restrict__ cent4,
                                           const int32_t *__restrict__ cell_of, const int32_t *__restrict__ order,
                                           const int32_t *__restrict__ cell_start, uint16_t *nbr,
                                           int32_t *nbr_count, int stride, int dummy, long long *counters, int i, int lane) {
  const float4 *centf = reinterpret_cast<const float4 *>(cent4 + 4LL * a.N);   // fp32 copies live behind cent4
  const double4 ci = reinterpret_cast<const double4 *>(cent4)[i];
  const float4 fi = centf[i];
  const int wi = __float_as_int(fi.w) & 0x0fffffff;     // molecule id (bits 28-30 hold the atom type)
  const int cell = cell_of[order[i]];
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);
  unsigned lt = (1u << lane) - 1u;
  uint16_t *row = nbr + (long long)i * stride;
  float lo = a.rl2_lo, hi = a.rl2_hi;
  asm volatile("" : "+r"(lt), "+l"(row));
  int cnt = 0, off = 0;
  // The 27 stencil cells are walked as 9 (x, y) columns.  The three cells of a column are adjacent in z,
  // hence contiguous in slot order unless the column wraps around the box: they are scanned as one run
  // (fewer ragged 32-candidate chunks, one set of per-run constants).  A cell whose box is out of reach
  // of this centroid is dropped from its run (the margin of rl2_hi covers the fp32 rounding).  The
  // image of a neighbour cell next to the home cell is known per cell: with >= 4 cells per dimension it
  // is the minimum image of every pair within r_list, so the fp32 pre-test needs no rint.
  const float gzl = fmaxf(fi.z - cz * a.edgef[2], 0.f), gzh = fmaxf((cz + 1) * a.edgef[2] - fi.z, 0.f);
  for (int ox = 0; ox < 3; ++ox) {
    const int ux = cx - 1 + ox, qx = ux < 0 ? ux + a.nc[0] : (ux >= a.nc[0] ? ux - a.nc[0] : ux);
    const float px0 = fi.x - (ux < 0 ? -a.boxf[0] : (ux >= a.nc[0] ? a.boxf[0] : 0.f));
    const float hx = ox == 0 ? fmaxf(fi.x - cx * a.edgef[0], 0.f) : (ox == 2 ? fmaxf((cx + 1) * a.edgef[0] - fi.x, 0.f) : 0.f);
    for (int oy = 0; oy < 3; ++oy) {
      const int uy = cy - 1 + oy, qy = uy < 0 ? uy + a.nc[1] : (uy >= a.nc[1] ? uy - a.nc[1] : uy);
      const float py0 = fi.y - (uy < 0 ? -a.boxf[1] : (uy >= a.nc[1] ? a.boxf[1] : 0.f));
      const float hy = oy == 0 ? fmaxf(fi.y - cy * a.edgef[1], 0.f) : (oy == 2 ? fmaxf((cy + 1) * a.edgef[1] - fi.y, 0.f) : 0.f);
      const float gxy = fmaf(hy, hy, hx * hx);
      const int cb = (qx * a.nc[1] + qy) * a.nc[2];
      int bq[3], eq[3];
      float sz[3];
      bool reach[3];
#pragma unroll
      for (int oz = 0; oz < 3; ++oz) {
        const int uz = cz - 1 + oz, qz = uz < 0 ? uz + a.nc[2] : (uz >= a.nc[2] ? uz - a.nc[2] : uz);
        bq[oz] = cell_start[cb + qz]; eq[oz] = cell_start[cb + qz + 1];
        sz[oz] = uz < 0 ? -a.boxf[2] : (uz >= a.nc[2] ? a.boxf[2] : 0.f);
        const float hz = oz == 0 ? gzl : (oz == 2 ? gzh : 0.f);
        reach[oz] = fmaf(hz, hz, gxy) < a.rl2_hi;
      }
      int oz = 0;
      while (oz < 3) {
        if (!reach[oz]) { off += eq[oz] - bq[oz]; ++oz; continue; }
        const int b = bq[oz];
        int e = eq[oz], oz2 = oz + 1, idx0 = off - b;           // staged index of slot k = idx0 + k
        float px = px0, py = py0, pz = fi.z - sz[oz];
        off += eq[oz] - bq[oz];
        while (oz2 < 3 && reach[oz2] && bq[oz2] == e && sz[oz2] == sz[oz]) { e = eq[oz2]; off += eq[oz2] - bq[oz2]; ++oz2; }
        // the inner loop decides the run time of a rebuild: keep its invariants in registers (ptxas
        // otherwise re-derives the image shifts and reloads the thresholds every iteration)
        asm volatile("" : "+f"(px), "+f"(py), "+f"(pz), "+f"(lo), "+f"(hi), "+r"(idx0), "+r"(e));
        const int last = e - 1;
        for (int k = b + lane; k - lane < e; k += 32) {
          const float4 fj = centf[min(k, last)];
          const float dxf = px - fj.x, dyf = py - fj.y, dzf = pz - fj.z;
          const float d2f = fmaf(dzf, dzf, fmaf(dyf, dyf, dxf * dxf));
          const int wj = __float_as_int(fj.w);
          bool hit = (k <= last) & (k != i) & ((wj & 0x0fffffff) != wi) & (d2f < hi);
          if (hit && !(d2f < lo)) hit = list_hit_exact(a, cent4, ci, k);      // the thin shell around r_list
          const unsigned mask = __ballot_sync(0xffffffffu, hit);
          if (FILL && hit) {
            const int pos = cnt + __popc(mask & lt);
            if (pos < stride) row[(pos & ~255) + ((pos & 31) << 3) + ((pos & 255) >> 5)] = (uint16_t)((idx0 + k) | ((wj >> 28) << 13));
          }
          cnt += __popc(mask);
        }
        oz = oz2;
      }
    }
  }
  if (FILL) {
    // pad the last 32-entry step with the dummy staged index (pair_staged.cu: no pre-test against it passes)
    const int n = min(cnt, stride), end = min((n + 31) & ~31, stride);
    for (int pos = n + lane; pos < end; pos += 32)
      row[(pos & ~255) + ((pos & 31) << 3) + ((pos & 255) >> 5)] = (uint16_t)dummy;
  }
  if (lane == 0) {
    if (FILL) {
      nbr_count[i] = min(cnt, stride);
      if (cnt > stride) counters[1] = 1;
    } else {
      nbr_count[i] = cnt;
    }
    atomicMax((unsigned long long *)&counters[2], (unsigned long long)cnt);
    atomicMax((unsigned long long *)&counters[5], (unsigned long long)off);   // staged-region size
  }
}

template <bool FILL>
__global__ void __launch_bounds__(256) k_list_build16(const CellArgs a, const double *__restrict__ cent4,
                                                      const int32_t *__restrict__ cell_of, const int32_t *__restrict__ order,
                                                      const int32_t *__restrict__ cell_start, uint16_t *nbr,
                                                      int32_t *nbr_count, int stride, int dummy, long long *counters) {
  if (cells_skip(a)) return;
  const int lane = threadIdx.x & 31;
  const int i = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (i >= a.N) return;
  if (i == 0 && lane == 0 && FILL) counters[0] += 1;
  list_row16<FILL>(a, cent4, cell_of, order, cell_start, nbr, nbr_count, stride, dummy, counters, i, lane);
}

// ---- export in atom indices (parity hook) ---------------------------------------------------------
__global__ void k_export_count(int N, const int32_t *__restrict__ order, const int32_t *__restrict__ nbr_count, int32_t *count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) count[order[i]] = nbr_count[i];
}
__global__ void k_export_fill(int N, const int32_t *__restrict__ order, const int32_t *__restrict__ nbr_count,
                              const int32_t *__restrict__ nbr, long long stride, const int32_t *__restrict__ start,
                              int32_t *out, long long cap) {
  const int lane = threadIdx.x & 31;
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const int a = order[i], n = nbr_count[i];
  const long long s0 = start[a];
  for (int k = lane; k < n; k += 32)
    if (s0 + k < cap) out[s0 + k] = order[nbr[i * stride + k]];
}

// staged format: translate the 16-bit staged index back to a slot, then to an atom
__global__ void k_export_fill16(const CellArgs a, const int32_t *__restrict__ cell_of, const int32_t *__restrict__ order,
                                const int32_t *__restrict__ cell_start, const int32_t *__restrict__ nbr_count,
                                const uint16_t *__restrict__ nbr, long long stride, const int32_t *__restrict__ start,
                                int32_t *out, long long cap) {
  const int lane = threadIdx.x & 31;
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= a.N) return;
  const int at = order[i], n = nbr_count[i];
  const int cell = cell_of[at];
  const int cz = cell % a.nc[2], cy = (cell / a.nc[2]) % a.nc[1], cx = cell / (a.nc[2] * a.nc[1]);
  int cb = 0, cn = 0;                       // lane s < 27: first slot and size of stencil cell s
  if (lane < 27) {
    const int ox = lane / 9, oy = (lane / 3) % 3, oz = lane % 3;
    const int qx = (cx - 1 + ox + a.nc[0]) % a.nc[0], qy = (cy - 1 + oy + a.nc[1]) % a.nc[1],
              qz = (cz - 1 + oz + a.nc[2]) % a.nc[2];
    const int c2 = (qx * a.nc[1] + qy) * a.nc[2] + qz;
    cb = cell_start[c2]; cn = cell_start[c2 + 1] - cb;
  }
  const long long s0 = start[at];
  for (int k0 = 0; k0 < n; k0 += 32) {
    const int k = k0 + lane;
    const int loc = k < n ? (int)(nbr[i * stride + (k & ~255) + ((k & 31) << 3) + ((k & 255) >> 5)] & 0x1fff) : 0;
    int off = 0, slot = -1;
    for (int s = 0; s < 27; ++s) {
      const int b = __shfl_sync(0xffffffffu, cb, s), c = __shfl_sync(0xffffffffu, cn, s);
      if (slot < 0 && loc < off + c) slot = b + loc - off;
      off += c;
    }
    if (k < n && s0 + k < cap) out[s0 + k] = order[slot];
  }
}

static CellArgs cell_args(qhp_system *s, bool force) {
  CellArgs a{};
  a.N = s->N; a.ncell = s->ncell;
  const double rl = s->r_cut + s->skin;
  for (int d = 0; d < 3; ++d) { a.nc[d] = s->nc[d]; a.box[d] = s->box[d]; a.inv_box[d] = s->inv_box[d]; }
  a.rl2 = rl * rl;
  {
    // bound on the fp32 error of d2: coordinates wrapped into [0, L) and the box edge are rounded to
    // fp32 (2^-24 relative each), the image count is at most 1; 4x safety
    double Lmax = 0.0;
    for (int d = 0; d < 3; ++d) { Lmax = fmax(Lmax, s->box[d]); a.boxf[d] = (float)s->box[d]; a.inv_boxf[d] = (float)s->inv_box[d]; a.edgef[d] = (float)(s->box[d] / s->nc[d]); }
    const double e = (5.0 * Lmax + rl) * ldexp(1.0, -24);
    const double m = 4.0 * (2.0 * sqrt(3.0) * rl * e + 4.0 * ldexp(1.0, -24) * a.rl2);
    a.rl2_lo = (float)(a.rl2 - m) * (1.0f - 1.2e-7f);
    a.rl2_hi = (float)(a.rl2 + m) * (1.0f + 1.2e-7f);
  }
  a.flag = force ? nullptr : &s->d2max[s->flag_idx];
  const double th = 0.5 * s->skin;
  a.thresh2 = th * th;
  return a;
}

// cells (assign, scan, fill, rank) of the current centroids Q_0
// The four cell kernels as one cooperative kernel (grid-wide barriers between the phases): inside
// qhp_step the chain is enqueued every step and returns at once unless a rebuild is due, so one launch
// instead of four takes 3 kernel boundaries off every step (they dominate the small boxes).
// Rest of the rebuild chain inside the same cooperative kernel (ra.on): contraction of the current modes into the
// new slot order (+ sorted centroids, fp32 copy, reference centroids) and the list build, its rows handed to the
// warps through a work counter -- one launch per step, which returns at once unless a rebuild is due.
struct RebuildArgs {
  int on, Pc, staged, stride, dummy;
  BoxArg bx;
  const double *Q, *Tc;
  const int32_t *type, *molid;
  double *pos4, *cent4, *cref;
  uint16_t *nbr16;
  int32_t *nbr;
  int32_t *nbr_count;
  long long stride32;
  long long *counters;           // [4] = work counter of the list phase
};
__global__ void __launch_bounds__(256) k_cells_fused(const CellArgs a, const double *__restrict__ Q0, int32_t *cell_of,
                                                     int32_t *cell_count, int32_t *cell_start, int32_t *cursor,
                                                     int32_t *tmp, int32_t *order, int32_t *rank, int32_t *cell_key, const RebuildArgs ra) {
  if (cells_skip(a)) return;                       // uniform over the grid: nobody reaches a barrier
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const int nthreads = gridDim.x * blockDim.x, t0 = blockIdx.x * blockDim.x + threadIdx.x;
  for (int i = t0; i < a.N; i += nthreads) {       // assign
    int q[3];
    double fr[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double sc = __dmul_rn(Q0[3LL * i + d], a.inv_box[d]);
      sc = __dsub_rn(sc, floor(sc));
      const double sn = __dmul_rn(sc, (double)a.nc[d]);
      int v = (int)sn;
      if (v > a.nc[d] - 1) v = a.nc[d] - 1;
      q[d] = v;
      fr[d] = fmin(fmax(sn - v, 0.0), 0.999999);
    }
    const int cell = (q[0] * a.nc[1] + q[1]) * a.nc[2] + q[2];
    cell_of[i] = cell;
    cell_key[i] = cell_subkey(fr[0], fr[1], fr[2]);
    atomicAdd(&cell_count[cell], 1);
  }
  grid.sync();
  if (blockIdx.x == 0) {                           // exclusive scan of the cell counts by one CTA
    __shared__ int32_t part[256];
    const int t = threadIdx.x, nt = blockDim.x, n = a.ncell;
    const int len = (n + nt - 1) / nt;
    const int b = min(n, t * len), e = min(n, b + len);
    int32_t sum = 0;
    for (int k = b; k < e; ++k) sum += cell_count[k];
    part[t] = sum;
    __syncthreads();
    for (int o = 1; o < nt; o <<= 1) {
      const int32_t v = (t >= o) ? part[t - o] : 0;
      __syncthreads();
      part[t] += v;
      __syncthreads();
    }
    int32_t run = part[t] - sum;
    for (int k = b; k < e; ++k) {
      const int32_t v = cell_count[k];
      cell_start[k] = run; cursor[k] = run; cell_count[k] = 0;
      run += v;
    }
    if (t == nt - 1) { cell_start[n] = part[t]; cursor[n] = part[t]; }
  }
  grid.sync();
  for (int i = t0; i < a.N; i += nthreads) tmp[atomicAdd(&cursor[cell_of[i]], 1)] = i;   // fill
  grid.sync();
  for (int i = t0; i < a.N; i += nthreads) {       // stable order inside each cell
    const int c = cell_of[i], b = cell_start[c], e = cell_start[c + 1], ki = cell_key[i];
    int cnt = 0;
    for (int k = b; k < e; ++k) {
      const int j = tmp[k], kj = cell_key[j];
      cnt += (kj < ki) || (kj == ki && j < i);
    }
    order[b + cnt] = i;
    rank[i] = b + cnt;
  }
  if (!ra.on) return;
  grid.sync();
  if (t0 == 0) { ra.counters[4] = 0; ra.counters[0] += 1; }
  for (long long d = t0; d < 3LL * a.N; d += nthreads)
    qhp_contract_dof(ra.bx, ra.Q, a.N, ra.Pc, ra.Tc, rank, ra.type, ra.molid, ra.pos4, ra.cent4, ra.cref, nullptr, 0,
                     a.thresh2, ra.counters, d);
  grid.sync();
  const int lane = threadIdx.x & 31;
  for (;;) {
    long long i = 0;
    if (lane == 0) i = (long long)atomicAdd((unsigned long long *)&ra.counters[4], 1ull);
    i = __shfl_sync(0xffffffffu, i, 0);
    if (i >= a.N) break;
    if (ra.staged) list_row16<true>(a, ra.cent4, cell_of, order, cell_start, ra.nbr16, ra.nbr_count, ra.stride, ra.dummy, ra.counters, (int)i, lane);
    else list_row32(a, ra.cent4, cell_of, order, cell_start, ra.nbr, ra.nbr_count, ra.stride32, ra.counters, i, lane);
  }
}

static int cells_only(qhp_system *s, const CellArgs &a, const RebuildArgs *fused = nullptr) {
  if (s->coop_blocks > 0) {
    const int tb = 256;
    int grid = (s->N + tb - 1) / tb;
    if (fused) grid = s->coop_blocks;                  // the list phase wants every resident warp
    if (grid > s->coop_blocks) grid = s->coop_blocks;
    CellArgs ac = a;
    const double *q0 = s->Q;
    RebuildArgs ra{};
    if (fused) ra = *fused;
    void *args[] = {&ac, &q0, &s->cell_of, &s->cell_count, &s->cell_start, &s->cell_cursor, &s->cell_tmp, &s->order, &s->rank, &s->cell_key, &ra};
    QHP_CUDA_OK(s, cudaLaunchCooperativeKernel((const void *)k_cells_fused, dim3(grid), dim3(tb), args, 0, s->stream));
    s->n_launch++;
    return QHP_OK;
  }
  const int tb = 256, grid = (s->N + tb - 1) / tb;
  k_cells_assign<<<grid, tb, 0, s->stream>>>(a, s->Q, s->cell_of, s->cell_count, s->cell_key);
  QHP_LAUNCH_OK(s);
  k_scan_excl<<<1, 1024, 0, s->stream>>>(a, s->cell_count, s->cell_start, s->cell_cursor, s->ncell, 1);
  QHP_LAUNCH_OK(s);
  k_cells_fill<<<grid, tb, 0, s->stream>>>(a, s->cell_of, s->cell_cursor, s->cell_tmp);
  QHP_LAUNCH_OK(s);
  k_cells_rank<<<grid, tb, 0, s->stream>>>(a, s->cell_of, s->cell_start, s->cell_tmp, s->cell_key, s->order, s->rank);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

static int list_build(qhp_system *s, const CellArgs &a, bool count_only) {
  const int tb = 256;
  const long long threads = 32LL * s->N;
  const unsigned grid = (unsigned)((threads + tb - 1) / tb);
  if (s->staged && count_only)
    k_list_build16<false><<<grid, tb, 0, s->stream>>>(a, s->cent4, s->cell_of, s->order, s->cell_start, nullptr, s->nbr_count,
                                                     (int)s->nbr_stride, s->staged_cap - 1, (long long *)s->counters);
  else if (s->staged)
    k_list_build16<true><<<grid, tb, 0, s->stream>>>(a, s->cent4, s->cell_of, s->order, s->cell_start, s->nbr16, s->nbr_count,
                                                    (int)s->nbr_stride, s->staged_cap - 1, (long long *)s->counters);
  else
    k_list_build<<<grid, tb, 0, s->stream>>>(a, s->cent4, s->cell_of, s->order, s->cell_start,
                                            count_only ? nullptr : s->nbr, s->nbr_count, s->nbr_stride,
                                            (long long *)s->counters);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_cells_rebuild(qhp_system *s, bool force) {
  const CellArgs a = cell_args(s, force);
  if (!force && s->coop_blocks > 0 && (s->staged ? s->nbr16 != nullptr : s->nbr != nullptr)) {
    // the per-step path: the whole chain (cells, contraction, list) as one cooperative launch
    RebuildArgs ra{};
    ra.on = 1; ra.Pc = s->Pc; ra.staged = s->staged ? 1 : 0; ra.stride = (int)s->nbr_stride; ra.dummy = s->staged_cap - 1;
    for (int d = 0; d < 3; ++d) { ra.bx.box[d] = s->box[d]; ra.bx.inv_box[d] = s->inv_box[d]; }
    ra.Q = s->Q; ra.Tc = s->d_Tc; ra.type = s->dt_.type; ra.molid = s->dt_.molid;
    ra.pos4 = s->pos4; ra.cent4 = s->cent4; ra.cref = s->cref;
    ra.nbr16 = s->nbr16; ra.nbr = s->nbr; ra.nbr_count = s->nbr_count; ra.stride32 = s->nbr_stride;
    ra.counters = (long long *)s->counters;
    return cells_only(s, a, &ra);
  }
  int rc = cells_only(s, a);
  if (rc) return rc;
  rc = qhp_nm_contract(s, true, force);
  if (rc) return rc;
  if (force) {
    // synchronising call sites only: size the fixed-stride table from a counting pass
    // the staged pair kernel serves the system if its geometry allows it (qhp_pair_setup) and the
    // densest 27-cell neighbourhood fits in shared memory with some room for drift between rebuilds
    s->staged = s->staged_ok;
    int64_t mx = 0, region_max = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
      QHP_CUDA_OK(s, cudaMemsetAsync(&s->counters[2], 0, sizeof(int64_t), s->stream));
      QHP_CUDA_OK(s, cudaMemsetAsync(&s->counters[5], 0, sizeof(int64_t), s->stream));
      rc = list_build(s, a, true);
      if (rc) return rc;
      int64_t region = 0;
      QHP_CUDA_OK(s, cudaMemcpyAsync(&mx, &s->counters[2], sizeof(int64_t), cudaMemcpyDeviceToHost, s->stream));
      QHP_CUDA_OK(s, cudaMemcpyAsync(&region, &s->counters[5], sizeof(int64_t), cudaMemcpyDeviceToHost, s->stream));
      QHP_CUDA_OK(s, cudaStreamSynchronize(s->stream));
      region_max = region;
      if (!s->staged || qhp_pair_staged_fit(s, region)) break;
      s->staged = false;                               // too dense: generic kernel and 32-bit list
    }
    const bool have = s->staged ? (s->nbr16 != nullptr) : (s->nbr != nullptr);
    if (!have || mx + 8 > s->nbr_stride) {
      int64_t stride = (int64_t)((double)mx * 1.4) + 32;
      stride = (stride + 255) / 256 * 256;                 // whole 256-entry row blocks (pair_staged.cu)
      if (stride < 4) stride = 4;
      if (s->nbr) cudaFree(s->nbr);
      if (s->nbr16) cudaFree(s->nbr16);
      s->nbr = nullptr; s->nbr16 = nullptr;
      s->nbr_stride = stride;
      const cudaError_t e = s->staged ? cudaMalloc(&s->nbr16, sizeof(uint16_t) * (size_t)stride * (size_t)s->N)
                                      : cudaMalloc(&s->nbr, sizeof(int32_t) * (size_t)stride * (size_t)s->N);
      if (e != cudaSuccess) {
        s->err = "neighbour table allocation failed";
        s->nbr = nullptr; s->nbr16 = nullptr;
        return QHP_ENOMEM;
      }
    }
    rc = qhp_pair_dense_prepare(s, region_max);          // pruned per-bead rows (pair_staged.cu): decide, allocate, mark stale
    if (rc) return rc;
  }
  return list_build(s, a, false);
}

int qhp_cells_export(qhp_system *s, int32_t *count, int32_t *nbr, int64_t cap, int64_t *total_host) {
  const int tb = 256;
  int32_t *start = nullptr;
  QHP_CUDA_OK(s, cudaMalloc(&start, sizeof(int32_t) * ((size_t)s->N + 1)));
  int32_t *cnt = count;
  int32_t *cnt_own = nullptr;
  if (!cnt) { QHP_CUDA_OK(s, cudaMalloc(&cnt_own, sizeof(int32_t) * (size_t)s->N)); cnt = cnt_own; }
  k_export_count<<<(s->N + tb - 1) / tb, tb, 0, s->stream>>>(s->N, s->order, s->nbr_count, cnt);
  QHP_LAUNCH_OK(s);
  CellArgs a{};
  a.flag = nullptr;
  k_scan_excl<<<1, 1024, 0, s->stream>>>(a, cnt, start, nullptr, s->N, 0);
  QHP_LAUNCH_OK(s);
  if (nbr) {
    const long long threads = 32LL * s->N;
    if (s->staged) {
      const CellArgs ca = cell_args(s, true);
      k_export_fill16<<<(unsigned)((threads + tb - 1) / tb), tb, 0, s->stream>>>(ca, s->cell_of, s->order, s->cell_start,
                                                                               s->nbr_count, s->nbr16, s->nbr_stride, start, nbr, cap);
    } else {
      k_export_fill<<<(unsigned)((threads + tb - 1) / tb), tb, 0, s->stream>>>(s->N, s->order, s->nbr_count, s->nbr,
                                                                             s->nbr_stride, start, nbr, cap);
    }
    QHP_LAUNCH_OK(s);
  }
  int32_t tot = 0;
  QHP_CUDA_OK(s, cudaMemcpyAsync(&tot, start + s->N, sizeof(int32_t), cudaMemcpyDeviceToHost, s->stream));
  QHP_CUDA_OK(s, cudaStreamSynchronize(s->stream));
  if (total_host) *total_host = tot;
  cudaFree(start);
  if (cnt_own) cudaFree(cnt_own);
  return QHP_OK;
}

// canonical order (cells, ties by atom index) of the current cell assignment into `order_out` (parity hook)
int qhp_cells_canonical_order(qhp_system *s, int32_t *order_out) {
  CellArgs a = cell_args(s, true);
  const int tb = 256, grid = (s->N + tb - 1) / tb;
  k_cells_rank<<<grid, tb, 0, s->stream>>>(a, s->cell_of, s->cell_start, s->cell_tmp, nullptr, order_out, nullptr);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

// cooperative launches need all CTAs resident: how many k_cells_fused CTAs fit on the device (0: unsupported)
int qhp_cells_setup(qhp_system *s) {
  int coop = 0, per_sm = 0, sms = 0;
  QHP_CUDA_OK(s, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, s->device));
  QHP_CUDA_OK(s, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device));
  s->coop_blocks = 0;
  if (!coop) return QHP_OK;
  QHP_CUDA_OK(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cells_fused, 256, 0));
  s->coop_blocks = per_sm * sms;
  return QHP_OK;
}

