// pair.cu -- bead-batched short-range pair forces V_s on the contracted beads (SURVEY.md §8(a) row
// R8; "the most time-consuming operation"; contraction PAPER.md:174-182 Eq. 20).
// Force field (BASELINE.json configs[0]): Lennard-Jones (Lorentz-Berthelot mixing, potential
// shifted to 0 at r_c) + damped-shifted-force Coulomb (Fennell-Gezelter), cutoff tested PER BEAD
// with the minimum image applied per bead pair (each bead is an independent periodic replica,
// PAPER.md:32); intramolecular pairs are excluded at list-build time.
//
// Work decomposition: a group of L lanes (4..32, inside one warp) owns one slot i and strides over
// its row of the centroid neighbour table; every list entry j is read ONCE and used for NB
// contracted beads (the list is shared by all beads); the L partial forces are
// combined with warp shuffles and lane 0 of the group stores F_i.  Full list (each ordered pair is
// evaluated from both sides): no atomics, deterministic summation order, fp64 throughout.
#include "qhp_internal.cuh"

struct PairArgs {
  int N, Pc, nt;
  int bead0, bead_end;      // this launch evaluates the contracted beads [bead0, bead_end)
  const double *pos4;       // [Pc][N] (x, y, z, type bits)
  double *Fs;               // [Pc][N][3]
  const int32_t *nbr, *nbr_count;
  long long stride;
  const double *pair_tab;   // [nt*nt][4] = qq, 4 eps, sigma^2, LJ shift
  double box[3], inv_box[3];
  double rc, rc2, alpha, alpha2, two_a_sqrtpi, erfc_rc, fshift;
  double *part;             // ENERGY: per-CTA partial sums of U_s
  unsigned long long *count;// ENERGY: in-cutoff pair-bead counter
};

template <int NB, int L, bool ENERGY>
__global__ void __launch_bounds__(128) k_pair(const PairArgs a) {
  extern __shared__ double tab[];
  for (int k = threadIdx.x; k < a.nt * a.nt * 4; k += blockDim.x) tab[k] = a.pair_tab[k];
  __syncthreads();
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long i = gid / L;
  const int sub = (int)(gid % L);
  const int b0 = a.bead0 + blockIdx.y * NB;
  const bool active = i < a.N;

  double xi[NB][3], F[NB][3];
  double U = 0.0;
  unsigned long long hits = 0;
  int ti = 0;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    F[b][0] = F[b][1] = F[b][2] = 0.0;
    xi[b][0] = xi[b][1] = xi[b][2] = 0.0;
    if (active && b0 + b < a.bead_end) {
      const double4 p = reinterpret_cast<const double4 *>(a.pos4)[(long long)(b0 + b) * a.N + i];
      xi[b][0] = p.x; xi[b][1] = p.y; xi[b][2] = p.z;
      ti = (int)__double_as_longlong(p.w);
    }
  }
  if (active) {
    const int n = a.nbr_count[i];
    const int32_t *row = a.nbr + i * a.stride;
    for (int k = sub; k < n; k += L) {
      const int j = row[k];
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b0 + b < a.bead_end) {
          const double4 pj = reinterpret_cast<const double4 *>(a.pos4)[(long long)(b0 + b) * a.N + j];
          double dx = xi[b][0] - pj.x, dy = xi[b][1] - pj.y, dz = xi[b][2] - pj.z;
          dx = fma(-a.box[0], rint(dx * a.inv_box[0]), dx);
          dy = fma(-a.box[1], rint(dy * a.inv_box[1]), dy);
          dz = fma(-a.box[2], rint(dz * a.inv_box[2]), dz);
          const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
          if (r2 < a.rc2) {
            const int tj = (int)__double_as_longlong(pj.w);
            const double *pt = tab + (ti * a.nt + tj) * 4;
            const double qq = pt[0], eps4 = pt[1], sig2 = pt[2];
            const double rinv = rsqrt(r2), r = r2 * rinv, rinv2 = rinv * rinv;
            const double er = erfc(a.alpha * r), ex = exp(-a.alpha2 * r2);
            double fr = qq * (er * rinv2 + a.two_a_sqrtpi * ex * rinv - a.fshift) * rinv;
            const double s2 = sig2 * rinv2, s6 = s2 * s2 * s2;
            fr += 6.0 * eps4 * (2.0 * s6 * s6 - s6) * rinv2;
            F[b][0] += fr * dx; F[b][1] += fr * dy; F[b][2] += fr * dz;
            if (ENERGY) {
              U += qq * (er * rinv - a.erfc_rc + a.fshift * (r - a.rc)) + eps4 * (s6 * s6 - s6) - pt[3];
              hits += 1;
            }
          }
        }
      }
    }
  }
  // combine the L lanes of the group
#pragma unroll
  for (int o = L / 2; o > 0; o >>= 1) {
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      F[b][0] += __shfl_xor_sync(0xffffffffu, F[b][0], o);
      F[b][1] += __shfl_xor_sync(0xffffffffu, F[b][1], o);
      F[b][2] += __shfl_xor_sync(0xffffffffu, F[b][2], o);
    }
  }
  if (active && sub == 0) {
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b0 + b < a.bead_end) {
        double *o = a.Fs + ((long long)(b0 + b) * a.N + i) * 3;
        o[0] = F[b][0]; o[1] = F[b][1]; o[2] = F[b][2];
      }
  }
  if (ENERGY) {
    __shared__ double su[4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      U += __shfl_xor_sync(0xffffffffu, U, o);
      hits += __shfl_xor_sync(0xffffffffu, hits, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { su[w] = U; atomicAdd(a.count, hits); }
    __syncthreads();
    if (threadIdx.x == 0) {
      double s = 0.0;
      for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += su[k];
      a.part[(long long)blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
  }
}

template <int NB, int L>
static void launch_pair(const PairArgs &a, dim3 grid, int tb, size_t smem, cudaStream_t st, bool energy) {
  if (energy) k_pair<NB, L, true><<<grid, tb, smem, st>>>(a);
  else k_pair<NB, L, false><<<grid, tb, smem, st>>>(a);
}

template <int NB>
static void launch_pair_L(int L, const PairArgs &a, dim3 grid, int tb, size_t smem, cudaStream_t st, bool energy) {
  switch (L) {
    case 4: launch_pair<NB, 4>(a, grid, tb, smem, st, energy); break;
    case 8: launch_pair<NB, 8>(a, grid, tb, smem, st, energy); break;
    case 16: launch_pair<NB, 16>(a, grid, tb, smem, st, energy); break;
    default: launch_pair<NB, 32>(a, grid, tb, smem, st, energy); break;
  }
}

// number of per-CTA energy partials the ENERGY variant writes (also sizes s->red)
int qhp_pair_geometry(const qhp_system *s, int *NB_out, int *L_out, unsigned *gx, unsigned *gy) {
  const int NB = s->Pc >= 4 ? 4 : (s->Pc >= 2 ? 2 : 1);
  const int chunks = (s->Pc + NB - 1) / NB;
  int L = 4;
  while (L < 32 && (long long)s->N * chunks * L < 148LL * 2048) L *= 2;
  const int tb = 128;
  const long long threads = (long long)s->N * L;
  *NB_out = NB; *L_out = L;
  *gx = (unsigned)((threads + tb - 1) / tb);
  *gy = (unsigned)chunks;
  return (int)(*gx * *gy);
}

int qhp_pair_staged_partials(const qhp_system *s);
int qhp_pair_staged_forces(qhp_system *s, bool energy, double *part, unsigned long long *count, int bead0, int nbeads);

// upper bound of the per-CTA energy partials of either kernel (sizes s->red)
int qhp_pair_partials(const qhp_system *s) {
  int NB, L; unsigned gx, gy;
  const int n = qhp_pair_geometry(s, &NB, &L, &gx, &gy);
  const int m = s->staged_ok ? qhp_pair_staged_partials(s) : 0;
  return n > m ? n : m;
}

int qhp_pair_forces_beads(qhp_system *s, bool energy, int bead0, int nbeads) {
  if (energy) {
    QHP_CUDA_OK(s, cudaMemsetAsync(&s->counters[3], 0, sizeof(int64_t), s->stream));
    QHP_CUDA_OK(s, cudaMemsetAsync(s->red + 4 * (size_t)s->n_tiles, 0, sizeof(double) * (size_t)qhp_pair_partials(s), s->stream));
  }
  if (s->staged)
    return qhp_pair_staged_forces(s, energy, s->red + 4 * (size_t)s->n_tiles, (unsigned long long *)&s->counters[3], bead0, nbeads);
  PairArgs a{};
  a.N = s->N; a.Pc = s->Pc; a.nt = s->nt; a.bead0 = bead0; a.bead_end = bead0 + nbeads;
  a.pos4 = s->pos4; a.Fs = s->Fs; a.nbr = s->nbr; a.nbr_count = s->nbr_count; a.stride = s->nbr_stride;
  a.pair_tab = s->pair_tab;
  for (int d = 0; d < 3; ++d) { a.box[d] = s->box[d]; a.inv_box[d] = s->inv_box[d]; }
  const double rc = s->r_cut, al = s->alpha;
  a.rc = rc; a.rc2 = rc * rc; a.alpha = al; a.alpha2 = al * al;
  a.two_a_sqrtpi = 2.0 * al / sqrt(QHP_PI);
  a.erfc_rc = erfc(al * rc) / rc;
  a.fshift = erfc(al * rc) / (rc * rc) + a.two_a_sqrtpi * exp(-al * al * rc * rc) / rc;
  int NB, L; unsigned gx, gy;
  qhp_pair_geometry(s, &NB, &L, &gx, &gy);
  gy = (unsigned)((nbeads + NB - 1) / NB);           // bead chunks of this slice
  a.part = s->red + 4 * (size_t)s->n_tiles;
  a.count = (unsigned long long *)&s->counters[3];
  const dim3 grid(gx, gy);
  const size_t smem = sizeof(double) * 4 * s->nt * s->nt;
  switch (NB) {
    case 4: launch_pair_L<4>(L, a, grid, 128, smem, s->stream, energy); break;
    case 2: launch_pair_L<2>(L, a, grid, 128, smem, s->stream, energy); break;
    default: launch_pair_L<1>(L, a, grid, 128, smem, s->stream, energy); break;
  }
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

// V_s forces of all contracted beads.  After qhp_set_comm (world > 1) this rank evaluates its own bead slice and the
// ranks exchange the slices: F_s is bead-major, so every rank's slice is one contiguous block and the exchange is one
// in-place all-gather on the library's stream (forces gathered over the polymer communicator, then
// projected).  The energy variant (observables, counters) always evaluates every bead locally.
int qhp_pair_forces(qhp_system *s, bool energy) {
  if (energy || s->shard_world <= 1) return qhp_pair_forces_beads(s, energy, 0, s->Pc);
  const int nb = s->Pc / s->shard_world;
  int rc = qhp_pair_forces_beads(s, false, s->shard_rank * nb, nb);
  if (rc) return rc;
  const size_t bytes = sizeof(double) * 3 * (size_t)s->N * nb;
  if (s->shard_allgather(s->shard_ctx, s->Fs, bytes, s->shard_rank, s->shard_world, (void *)s->stream) != 0) {
    s->err = "qhp_set_comm: the all-gather callback failed";
    return QHP_ECUDA;
  }
  return QHP_OK;
}
