// nm_kernels.cu -- normal-mode side of the hot path:
//   * bead <-> normal-mode transforms (Eq. 4),
//   * the fused integrator pass: [B] B A O A in normal modes (Eq. 16-17) with the
//     intramolecular forces V_f on all P beads, their projection on the modes
//     (Eq. 10-11), the expansion of the contracted slow forces and the contraction of the new
//     positions (Eq. 20) -- one read and one write of Q and Pm per step,
//   * bead-space force output (O7) and observables (Eq. 6, O8).
//
// Layout: Q, Pm are [P][3N] (mode-major, DOF contiguous).  One CTA = one tile of whole
// molecules; thread t of the CTA owns DOF 3*a0 + t of the tile for all P modes (coalesced
// 8-byte accesses for every mode), and the tile's bead positions / forces are exchanged through
// two shared-memory tiles [P][TD] so that the bonded terms can be evaluated per (molecule, bead).
// The P x P transform matrix is a kernel parameter, i.e. lives in the constant bank: with the
// loops fully unrolled every FMA takes its coefficient as an immediate constant operand.
#include <algorithm>

#include "qhp_internal.cuh"
#include "contract.cuh"
#include "philox.cuh"

template <int P> struct NmTab { double T[P * P]; };   // T[i*P+n], Eq. 2 eigenvectors
// Mass-independent coefficients of the A and O blocks per mode (kernel-parameter bank: they reach the
// FP64 instructions as constant operands, no loads): cs = cos(w dt/2), sw = sin(w dt/2)/w,
// ws = w sin(w dt/2), c1 = exp(-gamma_n dt), c2k = sqrt(kB T 418.4 (1 - c1^2)).  With the mass m of the
// DOF: s1 = sw/m, s2 = -m ws, noise amplitude = sqrt(m) c2k.
template <int P> struct ModeCoef { double cs[P], sw[P], ws[P], c1[P], c2k[P]; };

struct IntArgs {
  int N, Pc, nt, TD;
  long long ND;
  const qhp_tile *tiles;
  double *Q, *Pm;
  const double *coef;
  const int32_t *type, *molid, *mol_atom_start, *mol_bond_start, *mol_angle_start;
  const int32_t *bond_idx, *angle_idx;
  const double *bond_k, *bond_r0, *angle_k, *angle_th0, *tether_k, *mass;
  const int32_t *rank;
  double *pos4;
  const double *Fs;
  const double *cref;
  unsigned long long *d2max;
  int do_step;
  double w_fast, w_slow;   // kick weights (dt/2 * 418.4 units) of V_f and V_s in this pass
  long long step;
  const long long *step_base;   // NULL, or device: added to `step` for the Philox counters (CUDA-graph replays, qhp_api.cu)
  unsigned long long seed;
  double hdt;
  // adQTB (P = 1)
  const double *Fc;
  double *vseg;
  const int32_t *seg_slot;   // atom -> segment slot (qhp_seg_addr)
  int n_seg, n_loc;
  double qa, qbA;
  // outputs of the auxiliary kernels
  double *G;      // bead forces
  double *part;   // per-CTA partial sums [n_tiles][4]
  double kT;
};

// step index within the noise segment; under a CUDA-graph replay the baked index is shifted by the device-side base
// (replays never cross a segment boundary: qhp_api.cu)
__device__ __forceinline__ int seg_step(const IntArgs &a) {
  return a.step_base ? (int)((a.n_loc + *a.step_base) % a.n_seg) : a.n_loc;
}

// ---------------------------------------------------------------------------------------------
// V_f of one (molecule, bead): harmonic bonds, harmonic angles, optional tether (BASELINE.json
// configs[0]; oracle O3).  x, f point at the bead's row of the shared tiles; a0 = first atom of
// the tile.  The calling thread owns this (molecule, bead), so plain read-modify-write is safe.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double bonded_molecule(const IntArgs &a, int m, int a0,
                                                  const double *__restrict__ x, double *f) {
  double U = 0.0;
  const int b0 = a.mol_bond_start[m], b1 = a.mol_bond_start[m + 1];
  for (int b = b0; b < b1; ++b) {
    const int i = 3 * (a.bond_idx[2 * b] - a0), j = 3 * (a.bond_idx[2 * b + 1] - a0);
    const double dx = x[i] - x[j], dy = x[i + 1] - x[j + 1], dz = x[i + 2] - x[j + 2];
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    const double k = a.bond_k[b], dr = r - a.bond_r0[b];
    U += 0.5 * k * dr * dr;
    const double g = -k * dr / r;
    f[i] += g * dx; f[i + 1] += g * dy; f[i + 2] += g * dz;
    f[j] -= g * dx; f[j + 1] -= g * dy; f[j + 2] -= g * dz;
  }
  const int g0 = a.mol_angle_start[m], g1 = a.mol_angle_start[m + 1];
  for (int g = g0; g < g1; ++g) {
    const int i = 3 * (a.angle_idx[3 * g] - a0), j = 3 * (a.angle_idx[3 * g + 1] - a0),
              k = 3 * (a.angle_idx[3 * g + 2] - a0);                       // j = centre
    const double ux = x[i] - x[j], uy = x[i + 1] - x[j + 1], uz = x[i + 2] - x[j + 2];
    const double vx = x[k] - x[j], vy = x[k + 1] - x[j + 1], vz = x[k + 2] - x[j + 2];
    const double ru = sqrt(ux * ux + uy * uy + uz * uz), rv = sqrt(vx * vx + vy * vy + vz * vz);
    const double iruv = 1.0 / (ru * rv);
    double cs = (ux * vx + uy * vy + uz * vz) * iruv;
    cs = fmin(1.0, fmax(-1.0, cs));
    const double th = acos(cs), dth = th - a.angle_th0[g], ka = a.angle_k[g];
    U += 0.5 * ka * dth * dth;
    const double sn = sqrt(1.0 - cs * cs);
    const double gg = ka * dth / sn;
    const double cu = cs / (ru * ru), cv = cs / (rv * rv);
    const double fix = gg * (vx * iruv - cu * ux), fiy = gg * (vy * iruv - cu * uy), fiz = gg * (vz * iruv - cu * uz);
    const double fkx = gg * (ux * iruv - cv * vx), fky = gg * (uy * iruv - cv * vy), fkz = gg * (uz * iruv - cv * vz);
    f[i] += fix; f[i + 1] += fiy; f[i + 2] += fiz;
    f[k] += fkx; f[k + 1] += fky; f[k + 2] += fkz;
    f[j] -= fix + fkx; f[j + 1] -= fiy + fky; f[j + 2] -= fiz + fkz;
  }
  if (a.tether_k) {
    const int s0 = a.mol_atom_start[m], s1 = a.mol_atom_start[m + 1];
    for (int at = s0; at < s1; ++at) {
      const double k = a.tether_k[a.type[at]];
      const int i = 3 * (at - a0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const double xx = x[i + c];
        U += 0.5 * k * xx * xx;
        f[i + c] -= k * xx;
      }
    }
  }
  return U;
}

// x_i = sqrt(P) sum_n T_in Q_n for one DOF (Eq. 4).  The bead loop is rolled (its index is
// warp-uniform, so the coefficients come through the constant bank / uniform registers) and the
// mode sum runs in four independent partial sums; a fully unrolled P x P body overflowed the
// instruction cache at P = 32.
// The transfer matrix (O1) is a real DFT: columns n = 0, odd n (cos) and, for even P, n = P - 1 are
// symmetric under i -> P - i, columns of even n >= 2 (sin) antisymmetric and zero at i = 0, P/2.
// Beads i and P - i therefore share one cos sum A and one sin sum B (x_i = A + B, x_{P-i} = A - B),
// which halves the multiply-adds of the dense P x P transforms.
#define QHP_SIN_MODE(n) ((n) >= 2 && ((n) & 1) == 0)
template <int P>
__device__ __forceinline__ void modes_to_beads_tile(const NmTab<P> &tab, const double (&Qr)[P], double *xt, double *ft,
                                                    int TD, int t) {
  const double sp = sqrt((double)P);
  constexpr int NP = (P - 1) / 2;                 // pairs (i, P - i), i = 1 .. NP
  {                                               // i = 0 and, for even P, i = P/2: cos-type columns only
    double s0 = 0.0, s1 = 0.0, h0 = 0.0, h1 = 0.0;
#pragma unroll
    for (int n = 0; n < P; ++n)
      if (!QHP_SIN_MODE(n)) {
        if (n & 2) { s1 = fma(tab.T[n], Qr[n], s1); if (P % 2 == 0) h1 = fma(tab.T[(P / 2) * P + n], Qr[n], h1); }
        else { s0 = fma(tab.T[n], Qr[n], s0); if (P % 2 == 0) h0 = fma(tab.T[(P / 2) * P + n], Qr[n], h0); }
      }
    xt[t] = sp * (s0 + s1); ft[t] = 0.0;
    if (P % 2 == 0 && P > 1) { xt[(P / 2) * TD + t] = sp * (h0 + h1); ft[(P / 2) * TD + t] = 0.0; }
  }
#pragma unroll 1
  for (int i = 1; i <= NP; ++i) {
    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
#pragma unroll
    for (int n = 0; n < P; ++n) {
      if (QHP_SIN_MODE(n)) { if (n & 2) b1 = fma(tab.T[i * P + n], Qr[n], b1); else b0 = fma(tab.T[i * P + n], Qr[n], b0); }
      else { if (n & 2) a1 = fma(tab.T[i * P + n], Qr[n], a1); else a0 = fma(tab.T[i * P + n], Qr[n], a0); }
    }
    const double A = a0 + a1, B = b0 + b1;
    xt[i * TD + t] = sp * (A + B); ft[i * TD + t] = 0.0;
    xt[(P - i) * TD + t] = sp * (A - B); ft[(P - i) * TD + t] = 0.0;
  }
}

// fr[n] = (1/sqrt P) sum_i T_in F^f_i (Eq. 10-11) + (1/sqrt P') sum_j T'_jn Fs_j (n < P'), one DOF
// wf, ws: weights of the fast (V_f) and slow (V_s) parts: 1, 1 for the total force; the integrator
// passes the kick weights of the two parts, which differ under BAOAB-RESPA (Eq. 19).
template <int P>
__device__ __forceinline__ void project_forces_tile(const IntArgs &a, const NmTab<P> &tab, const NmTab<P> &ctab,
                                                    const double *ft, int TD, int t, int atom, int c, double (&fr)[P],
                                                    double wf = 1.0, double ws = 1.0) {
  constexpr int NP = (P - 1) / 2;
  {
    const double F0 = ft[t], Fh = (P % 2 == 0 && P > 1) ? ft[(P / 2) * TD + t] : 0.0;
#pragma unroll
    for (int n = 0; n < P; ++n) {
      if (QHP_SIN_MODE(n)) fr[n] = 0.0;
      else fr[n] = (P % 2 == 0 && P > 1) ? fma(tab.T[(P / 2) * P + n], Fh, tab.T[n] * F0) : tab.T[n] * F0;
    }
  }
#pragma unroll 1
  for (int i = 1; i <= NP; ++i) {
    const double Fi = ft[i * TD + t], Fm = ft[(P - i) * TD + t];
    const double S = Fi + Fm, D = Fi - Fm;
#pragma unroll
    for (int n = 0; n < P; ++n) fr[n] = fma(tab.T[i * P + n], QHP_SIN_MODE(n) ? D : S, fr[n]);
  }
  const double isp = wf / sqrt((double)P);
#pragma unroll
  for (int n = 0; n < P; ++n) fr[n] *= isp;
  // slow forces of the contracted beads, chain rule on Eq. 20
  const int Pc = a.Pc;
  const double ispc = ws / sqrt((double)Pc);
  const long long slot = a.rank[atom];
  for (int j = 0; j < Pc; ++j) {
    const double Fj = a.Fs[((long long)j * a.N + slot) * 3 + c] * ispc;
#pragma unroll
    for (int n = 0; n < P; ++n)
      if (n < Pc) fr[n] = fma(ctab.T[j * Pc + n], Fj, fr[n]);
  }
}

// V_f of every (molecule, bead) of the tile: positions in xt, forces accumulated into ft
__device__ __forceinline__ double bonded_tile(const IntArgs &a, const qhp_tile tl, int P, const double *xt, double *ft) {
  double U = 0.0;
  const int nm = tl.m1 - tl.m0, TD = a.TD;
  for (int w = threadIdx.x; w < nm * P; w += blockDim.x) {
    const int m = tl.m0 + w % nm, bead = w / nm;
    U += bonded_molecule(a, m, tl.a0, xt + bead * TD, ft + bead * TD);
  }
  return U;
}

// ---------------------------------------------------------------------------------------------
// Common front end of the force / observable kernels for one tile:
//   Qr[n]  <- Q_n of this thread's DOF, x_i -> shared tile, V_f forces per (molecule, bead),
//   fr[n]  <- projected fast + expanded slow forces.
// Returns this thread's share of sum_i V_f(x_i).
// ---------------------------------------------------------------------------------------------
template <int P>
__device__ __forceinline__ double tile_forces(const IntArgs &a, const NmTab<P> &tab, const NmTab<P> &ctab,
                                              const qhp_tile tl, double *xt, double *ft,
                                              bool active, long long dof, int atom, int c,
                                              double (&Qr)[P], double (&fr)[P]) {
  const int t = threadIdx.x, TD = a.TD;
  if (active) {
#pragma unroll
    for (int n = 0; n < P; ++n) Qr[n] = a.Q[n * a.ND + dof];
    modes_to_beads_tile<P>(tab, Qr, xt, ft, TD, t);
  }
  __syncthreads();
  const double U = bonded_tile(a, tl, P, xt, ft);
  __syncthreads();
  if (active) project_forces_tile<P>(a, tab, ctab, ft, TD, t, atom, c, fr);
  return U;
}

__device__ __forceinline__ double block_max(double v, double *scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) scratch[w] = v;
  __syncthreads();
  v = (l < nw) ? scratch[l] : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// deterministic block sum (fixed tree)
__device__ __forceinline__ double block_sum(double v, double *scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) scratch[w] = v;
  __syncthreads();
  v = (l < nw) ? scratch[l] : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---------------------------------------------------------------------------------------------
// Fused integrator pass.  THERMO: 0 none, 1 PILE/TRPMD, 2 adQTB (P = 1).
//   kick_prev: apply the final B(dt/2) of the previous step (forces at the current Q);
//   do_step  : B(dt/2) A(dt/2) O(dt) A(dt/2) of this step, then write the contracted positions
//              of the new Q (slot order) and the list-validity statistic max |xc - cref|^2.
// ---------------------------------------------------------------------------------------------
// CTA size and residency: 48-atom tiles (160 threads, three CTAs per SM) for P >= 24, else 96-atom tiles
template <int P, int THERMO, int PCM>   // PCM: compile-time bound on the contracted beads P'
__global__ void __launch_bounds__(P >= 24 ? 160 : 288, P >= 24 ? 3 : 1) k_integrate(const IntArgs a, const NmTab<P> tab, const NmTab<P> ctab,
                                                                                   const ModeCoef<P> mc) {
  extern __shared__ double sm[];
  const int TD = a.TD, t = threadIdx.x;
  double *xt = sm, *ft = sm + P * TD, *scratch = ft + P * TD;
  const qhp_tile tl = a.tiles[blockIdx.x];
  const int nd = 3 * (tl.a1 - tl.a0);
  const bool active = t < nd;
  const long long dof = 3LL * tl.a0 + t;
  const int atom = tl.a0 + t / 3, c = t % 3;
  if (blockIdx.x == 0 && t == 0 && a.do_step) a.d2max[(a.step + 1) & 1] = 0ull;

  // loads that do not depend on the tile exchange are issued first, so that their latency overlaps
  // phases 1-3 (the P <= 8 kernels are latency-bound: one short dependent chain per CTA)
  constexpr int PF = P < 8 ? P : 8;                    // momenta in flight
  double pl[PF];
  double fc_early = 0.0;
  int ty = 0;
  if (active) {
    ty = a.type[atom];
    if (P <= 8) {
#pragma unroll
      for (int k = 0; k < PF; ++k) pl[k] = a.Pm[k * a.ND + dof];
    }
    if (THERMO == 2 && a.do_step) fc_early = a.Fc[qhp_seg_addr(a.seg_slot[atom], a.n_seg, seg_step(a)) + c];
  }

  // ---- phase 1: Q -> bead positions (shared tile), V_f per (molecule, bead) -------------------------
  {
    double Qr[P];
    if (active) {
#pragma unroll
      for (int n = 0; n < P; ++n) Qr[n] = a.Q[n * a.ND + dof];
      modes_to_beads_tile<P>(tab, Qr, xt, ft, TD, t);
    }
    __syncthreads();
    bonded_tile(a, tl, P, xt, ft);
    __syncthreads();
    // the positions are dead: park this DOF's Q_n in its own column of xt (frees the registers for fr)
    if (active) {
#pragma unroll
      for (int n = 0; n < P; ++n) xt[n * TD + t] = Qr[n];
    }
  }
  // ---- phase 2: normal-mode forces of this DOF ---------------------------------------------------------
  double fr[P];
  if (active) project_forces_tile<P>(a, tab, ctab, ft, TD, t, atom, c, fr, a.w_fast, a.w_slow);   // fr = momentum kick
  // ---- phase 3 (PILE): one Philox call per (atom, mode) gives the three Cartesian normals; they are
  //      exchanged through the force tile, which is dead once every thread has its fr ---------------------
  if (THERMO == 1 && a.do_step) {
    __syncthreads();
    const int na = tl.a1 - tl.a0;
    for (int w = t; w < na * P; w += blockDim.x) {
      const int al = w % na, n = w / na;
      double z[3];
      qhp_normals3(a.seed, (uint32_t)(tl.a0 + al), (uint32_t)n, QHP_TAG_PILE, (uint64_t)(a.step + (a.step_base ? *a.step_base : 0LL)), z);
      ft[n * TD + 3 * al] = z[0]; ft[n * TD + 3 * al + 1] = z[1]; ft[n * TD + 3 * al + 2] = z[2];
    }
    __syncthreads();
  }
  // ---- phase 4: B A O A per mode, contraction of the new positions -----------------------------------------
  double d2 = 0.0;
  if (active) {
    const double m = a.mass[ty], minv = 1.0 / m, sqm = sqrt(m);
    double xc[PCM];                     // contracted beads (first Pc entries used)
#pragma unroll
    for (int j = 0; j < PCM; ++j) xc[j] = 0.0;
    // momenta are fetched eight modes ahead of their use: the stores of one mode must not
    // serialise the loads of the next (Q and Pm may alias as far as the compiler knows)
#pragma unroll
    for (int n = 0; n < P; ++n) {
      if (n % PF == 0 && P > 8) {
#pragma unroll
        for (int k = 0; k < PF; ++k)
          if (n + k < P) pl[k] = a.Pm[(n + k) * a.ND + dof];
      }
      double q = xt[n * TD + t];
      double p = pl[n % PF];
      p += fr[n];                       // B: pending half kick of the last step + first half kick of this one
      if (a.do_step) {
        const double cs = mc.cs[n], s1 = mc.sw[n] * minv, s2 = -(mc.ws[n] * m);
        // A(dt/2): centroid translation / exact free ring-polymer rotation
        if (n == 0) q += a.hdt * p * minv;
        else { const double qn = cs * q + s1 * p; p = s2 * q + cs * p; q = qn; }
        // O(dt)
        if (THERMO == 1) {
          p = mc.c1[n] * p + (mc.c2k[n] * sqm) * ft[n * TD + t];
        } else if (THERMO == 2) {
          // classical BAOAB carrying the coloured force (Eq. 12, l.199; readings G14, G16)
          const long long k = qhp_seg_addr(a.seg_slot[atom], a.n_seg, seg_step(a)) + c;
          const double pn = a.qa * p + a.qbA * fc_early;
          a.vseg[k] = (p + pn) / (2.0 * m);
          p = pn;
        }
        // A(dt/2)
        if (n == 0) q += a.hdt * p * minv;
        else { const double qn = cs * q + s1 * p; p = s2 * q + cs * p; q = qn; }
        a.Q[n * a.ND + dof] = q;
        // contraction of the new positions (Eq. 20): only the first Pc modes contribute
        if (n < PCM && n < a.Pc) {
#pragma unroll
          for (int j = 0; j < PCM; ++j)
            if (j < a.Pc) xc[j] = fma(ctab.T[j * a.Pc + n], q, xc[j]);
        }
      }
      a.Pm[n * a.ND + dof] = p;
    }
    if (a.do_step) {
      // contracted positions into slot order + list-validity statistic
      const double spc = sqrt((double)a.Pc);
      const long long slot = a.rank[atom];
      const double cr = a.cref[dof];
#pragma unroll
      for (int j = 0; j < PCM; ++j)
        if (j < a.Pc) {
          const double x = spc * xc[j];
          a.pos4[((long long)j * a.N + slot) * 4 + c] = x;
          const double dd = x - cr;
          d2 = fmax(d2, dd * dd);
        }
    }
  }
  if (a.do_step) {
    // per-atom |xc - cref|^2 <= sum over components of the per-component maxima over beads
    __syncthreads();
    xt[t] = d2;
    __syncthreads();
    double v = 0.0;
    if (active && c == 0) v = xt[t] + xt[t + 1] + xt[t + 2];
    v = block_max(v, scratch);
    if (t == 0) atomicMax(&a.d2max[a.step & 1], (unsigned long long)__double_as_longlong(v));
  }
}

// ---------------------------------------------------------------------------------------------
// P = 1 (classical BAOAB, adQTB) with molecules of at most 4 atoms: one THREAD per molecule.  With a
// single bead there is no normal-mode transform, so the tile exchange of k_integrate only served the
// bonded terms; a thread that owns a whole molecule needs no shared memory and no barrier, and the
// kernel is no longer a chain of short latency-bound phases (C3: 0.09 -> see profiles).
// Forces are accumulated in registers through predicated adds (static indices, no local memory).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void acc4(double (&f)[4][3], int ai, double gx, double gy, double gz) {
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (ai == k) { f[k][0] += gx; f[k][1] += gy; f[k][2] += gz; }
}

template <int THERMO>
__global__ void __launch_bounds__(128) k_integrate_mol1(const IntArgs a, int n_mol) {
  __shared__ double scratch[32];
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (blockIdx.x == 0 && threadIdx.x == 0 && a.do_step) a.d2max[(a.step + 1) & 1] = 0ull;
  double d2 = 0.0;
  if (m < n_mol) {
    const int s0 = a.mol_atom_start[m], na = a.mol_atom_start[m + 1] - s0;
    const double *x = a.Q + 3LL * s0;                 // P = 1: bead positions are Q_0
    double f[4][3];
#pragma unroll
    for (int k = 0; k < 4; ++k) f[k][0] = f[k][1] = f[k][2] = 0.0;
    for (int b = a.mol_bond_start[m]; b < a.mol_bond_start[m + 1]; ++b) {
      const int ai = a.bond_idx[2 * b] - s0, aj = a.bond_idx[2 * b + 1] - s0;
      const double dx = x[3 * ai] - x[3 * aj], dy = x[3 * ai + 1] - x[3 * aj + 1], dz = x[3 * ai + 2] - x[3 * aj + 2];
      const double r = sqrt(dx * dx + dy * dy + dz * dz);
      const double g = -a.bond_k[b] * (r - a.bond_r0[b]) / r;
      acc4(f, ai, g * dx, g * dy, g * dz);
      acc4(f, aj, -g * dx, -g * dy, -g * dz);
    }
    for (int g = a.mol_angle_start[m]; g < a.mol_angle_start[m + 1]; ++g) {
      const int ai = a.angle_idx[3 * g] - s0, aj = a.angle_idx[3 * g + 1] - s0, ak = a.angle_idx[3 * g + 2] - s0;   // aj = centre
      const double ux = x[3 * ai] - x[3 * aj], uy = x[3 * ai + 1] - x[3 * aj + 1], uz = x[3 * ai + 2] - x[3 * aj + 2];
      const double vx = x[3 * ak] - x[3 * aj], vy = x[3 * ak + 1] - x[3 * aj + 1], vz = x[3 * ak + 2] - x[3 * aj + 2];
      const double ru = sqrt(ux * ux + uy * uy + uz * uz), rv = sqrt(vx * vx + vy * vy + vz * vz);
      const double iruv = 1.0 / (ru * rv);
      double cs = (ux * vx + uy * vy + uz * vz) * iruv;
      cs = fmin(1.0, fmax(-1.0, cs));
      const double dth = acos(cs) - a.angle_th0[g];
      const double gg = a.angle_k[g] * dth / sqrt(1.0 - cs * cs);
      const double cu = cs / (ru * ru), cv = cs / (rv * rv);
      const double fix = gg * (vx * iruv - cu * ux), fiy = gg * (vy * iruv - cu * uy), fiz = gg * (vz * iruv - cu * uz);
      const double fkx = gg * (ux * iruv - cv * vx), fky = gg * (uy * iruv - cv * vy), fkz = gg * (uz * iruv - cv * vz);
      acc4(f, ai, fix, fiy, fiz);
      acc4(f, ak, fkx, fky, fkz);
      acc4(f, aj, -(fix + fkx), -(fiy + fky), -(fiz + fkz));
    }
    if (a.tether_k)
      for (int al = 0; al < na; ++al) {
        const double k = a.tether_k[a.type[s0 + al]];
        acc4(f, al, -k * x[3 * al], -k * x[3 * al + 1], -k * x[3 * al + 2]);
      }
    // every position of the molecule has been read: update its atoms in place.  Two sweeps: all loads of the
    // molecule first (independent, so their latencies overlap; the kernel has one thread per molecule and is
    // latency-bound), then the arithmetic and the stores.
    int ty_[4];
    long long slot_[4], segb_[4];
    double q_[4][3], p_[4][3], fs_[4][3], fc_[4][3], cr_[4][3];
#pragma unroll
    for (int al = 0; al < 4; ++al) {
      if (al >= na) break;
      const int atom = s0 + al;
      ty_[al] = __ldg(a.type + atom);
      slot_[al] = __ldg(a.rank + atom);
      segb_[al] = THERMO == 2 ? qhp_seg_addr(__ldg(a.seg_slot + atom), a.n_seg, seg_step(a)) : 0;
    }
#pragma unroll
    for (int al = 0; al < 4; ++al) {
      if (al >= na) break;
      const int atom = s0 + al;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const long long dof = 3LL * atom + c;
        q_[al][c] = a.Q[dof]; p_[al][c] = a.Pm[dof];
        fs_[al][c] = __ldg(a.Fs + slot_[al] * 3 + c);
        fc_[al][c] = (THERMO == 2 && a.do_step) ? __ldg(a.Fc + segb_[al] + c) : 0.0;
        cr_[al][c] = a.do_step ? __ldg(a.cref + dof) : 0.0;
      }
    }
#pragma unroll
    for (int al = 0; al < 4; ++al) {
      if (al >= na) break;
      const int atom = s0 + al;
      const int ty = ty_[al];
      const double mass = __ldg(a.mass + ty);
      const long long slot = slot_[al];
      const double *cf = a.coef + ty * QHP_NCOEF;
      double z[3] = {0.0, 0.0, 0.0};
      if (THERMO == 1 && a.do_step) qhp_normals3(a.seed, (uint32_t)atom, 0u, QHP_TAG_PILE, (uint64_t)(a.step + (a.step_base ? *a.step_base : 0LL)), z);
      double dsum = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const long long dof = 3LL * atom + c;
        double q = q_[al][c], p = p_[al][c];
        p += a.w_fast * f[al][c] + a.w_slow * fs_[al][c];
        if (a.do_step) {
          q += a.hdt * p / mass;
          if (THERMO == 1) {
            p = __ldg(cf + 3) * p + __ldg(cf + 4) * z[c];
          } else if (THERMO == 2) {
            const long long k = segb_[al] + c;
            const double pn = a.qa * p + a.qbA * fc_[al][c];
            a.vseg[k] = (p + pn) / (2.0 * mass);
            p = pn;
          }
          q += a.hdt * p / mass;
          a.Q[dof] = q;
          a.pos4[slot * 4 + c] = q;
          const double dd = q - cr_[al][c];
          dsum += dd * dd;
        }
        a.Pm[dof] = p;
      }
      d2 = fmax(d2, dsum);
    }
  }
  if (a.do_step) {
    d2 = block_max(d2, scratch);
    if (threadIdx.x == 0) atomicMax(&a.d2max[a.step & 1], (unsigned long long)__double_as_longlong(d2));
  }
}

// bead-space forces G_i = sqrt(P) sum_n T_in f_n (O7)
template <int P>
__global__ void __launch_bounds__(288) k_bead_forces(const IntArgs a, const NmTab<P> tab, const NmTab<P> ctab) {
  extern __shared__ double sm[];
  const int TD = a.TD, t = threadIdx.x;
  double *xt = sm, *ft = sm + P * TD;
  const qhp_tile tl = a.tiles[blockIdx.x];
  const bool active = t < 3 * (tl.a1 - tl.a0);
  const long long dof = 3LL * tl.a0 + t;
  const int atom = tl.a0 + t / 3, c = t % 3;
  double Qr[P], fr[P];
  tile_forces<P>(a, tab, ctab, tl, xt, ft, active, dof, atom, c, Qr, fr);
  if (active) {
    const double sp = sqrt((double)P);
#pragma unroll
    for (int i = 0; i < P; ++i) {
      double s = 0.0;
#pragma unroll
      for (int n = 0; n < P; ++n) s += tab.T[i * P + n] * fr[n];
      a.G[i * a.ND + dof] = sp * s;
    }
  }
}

// partial sums of the observables (O8): part[cta] = {sum_{n>0} Q_n f_n, sum_i V_f(x_i), sum Pm^2/2m}
template <int P>
__global__ void __launch_bounds__(288) k_observe(const IntArgs a, const NmTab<P> tab, const NmTab<P> ctab) {
  extern __shared__ double sm[];
  const int TD = a.TD, t = threadIdx.x;
  double *xt = sm, *ft = sm + P * TD, *scratch = ft + P * TD;
  const qhp_tile tl = a.tiles[blockIdx.x];
  const bool active = t < 3 * (tl.a1 - tl.a0);
  const long long dof = 3LL * tl.a0 + t;
  const int atom = tl.a0 + t / 3, c = t % 3;
  double Qr[P], fr[P];
  double U = tile_forces<P>(a, tab, ctab, tl, xt, ft, active, dof, atom, c, Qr, fr);
  double vir = 0.0, kin = 0.0;
  if (active) {
    const double m = a.mass[a.type[atom]];
#pragma unroll
    for (int n = 0; n < P; ++n) {
      if (n > 0) vir += Qr[n] * fr[n];
      const double p = a.Pm[n * a.ND + dof];
      kin += p * p / (2.0 * m);
    }
  }
  vir = block_sum(vir, scratch);
  U = block_sum(U, scratch);
  kin = block_sum(kin, scratch);
  if (t == 0) {
    a.part[4 * blockIdx.x + 0] = vir;
    a.part[4 * blockIdx.x + 1] = U;
    a.part[4 * blockIdx.x + 2] = kin;
    a.part[4 * blockIdx.x + 3] = 0.0;
  }
}

// final fixed-order reduction of the per-CTA partial sums and of the pair-energy partials
__global__ void k_observe_final(const double *part, int n_part, const double *pair_part, int n_pair,
                                double *obs, int N, int P, int Pc, double kT) {
  __shared__ double scratch[32];
  double v = 0, u = 0, k = 0, us = 0;
  for (int i = threadIdx.x; i < n_part; i += blockDim.x) { v += part[4 * i]; u += part[4 * i + 1]; k += part[4 * i + 2]; }
  for (int i = threadIdx.x; i < n_pair; i += blockDim.x) us += pair_part[i];
  v = block_sum(v, scratch); u = block_sum(u, scratch); k = block_sum(k, scratch); us = block_sum(us, scratch);
  if (threadIdx.x == 0) {
    obs[0] = 1.5 * N * kT - 0.5 * v;
    obs[1] = u / P + 0.5 * us / Pc;       // full list: every pair energy was counted twice
    obs[2] = k / QHP_ACC;
    obs[3] = 2.0 * obs[2] / (3.0 * (double)N * (double)P * QHP_KB);
  }
}

// ---- plain per-DOF transforms (no tile) ---------------------------------------------------------
template <int P>
__global__ void k_to_modes(const double *__restrict__ xb, const double *__restrict__ pb, double *Q, double *Pm,
                           long long ND, const NmTab<P> tab) {
  const long long d = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= ND) return;
  const double sp = sqrt((double)P);
  for (int which = 0; which < 2; ++which) {
    const double *in = which ? pb : xb;
    double *out = which ? Pm : Q;
    if (!in) continue;
    double v[P];
#pragma unroll
    for (int i = 0; i < P; ++i) v[i] = in[i * ND + d];
#pragma unroll
    for (int n = 0; n < P; ++n) {
      double s = 0.0;
#pragma unroll
      for (int i = 0; i < P; ++i) s += tab.T[i * P + n] * v[i];
      out[n * ND + d] = s / sp;
    }
  }
}

template <int P>
__global__ void k_to_beads(const double *__restrict__ Q, const double *__restrict__ Pm, double *xb, double *pb,
                           long long ND, const NmTab<P> tab) {
  const long long d = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= ND) return;
  const double sp = sqrt((double)P);
  for (int which = 0; which < 2; ++which) {
    const double *in = which ? Pm : Q;
    double *out = which ? pb : xb;
    if (!out) continue;
    double v[P];
#pragma unroll
    for (int n = 0; n < P; ++n) v[n] = in[n * ND + d];
#pragma unroll
    for (int i = 0; i < P; ++i) {
      double s = 0.0;
#pragma unroll
      for (int n = 0; n < P; ++n) s += tab.T[i * P + n] * v[n];
      out[i * ND + d] = sp * s;
    }
  }
}

// Contraction (Eq. 20) of the current Q.  mode 0: write pos4 in slot order (after a list rebuild
// also cent4 = sorted centroids + molecule id, cref = centroids in atom order, pos4.w = type);
// mode 1: write xc_out [Pc][N][3] in atom order (parity hook).
// `need` (may be NULL): device flag words; the kernel returns at once unless forced or the
// list-validity statistic exceeds the threshold.
__global__ void k_contract(const BoxArg bx, const double *__restrict__ Q, int N, int Pc, const double *__restrict__ Tc,
                           const int32_t *__restrict__ rank, const int32_t *__restrict__ type,
                           const int32_t *__restrict__ molid, double *pos4, double *cent4, double *cref,
                           double *xc_out, int mode, const unsigned long long *d2max, double thresh2,
                           long long *counters) {
  if (d2max && __longlong_as_double((long long)*d2max) < thresh2) return;
  const long long d = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= 3LL * N) return;
  qhp_contract_dof(bx, Q, N, Pc, Tc, rank, type, molid, pos4, cent4, cref, xc_out, mode, thresh2, counters, d);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <int P> static NmTab<P> make_tab(const std::vector<double> &T, int n) {
  NmTab<P> t;
  for (int k = 0; k < P * P; ++k) t.T[k] = 0.0;
  for (int k = 0; k < n * n; ++k) t.T[k] = T[k];   // dense [n][n] with stride n (n = P or Pc)
  return t;
}

template <int P> static ModeCoef<P> make_mode_coef(const qhp_system *s) {
  ModeCoef<P> mc;
  const double kTA = QHP_KB * s->T * QHP_ACC;
  for (int n = 0; n < P; ++n) {
    const double w = n < (int)s->omega.size() ? s->omega[n] : 0.0, h = 0.5 * s->dt;
    if (s->a_block == QHP_ABLOCK_CAYLEY) {           // BCOCB: rotation by atan(w h) instead of w h (G25)
      const double nrm = 1.0 / sqrt(1.0 + (w * h) * (w * h));
      mc.cs[n] = nrm;
      mc.sw[n] = n ? nrm * h : 0.0;
      mc.ws[n] = n ? nrm * w * w * h : 0.0;
    } else {
      mc.cs[n] = cos(w * h);
      mc.sw[n] = n ? sin(w * h) / w : 0.0;
      mc.ws[n] = n ? w * sin(w * h) : 0.0;
    }
    const double g = (n == 0) ? s->th.gamma0 : std::max(s->th.gamma0, w);
    mc.c1[n] = exp(-g * s->dt);
    mc.c2k[n] = sqrt(kTA * (1.0 - mc.c1[n] * mc.c1[n]));
  }
  return mc;
}

static IntArgs make_args(qhp_system *s) {
  IntArgs a{};
  a.N = s->N; a.Pc = s->Pc; a.nt = s->nt; a.TD = 3 * s->tile_atoms; a.ND = 3LL * s->N;
  a.tiles = s->dt_.tiles; a.Q = s->Q; a.Pm = s->Pm; a.coef = s->coef;
  a.type = s->dt_.type; a.molid = s->dt_.molid; a.mol_atom_start = s->dt_.mol_atom_start;
  a.mol_bond_start = s->dt_.mol_bond_start; a.mol_angle_start = s->dt_.mol_angle_start;
  a.bond_idx = s->dt_.bond_idx; a.angle_idx = s->dt_.angle_idx;
  a.bond_k = s->dt_.bond_k; a.bond_r0 = s->dt_.bond_r0; a.angle_k = s->dt_.angle_k; a.angle_th0 = s->dt_.angle_th0;
  a.tether_k = s->has_tether ? s->dt_.tether_k : nullptr; a.mass = s->dt_.mass;
  a.rank = s->rank; a.pos4 = s->pos4; a.Fs = s->Fs; a.cref = s->cref; a.d2max = s->d2max;
  a.seed = s->th.seed; a.hdt = 0.5 * s->dt; a.w_fast = 1.0; a.w_slow = 1.0;
  a.Fc = s->Fc; a.vseg = s->vseg; a.seg_slot = s->seg_slot; a.n_seg = s->n_seg;
  a.kT = QHP_KB * s->T;
  return a;
}

#define QHP_DISPATCH_P(s, FN)                      \
  switch ((s)->P) {                                \
    case 1: FN(1); break;                          \
    case 2: FN(2); break;                          \
    case 3: FN(3); break;                          \
    case 4: FN(4); break;                          \
    case 5: FN(5); break;                          \
    case 6: FN(6); break;                          \
    case 8: FN(8); break;                          \
    case 12: FN(12); break;                        \
    case 16: FN(16); break;                        \
    case 24: FN(24); break;                        \
    case 32: FN(32); break;                        \
    default: (s)->err = "unsupported P"; return QHP_EINVAL; \
  }

template <typename K> static cudaError_t set_smem(K kern, size_t bytes) {
  return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// kick_prev: the second half kick of the previous step is still pending (forces at the current Q);
// do_step: first half kick + A O A of step `step`.  Under RESPA (n_alt > 1, Eq. 19) V_s kicks
// with n_alt dt/2 only around every n_alt-th inner step, V_f with dt/2 around every inner step.
int qhp_nm_integrate(qhp_system *s, bool kick_prev, bool do_step, int64_t step) {
  IntArgs a = make_args(s);
  const double hA = 0.5 * s->dt * QHP_ACC;
  const int na = s->n_alt;
  a.do_step = do_step; a.step = step;
  a.step_base = s->graph_capturing ? s->graph_step_base : nullptr;
  a.w_fast = (kick_prev ? hA : 0.0) + (do_step ? hA : 0.0);
  a.w_slow = (kick_prev && step % na == 0 ? na * hA : 0.0) + (do_step && step % na == 0 ? na * hA : 0.0);
  if (do_step) s->flag_idx = (int)(step & 1);
  if (s->th.kind == QHP_THERMO_ADQTB) {
    a.n_loc = (int)(step % s->n_seg);
    a.qa = exp(-s->th.gamma0 * s->dt);
    a.qbA = sqrt((1.0 - a.qa * a.qa) * s->dt / (2.0 * s->th.gamma0)) * QHP_ACC;
  }
  const size_t smem = s->int_smem;
  const int thermo = s->th.kind;
  if (s->P == 1 && s->int_mol1) {
    const int tb = 128, grid = (s->n_mol + tb - 1) / tb;
    if (thermo == QHP_THERMO_ADQTB) k_integrate_mol1<2><<<grid, tb, 0, s->stream>>>(a, s->n_mol);
    else if (thermo == QHP_THERMO_PILE) k_integrate_mol1<1><<<grid, tb, 0, s->stream>>>(a, s->n_mol);
    else k_integrate_mol1<0><<<grid, tb, 0, s->stream>>>(a, s->n_mol);
    QHP_LAUNCH_OK(s);
    return QHP_OK;
  }
#define LAUNCH_INT(PP, TH, PCM)                                                                  \
  {                                                                                              \
    QHP_CUDA_OK(s, set_smem(k_integrate<PP, TH, PCM>, smem));                                    \
    k_integrate<PP, TH, PCM><<<s->n_tiles, s->tile_threads, smem, s->stream>>>(a, make_tab<PP>(s->T_P, PP), make_tab<PP>(s->T_Pc, s->Pc), \
                                                                               make_mode_coef<PP>(s));                              \
  }
#define FN(PP)                                                                                   \
  {                                                                                              \
    constexpr int PC4 = PP < 4 ? PP : 4;                                                         \
    if (thermo == QHP_THERMO_ADQTB) LAUNCH_INT(1, 2, 1)                                          \
    else if (thermo == QHP_THERMO_PILE) {                                                        \
      if (s->Pc <= PC4) LAUNCH_INT(PP, 1, PC4) else LAUNCH_INT(PP, 1, PP)                        \
    } else {                                                                                     \
      if (s->Pc <= PC4) LAUNCH_INT(PP, 0, PC4) else LAUNCH_INT(PP, 0, PP)                        \
    }                                                                                            \
  }
  QHP_DISPATCH_P(s, FN)
#undef FN
#undef LAUNCH_INT
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_bead_forces(qhp_system *s, double *G) {
  IntArgs a = make_args(s);
  a.G = G;
  const size_t smem = s->int_smem;
#define FN(PP)                                                                               \
  {                                                                                          \
    QHP_CUDA_OK(s, set_smem(k_bead_forces<PP>, smem));                                       \
    k_bead_forces<PP><<<s->n_tiles, s->tile_threads, smem, s->stream>>>(a, make_tab<PP>(s->T_P, PP), make_tab<PP>(s->T_Pc, s->Pc)); \
  }
  QHP_DISPATCH_P(s, FN)
#undef FN
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_observe(qhp_system *s) {
  IntArgs a = make_args(s);
  a.part = s->red;
  const size_t smem = s->int_smem;
#define FN(PP)                                                                               \
  {                                                                                          \
    QHP_CUDA_OK(s, set_smem(k_observe<PP>, smem));                                           \
    k_observe<PP><<<s->n_tiles, s->tile_threads, smem, s->stream>>>(a, make_tab<PP>(s->T_P, PP), make_tab<PP>(s->T_Pc, s->Pc)); \
  }
  QHP_DISPATCH_P(s, FN)
#undef FN
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

// pair-energy partials live behind the tile partials in s->red: [4*n_tiles .. 4*n_tiles + n_pair)
int qhp_nm_observe_final(qhp_system *s, int n_pair) {
  k_observe_final<<<1, 256, 0, s->stream>>>(s->red, s->n_tiles, s->red + 4 * (size_t)s->n_tiles, n_pair, s->obs,
                                            s->N, s->P, s->Pc, QHP_KB * s->T);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_to_modes(qhp_system *s, const double *xb, const double *pb) {
  const long long ND = 3LL * s->N;
  const int tb = 128;
  const unsigned grid = (unsigned)((ND + tb - 1) / tb);
#define FN(PP) k_to_modes<PP><<<grid, tb, 0, s->stream>>>(xb, pb, s->Q, s->Pm, ND, make_tab<PP>(s->T_P, PP));
  QHP_DISPATCH_P(s, FN)
#undef FN
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_to_beads(qhp_system *s, double *xb, double *pb) {
  const long long ND = 3LL * s->N;
  const int tb = 128;
  const unsigned grid = (unsigned)((ND + tb - 1) / tb);
#define FN(PP) k_to_beads<PP><<<grid, tb, 0, s->stream>>>(s->Q, s->Pm, xb, pb, ND, make_tab<PP>(s->T_P, PP));
  QHP_DISPATCH_P(s, FN)
#undef FN
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_contract(qhp_system *s, bool rebuild_mode, bool force) {
  const long long ND = 3LL * s->N;
  const int tb = 256;
  const unsigned grid = (unsigned)((ND + tb - 1) / tb);
  const double th = 0.5 * s->skin;
  // in rebuild mode the kernel reads the statistic written by the last integrator pass
  const unsigned long long *flag = (rebuild_mode && !force) ? &s->d2max[s->flag_idx] : nullptr;
  BoxArg bx;
  for (int d = 0; d < 3; ++d) { bx.box[d] = s->box[d]; bx.inv_box[d] = s->inv_box[d]; }
  k_contract<<<grid, tb, 0, s->stream>>>(bx, s->Q, s->N, s->Pc, s->d_Tc, s->rank, s->dt_.type, s->dt_.molid,
                                        s->pos4, rebuild_mode ? s->cent4 : nullptr, s->cref, nullptr, 0,
                                        flag, th * th, (long long *)s->counters);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

int qhp_nm_contracted_out(qhp_system *s, double *xc) {
  const long long ND = 3LL * s->N;
  const int tb = 256;
  const unsigned grid = (unsigned)((ND + tb - 1) / tb);
  k_contract<<<grid, tb, 0, s->stream>>>(BoxArg{}, s->Q, s->N, s->Pc, s->d_Tc, nullptr, s->dt_.type, s->dt_.molid,
                                        nullptr, nullptr, nullptr, xc, 1, nullptr, 0.0, nullptr);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}
