/*
 * qhp_oracle.c -- plain, slow, single-threaded fp64 CPU ORACLE for the Quantum-HP hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with the CUDA path (paper_2212_03137_b200/csrc); the two sides only agree
 * on the Philox4x32-10 *specification* and on the paper's formulas.
 *
 * Written from /root/reference/PAPER.md (arXiv 2212.03137); "PAPER.md:<line>" cites it.
 * Where the paper is silent the reading is SURVEY.md §8(c) (O1..O11, G1..G23), restated in
 * DESIGN.md "Readings".  No blocking, fusion or reordering beyond what the formulas state.
 *
 * Units: Angstrom, ps, amu, kcal/mol, K, e.  Momenta in amu*A/ps; forces in kcal/mol/A and
 * multiplied by QO_ACC = 418.4 when they act on momenta.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see the header of each function.
 * Parity unpinned (beyond GPU-vs-oracle agreement): gamma_z(omega) trajectories and energies
 * on the water boxes (no closed form, no printed value in the paper).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -o libqhp_oracle.so qhp_oracle.c -lm
 * (-ffp-contract=off: the neighbour-object arithmetic must not be fused implicitly; the
 * explicit fma() calls below are part of its definition.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define QO_KB   1.987204258640832e-3   /* kcal/mol/K */
#define QO_HBAR 1.5178728306651436e-2  /* kcal/mol*ps */
#define QO_ACC  418.4                  /* kcal/mol -> amu A^2/ps^2 */
#define QO_COUL 332.063713             /* kcal*A/(mol*e^2) */
#define QO_PI   3.14159265358979323846

typedef struct {
  int32_t n_atoms, n_types, n_bonds, n_angles;
  const int32_t *type, *mol;
  const double *mass, *charge, *lj_eps, *lj_sigma;
  const double *tether_k;                 /* [n_types] or NULL: V = 1/2 k |x|^2 (harmonic pins) */
  const int32_t *bond_idx;  const double *bond_k, *bond_r0;
  const int32_t *angle_idx; const double *angle_k, *angle_th0;
  double box[3];
  double r_cut, dsf_alpha, skin;
} qo_topology;

/* ------------------------------------------------------------------------------------------
 * O6  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): counter-based generator.
 * Pin: the three published known-answer vectors (tests/golden/philox4x32_10_kat.txt).
 * ------------------------------------------------------------------------------------------ */
void qo_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Three standard normals of one (atom, mode, step) of stream `tag` (3 = PILE, 4 = QTB white
 * noise).  key = (seed_lo, seed_hi); counter = (atom, mode | tag<<24, step_lo, step_hi);
 * u_k = (w_k + 0.5) 2^-32; Box-Muller.  SURVEY.md O6. */
void qo_normals3(uint64_t seed, uint32_t atom, uint32_t mode, uint32_t tag, uint64_t step,
                 double z[3]) {
  uint32_t ctr[4] = { atom, mode | (tag << 24), (uint32_t)step, (uint32_t)(step >> 32) };
  uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
  uint32_t w[4];
  qo_philox4x32_10(ctr, key, w);
  const double s = 1.0 / 4294967296.0;
  double u0 = ((double)w[0] + 0.5) * s, u1 = ((double)w[1] + 0.5) * s;
  double u2 = ((double)w[2] + 0.5) * s, u3 = ((double)w[3] + 0.5) * s;
  double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
  z[0] = r0 * cos(2.0 * QO_PI * u1);
  z[1] = r0 * sin(2.0 * QO_PI * u1);
  z[2] = r1 * cos(2.0 * QO_PI * u3);
}

/* ------------------------------------------------------------------------------------------
 * O1  Normal-mode matrix T^(P) and frequencies (Eq. 2 and Eq. 4).
 * Columns = eigenvectors of the cyclic matrix of Eq. 2, ascending eigenvalue; cos before sin
 * inside each degenerate pair (reading G1).  T[i*P + n].
 * Pins: T^T T = I, T^T A T = diag(4 sin^2(pi k/P)) to 1e-14; P = 2 special case.
 * ------------------------------------------------------------------------------------------ */
static int qo_mode_k(int P, int n) {           /* wave number k(n) */
  if (n == 0) return 0;
  if (P % 2 == 0 && n == P - 1) return P / 2;
  return (n + 1) / 2;
}

void qo_nm_matrix(int P, double *T) {
  for (int i = 0; i < P; ++i) {
    T[i * P + 0] = 1.0 / sqrt((double)P);
    for (int n = 1; n < P; ++n) {
      int k = qo_mode_k(P, n);
      if (P % 2 == 0 && n == P - 1)
        T[i * P + n] = ((i % 2) ? -1.0 : 1.0) / sqrt((double)P);
      else if (n % 2 == 1)
        T[i * P + n] = sqrt(2.0 / P) * cos(2.0 * QO_PI * (double)k * (double)i / (double)P);
      else
        T[i * P + n] = sqrt(2.0 / P) * sin(2.0 * QO_PI * (double)k * (double)i / (double)P);
    }
  }
}

/* omega_n = (2 P kB T / hbar) sin(pi k(n) / P): square roots of the eigenvalues of Eq. 2
 * (physical beta: the scaled normal modes absorb the factor P, reading G6).  rad/ps. */
void qo_nm_freq(int P, double T_K, double *omega) {
  for (int n = 0; n < P; ++n)
    omega[n] = 2.0 * P * QO_KB * T_K / QO_HBAR * sin(QO_PI * (double)qo_mode_k(P, n) / (double)P);
}

/* Q_n = (1/sqrt P) sum_i T[i][n] x_i  (Q_0 = centroid).  x, Q: [P][ndof]. */
void qo_beads_to_nm(int P, int64_t ndof, const double *x, double *Q) {
  double *T = (double *)malloc(sizeof(double) * P * P);
  qo_nm_matrix(P, T);
  double sp = sqrt((double)P);
  for (int n = 0; n < P; ++n)
    for (int64_t d = 0; d < ndof; ++d) {
      double s = 0.0;
      for (int i = 0; i < P; ++i) s += T[i * P + n] * x[(int64_t)i * ndof + d];
      Q[(int64_t)n * ndof + d] = s / sp;
    }
  free(T);
}

/* x_i = sqrt(P) sum_n T[i][n] Q_n   (= Eq. 4, since sqrt(P) T[i][0] = 1). */
void qo_nm_to_beads(int P, int64_t ndof, const double *Q, double *x) {
  double *T = (double *)malloc(sizeof(double) * P * P);
  qo_nm_matrix(P, T);
  double sp = sqrt((double)P);
  for (int i = 0; i < P; ++i)
    for (int64_t d = 0; d < ndof; ++d) {
      double s = 0.0;
      for (int n = 0; n < P; ++n) s += T[i * P + n] * Q[(int64_t)n * ndof + d];
      x[(int64_t)i * ndof + d] = sp * s;
    }
  free(T);
}

/* ------------------------------------------------------------------------------------------
 * O2  Ring-polymer contraction (Eq. 20): the Pc lowest-frequency amplitudes
 * Q_n of the full polymer fed unchanged into the Pc-bead transform (literal reading G3).
 * Pins: C(P,P) = I; C(P,1) = 1/P; rows sum to 1.
 * ------------------------------------------------------------------------------------------ */
/* Variant of reading G3 (default 0 = literal Eq. 20).  1 = trigonometric interpolation: for even Pc < P the
 * highest contracted mode is the Nyquist mode of the Pc-bead polymer but the cos member of a degenerate pair
 * of the full one; evaluating the band-limited interpolant of the P beads at the Pc points gives that mode
 * the amplitude sqrt(2) Q_{Pc-1} (the sin partner vanishes there).  Pins (tests/test_oracle_nm.py): equals
 * scipy.signal.resample of the bead positions; C(P,P) = I; odd Pc unchanged; forces = -gradient. */
static int qo_contraction_variant = 0;
void qo_set_contraction_variant(int v) { qo_contraction_variant = v; }
static double qo_top_mode_scale(int P, int Pc) {
  return (qo_contraction_variant == 1 && Pc % 2 == 0 && Pc < P) ? sqrt(2.0) : 1.0;
}

void qo_contract(int P, int Pc, int64_t ndof, const double *Q, double *xc) {
  double sc = qo_top_mode_scale(P, Pc);
  if (sc == 1.0) { qo_nm_to_beads(Pc, ndof, Q, xc); return; }   /* uses rows n < Pc of Q only ([P][ndof] layout) */
  double *Qs = (double *)malloc(sizeof(double) * (size_t)Pc * ndof);
  memcpy(Qs, Q, sizeof(double) * (size_t)Pc * ndof);
  for (int64_t d = 0; d < ndof; ++d) Qs[(int64_t)(Pc - 1) * ndof + d] *= sc;
  qo_nm_to_beads(Pc, ndof, Qs, xc);
  free(Qs);
}

/* f^s_n = (1/sqrt Pc) sum_j T^(Pc)[j][n] Fc_j for n < Pc, 0 otherwise (chain rule on Eq. 20). */
void qo_expand_force(int P, int Pc, int64_t ndof, const double *Fc, double *fs) {
  qo_beads_to_nm(Pc, ndof, Fc, fs);
  double sc = qo_top_mode_scale(P, Pc);
  if (sc != 1.0) for (int64_t d = 0; d < ndof; ++d) fs[(int64_t)(Pc - 1) * ndof + d] *= sc;
  for (int64_t e = (int64_t)Pc * ndof; e < (int64_t)P * ndof; ++e) fs[e] = 0.0;
}

/* ------------------------------------------------------------------------------------------
 * O3  Potential (BASELINE.json configs[0]; V = V_s + V_f, Eq. 18).
 * V_f: harmonic bonds 1/2 k (r-r0)^2, harmonic angles 1/2 k (th-th0)^2, optional tether.
 * Positions are unwrapped; bonded terms use plain differences.
 * Pins: central finite differences; sum F = 0 (without tether).
 * ------------------------------------------------------------------------------------------ */
double qo_force_fast(const qo_topology *t, const double *x, double *F) {
  double U = 0.0;
  for (int b = 0; b < t->n_bonds; ++b) {
    int i = t->bond_idx[2 * b], j = t->bond_idx[2 * b + 1];
    double d[3] = { x[3*i] - x[3*j], x[3*i+1] - x[3*j+1], x[3*i+2] - x[3*j+2] };
    double r = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
    double dr = r - t->bond_r0[b];
    U += 0.5 * t->bond_k[b] * dr * dr;
    double g = -t->bond_k[b] * dr / r;
    for (int c = 0; c < 3; ++c) { F[3*i+c] += g * d[c]; F[3*j+c] -= g * d[c]; }
  }
  for (int a = 0; a < t->n_angles; ++a) {
    int i = t->angle_idx[3*a], j = t->angle_idx[3*a+1], k = t->angle_idx[3*a+2]; /* j = centre */
    double u[3], v[3];
    for (int c = 0; c < 3; ++c) { u[c] = x[3*i+c] - x[3*j+c]; v[c] = x[3*k+c] - x[3*j+c]; }
    double ru = sqrt(u[0]*u[0] + u[1]*u[1] + u[2]*u[2]);
    double rv = sqrt(v[0]*v[0] + v[1]*v[1] + v[2]*v[2]);
    double cs = (u[0]*v[0] + u[1]*v[1] + u[2]*v[2]) / (ru * rv);
    if (cs > 1.0) cs = 1.0;
    if (cs < -1.0) cs = -1.0;
    double th = acos(cs);
    double dth = th - t->angle_th0[a];
    U += 0.5 * t->angle_k[a] * dth * dth;
    double sn = sqrt(1.0 - cs * cs);
    double g = t->angle_k[a] * dth / sn;      /* = -dV/dth * dth/dcos */
    for (int c = 0; c < 3; ++c) {
      double fi = g * (v[c] / (ru * rv) - cs * u[c] / (ru * ru));
      double fk = g * (u[c] / (ru * rv) - cs * v[c] / (rv * rv));
      F[3*i+c] += fi; F[3*k+c] += fk; F[3*j+c] -= fi + fk;
    }
  }
  if (t->tether_k)
    for (int i = 0; i < t->n_atoms; ++i) {
      double k = t->tether_k[t->type[i]];
      for (int c = 0; c < 3; ++c) { U += 0.5 * k * x[3*i+c] * x[3*i+c]; F[3*i+c] -= k * x[3*i+c]; }
    }
  return U;
}

/* One intermolecular pair inside the cutoff: O-O style Lennard-Jones (Lorentz-Berthelot mixing,
 * potential shifted to 0 at r_c) + damped-shifted-force Coulomb (Fennell-Gezelter), SURVEY O3.
 * d = x_i - x_j (minimum image), r2 = |d|^2 < rc^2.  Adds to F_i, subtracts from F_j. */
static double qo_pair(const qo_topology *t, int i, int j, const double d[3], double r2,
                      double *F) {
  double rc = t->r_cut, al = t->dsf_alpha;
  double r = sqrt(r2);
  double qq = QO_COUL * t->charge[t->type[i]] * t->charge[t->type[j]];
  double two_a_sqrtpi = 2.0 * al / sqrt(QO_PI);
  double erfc_rc = erfc(al * rc) / rc;
  double fshift = erfc(al * rc) / (rc * rc) + two_a_sqrtpi * exp(-al * al * rc * rc) / rc;
  double U = qq * (erfc(al * r) / r - erfc_rc + fshift * (r - rc));
  double fmag = qq * (erfc(al * r) / r2 + two_a_sqrtpi * exp(-al * al * r2) / r - fshift);
  double ei = t->lj_eps[t->type[i]], ej = t->lj_eps[t->type[j]];
  if (ei > 0.0 && ej > 0.0) {
    double eps = sqrt(ei * ej);
    double sig = 0.5 * (t->lj_sigma[t->type[i]] + t->lj_sigma[t->type[j]]);
    double s6 = pow(sig / r, 6.0), c6 = pow(sig / rc, 6.0);
    U += 4.0 * eps * (s6 * s6 - s6) - 4.0 * eps * (c6 * c6 - c6);
    fmag += 24.0 * eps * (2.0 * s6 * s6 - s6) / r;
  }
  for (int c = 0; c < 3; ++c) {
    double f = fmag * d[c] / r;
    F[3*i+c] += f; F[3*j+c] -= f;
  }
  return U;
}

/* minimum-image difference and squared distance with the explicit-fma arithmetic of O4 */
static double qo_min_image(const qo_topology *t, const double *xi, const double *xj, double d[3]) {
  for (int c = 0; c < 3; ++c) {
    double L = t->box[c], invL = 1.0 / L;
    double dx = xi[c] - xj[c];
    d[c] = fma(-L, rint(dx * invL), dx);
  }
  return fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
}

/* V_s by O(N^2) brute force over all i<j in different molecules (one periodic replica). */
double qo_force_slow_brute(const qo_topology *t, const double *x, double *F) {
  double U = 0.0, rc2 = t->r_cut * t->r_cut;
  for (int i = 0; i < t->n_atoms; ++i)
    for (int j = i + 1; j < t->n_atoms; ++j) {
      if (t->mol[i] == t->mol[j]) continue;
      double d[3];
      double r2 = qo_min_image(t, x + 3*i, x + 3*j, d);
      if (r2 < rc2) U += qo_pair(t, i, j, d, r2, F);
    }
  return U;
}

/* V_s with the oracle's own simple cell list built on THIS replica's positions (cells >= r_c,
 * 27-cell stencil); used for N too large for O(N^2).  Pin: equals qo_force_slow_brute on
 * small boxes (tests).  Falls back to brute force when a box edge holds < 3 cells. */
double qo_force_slow_cells(const qo_topology *t, const double *x, double *F) {
  int nc[3];
  for (int c = 0; c < 3; ++c) nc[c] = (int)floor(t->box[c] / t->r_cut);
  if (nc[0] < 3 || nc[1] < 3 || nc[2] < 3) return qo_force_slow_brute(t, x, F);
  int N = t->n_atoms, ncell = nc[0] * nc[1] * nc[2];
  int *head = (int *)malloc(sizeof(int) * ncell), *next = (int *)malloc(sizeof(int) * N);
  int *cid = (int *)malloc(sizeof(int) * 3 * N);
  for (int c = 0; c < ncell; ++c) head[c] = -1;
  for (int i = N - 1; i >= 0; --i) {
    int q[3];
    for (int c = 0; c < 3; ++c) {
      double s = x[3*i+c] / t->box[c];
      s -= floor(s);
      q[c] = (int)(s * nc[c]);
      if (q[c] >= nc[c]) q[c] = nc[c] - 1;
      cid[3*i+c] = q[c];
    }
    int cell = (q[0] * nc[1] + q[1]) * nc[2] + q[2];
    next[i] = head[cell]; head[cell] = i;
  }
  double U = 0.0, rc2 = t->r_cut * t->r_cut;
  for (int i = 0; i < N; ++i)
    for (int ox = -1; ox <= 1; ++ox) for (int oy = -1; oy <= 1; ++oy) for (int oz = -1; oz <= 1; ++oz) {
      int cx = (cid[3*i] + ox + nc[0]) % nc[0], cy = (cid[3*i+1] + oy + nc[1]) % nc[1];
      int cz = (cid[3*i+2] + oz + nc[2]) % nc[2];
      for (int j = head[(cx * nc[1] + cy) * nc[2] + cz]; j >= 0; j = next[j]) {
        if (j <= i || t->mol[i] == t->mol[j]) continue;
        double d[3];
        double r2 = qo_min_image(t, x + 3*i, x + 3*j, d);
        if (r2 < rc2) U += qo_pair(t, i, j, d, r2, F);
      }
    }
  free(head); free(next); free(cid);
  return U;
}

/* ------------------------------------------------------------------------------------------
 * O4  Neighbour objects on centroid positions (lists "computed with respect to
 * centroid positions", shared by all beads).  Canonical integer objects, bit-exact contract.
 * Pins: permutation / prefix-sum invariants; pair set by brute force is the definition.
 * ------------------------------------------------------------------------------------------ */
void qo_cells(const qo_topology *t, const double *c, int32_t nc[3], int32_t *cell_of,
              int32_t *order, int32_t *cell_start) {
  double rl = t->r_cut + t->skin;
  for (int d = 0; d < 3; ++d) { nc[d] = (int)floor(t->box[d] / rl); if (nc[d] < 1) nc[d] = 1; }
  int N = t->n_atoms, ncell = nc[0] * nc[1] * nc[2];
  for (int i = 0; i < N; ++i) {
    int q[3];
    for (int d = 0; d < 3; ++d) {
      double invL = 1.0 / t->box[d];
      double s = c[3*i+d] * invL;
      s = s - floor(s);
      q[d] = (int)(s * (double)nc[d]);
      if (q[d] > nc[d] - 1) q[d] = nc[d] - 1;
    }
    cell_of[i] = (q[0] * nc[1] + q[1]) * nc[2] + q[2];
  }
  for (int k = 0; k <= ncell; ++k) cell_start[k] = 0;
  for (int i = 0; i < N; ++i) cell_start[cell_of[i] + 1]++;
  for (int k = 0; k < ncell; ++k) cell_start[k + 1] += cell_start[k];
  int *fill = (int *)malloc(sizeof(int) * (ncell > 0 ? ncell : 1));
  for (int k = 0; k < ncell; ++k) fill[k] = cell_start[k];
  for (int i = 0; i < N; ++i) order[fill[cell_of[i]]++] = i;    /* stable: ties by atom index */
  free(fill);
}

/* Pair set {(i,j): i<j, mol_i != mol_j, d2 < r_list^2}, lexicographic order, by brute force.
 * Returns the number of pairs; writes at most `cap` of them into pairs[2*k], pairs[2*k+1]. */
int64_t qo_pairs_brute(const qo_topology *t, const double *c, int32_t *pairs, int64_t cap) {
  double rl = t->r_cut + t->skin, rl2 = rl * rl;
  int64_t n = 0;
  for (int i = 0; i < t->n_atoms; ++i)
    for (int j = i + 1; j < t->n_atoms; ++j) {
      if (t->mol[i] == t->mol[j]) continue;
      double d[3];
      double d2 = qo_min_image(t, c + 3*i, c + 3*j, d);
      if (d2 < rl2) { if (n < cap) { pairs[2*n] = i; pairs[2*n+1] = j; } ++n; }
    }
  return n;
}

/* Neighbours of ONE atom i (all j != i, other molecule, d2 < r_list^2), ascending j: lets the
 * tests sample the pair set of boxes too large for qo_pairs_brute.  Returns the count. */
int32_t qo_neighbours_of(const qo_topology *t, const double *c, int32_t i, int32_t *nb, int32_t cap) {
  double rl = t->r_cut + t->skin, rl2 = rl * rl;
  int32_t n = 0;
  for (int j = 0; j < t->n_atoms; ++j) {
    if (j == i || t->mol[i] == t->mol[j]) continue;
    double d[3];
    double d2 = (i < j) ? qo_min_image(t, c + 3*i, c + 3*j, d) : qo_min_image(t, c + 3*j, c + 3*i, d);
    if (d2 < rl2) { if (n < cap) nb[n] = j; ++n; }
  }
  return n;
}

/* ------------------------------------------------------------------------------------------
 * O5 steps 5-7 + O8: normal-mode forces f_n(Q) and potential energies.
 *   x = NM->bead(Q) (Eq. 4); xc = contract(Q) (Eq. 20); F^f_i = -grad V_f(x_i);
 *   Fc_j = -grad V_s(xc_j); f_n = (1/sqrt P) sum_i T[i][n] F^f_i + f^s_n  (Eq. 10-11).
 * e[0] = (1/P) sum_i V_f(x_i), e[1] = (1/Pc) sum_j V_s(xc_j)  (Eq. 20).
 * ------------------------------------------------------------------------------------------ */
void qo_nm_forces(const qo_topology *t, int P, int Pc, const double *Q, double *f, double e[2],
                  int use_cells) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *x = (double *)malloc(sizeof(double) * P * nd);
  double *Ff = (double *)calloc((size_t)(P * nd), sizeof(double));
  double *xc = (double *)malloc(sizeof(double) * Pc * nd);
  double *Fc = (double *)calloc((size_t)(Pc * nd), sizeof(double));
  double *fs = (double *)malloc(sizeof(double) * P * nd);
  qo_nm_to_beads(P, nd, Q, x);
  qo_contract(P, Pc, nd, Q, xc);
  double uf = 0.0, us = 0.0;
  for (int i = 0; i < P; ++i) uf += qo_force_fast(t, x + i * nd, Ff + i * nd);
  for (int j = 0; j < Pc; ++j)
    us += use_cells ? qo_force_slow_cells(t, xc + j * nd, Fc + j * nd)
                    : qo_force_slow_brute(t, xc + j * nd, Fc + j * nd);
  qo_beads_to_nm(P, nd, Ff, f);
  qo_expand_force(P, Pc, nd, Fc, fs);
  for (int64_t k = 0; k < P * nd; ++k) f[k] += fs[k];
  if (e) { e[0] = uf / P; e[1] = us / Pc; }
  free(x); free(Ff); free(xc); free(Fc); free(fs);
}

/* O7: bead-space forces G_i = F^f_i + (P/Pc) sum_j C[j][i] Fc_j  with the contraction matrix
 * C = (sqrt Pc / sqrt P) T^(Pc) [I 0] T^(P)^T written out (independent route from qo_nm_forces;
 * the test pins G == NM->bead(f)).  G: [P][ndof]. */
void qo_bead_forces(const qo_topology *t, int P, int Pc, const double *xb, double *G, int use_cells) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *T = (double *)malloc(sizeof(double) * P * P), *Tc = (double *)malloc(sizeof(double) * Pc * Pc);
  double *C = (double *)malloc(sizeof(double) * Pc * P);
  qo_nm_matrix(P, T); qo_nm_matrix(Pc, Tc);
  for (int j = 0; j < Pc; ++j) for (int i = 0; i < P; ++i) {
    double s = 0.0;
    for (int n = 0; n < Pc; ++n) s += (n == Pc - 1 ? qo_top_mode_scale(P, Pc) : 1.0) * Tc[j * Pc + n] * T[i * P + n];
    C[j * P + i] = sqrt((double)Pc) / sqrt((double)P) * s;
  }
  double *xc = (double *)calloc((size_t)(Pc * nd), sizeof(double));
  double *Fc = (double *)calloc((size_t)(Pc * nd), sizeof(double));
  for (int j = 0; j < Pc; ++j) for (int i = 0; i < P; ++i) for (int64_t d = 0; d < nd; ++d)
    xc[j * nd + d] += C[j * P + i] * xb[i * nd + d];
  memset(G, 0, sizeof(double) * P * nd);
  for (int i = 0; i < P; ++i) qo_force_fast(t, xb + i * nd, G + i * nd);
  for (int j = 0; j < Pc; ++j) {
    if (use_cells) qo_force_slow_cells(t, xc + j * nd, Fc + j * nd);
    else qo_force_slow_brute(t, xc + j * nd, Fc + j * nd);
  }
  for (int i = 0; i < P; ++i) for (int j = 0; j < Pc; ++j) for (int64_t d = 0; d < nd; ++d)
    G[i * nd + d] += (double)P / (double)Pc * C[j * P + i] * Fc[j * nd + d];
  free(T); free(Tc); free(C); free(xc); free(Fc);
}

/* O8 observables: out[0] = K_CV = (3N/2) kB T - 1/2 sum_{n>0} Q_n . f_n ; out[1] = U (Eq. 20);
 * out[2] = K_nm = sum_n Pm_n^2 / 2m (kcal/mol); out[3] = T_inst = 2 K_nm / (3 N P kB). */
void qo_observables(const qo_topology *t, int P, int Pc, double T_K, const double *Q,
                    const double *Pm, double out[4], int use_cells) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *f = (double *)malloc(sizeof(double) * P * nd);
  double e[2];
  qo_nm_forces(t, P, Pc, Q, f, e, use_cells);
  double vir = 0.0, k = 0.0;
  for (int n = 1; n < P; ++n) for (int64_t d = 0; d < nd; ++d) vir += Q[n * nd + d] * f[n * nd + d];
  for (int n = 0; n < P; ++n) for (int64_t d = 0; d < nd; ++d) {
    double m = t->mass[t->type[d / 3]];
    k += Pm[n * nd + d] * Pm[n * nd + d] / (2.0 * m);
  }
  out[0] = 1.5 * t->n_atoms * QO_KB * T_K - 0.5 * vir;
  out[1] = e[0] + e[1];
  out[2] = k / QO_ACC;
  out[3] = 2.0 * out[2] / (3.0 * t->n_atoms * P * QO_KB);
  free(f);
}

/* ------------------------------------------------------------------------------------------
 * O5  RPMD step: B(dt/2) A(dt/2) O(dt) A(dt/2) B(dt/2) in normal modes (PAPER.md:144-149,
 * Eq. 16-17).  gamma_n = max(gamma0, omega_n) for n > 0, gamma0 for the centroid (l.146);
 * exact Ornstein-Uhlenbeck O step (reading G5).  thermo: 0 = none (skip O), 1 = PILE/TRPMD.
 * State: Q, Pm, f ([P][3N]; f = NM force at the current Q, must be valid on entry).
 * Pins: A block conserves each mode's energy; c1^2 + c2^2 = 1; P = 1 == classical BAOAB;
 * harmonic <q^2> closed form (statistical).
 * ------------------------------------------------------------------------------------------ */
/* A(dt/2) O(dt) A(dt/2) of one step (O5 items 2-4), shared by qo_rpmd_steps and qo_rpmd_respa_steps */
/* a_block = 0: exact harmonic A(dt/2) (Eq. 17).  a_block = 1: the BCOCB variant ("the exact
 * integration of e^{iL_A dt/2} is replaced by a numerical scheme", ref. [66] of the paper): the half-step
 * is the square root of the Cayley transform cay(dt A) = (1 - dt A/2)^-1 (1 + dt A/2) of the free
 * ring-polymer generator A = [[0, 1/m], [-m w^2, 0]] of each mode, whose closed form is
 *   cay(dt A)^(1/2) = (1 + (w dt/2)^2)^(-1/2) [[1, dt/(2m)], [-m w^2 dt/2, 1]]        (reading G25)
 * (a rotation by atan(w dt/2) instead of w dt/2; the centroid, w = 0, is the same translation). */
static void qo_aoa(const qo_topology *t, int P, double dt, double T_K, int thermo, double gamma0,
                   uint64_t seed, int64_t step, const double *om, double *Q, double *Pm, int a_block) {
  int N = t->n_atoms;
  int64_t nd = 3 * (int64_t)N;
  for (int half = 0; half < 2; ++half) {
    /* 2./4. A(dt/2): centroid translation, exact harmonic rotation of the fluctuation modes */
    for (int n = 0; n < P; ++n) for (int a = 0; a < N; ++a) {
      double m = t->mass[t->type[a]];
      for (int c = 0; c < 3; ++c) {
        int64_t k = n * nd + 3 * a + c;
        if (n == 0) { Q[k] += 0.5 * dt * Pm[k] / m; }
        else if (a_block == 1) {
          double w = om[n], a = 0.5 * w * dt, nrm = 1.0 / sqrt(1.0 + a * a);
          double q = Q[k], p = Pm[k];
          Q[k]  = nrm * (q + 0.5 * dt / m * p);
          Pm[k] = nrm * (-m * w * w * 0.5 * dt * q + p);
        }
        else {
          double w = om[n], cs = cos(w * 0.5 * dt), sn = sin(w * 0.5 * dt);
          double q = Q[k], p = Pm[k];
          Q[k]  = cs * q + sn / (m * w) * p;
          Pm[k] = -m * w * sn * q + cs * p;
        }
      }
    }
    /* 3. O(dt) between the two A half-steps */
    if (half == 0 && thermo == 1)
      for (int n = 0; n < P; ++n) {
        double g = (n == 0) ? gamma0 : (gamma0 > om[n] ? gamma0 : om[n]);
        double c1 = exp(-g * dt), c2 = sqrt(1.0 - c1 * c1);
        for (int a = 0; a < N; ++a) {
          double z[3];
          qo_normals3(seed, (uint32_t)a, (uint32_t)n, 3u, (uint64_t)step, z);
          double sg = sqrt(t->mass[t->type[a]] * QO_KB * T_K * QO_ACC);
          for (int c = 0; c < 3; ++c) {
            int64_t k = n * nd + 3 * a + c;
            Pm[k] = c1 * Pm[k] + sg * c2 * z[c];
          }
        }
      }
  }
}

static void qo_rpmd_steps_ab(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                             double gamma0, uint64_t seed, int64_t step0, int64_t nsteps,
                             double *Q, double *Pm, double *f, int use_cells, int a_block) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *om = (double *)malloc(sizeof(double) * P);
  qo_nm_freq(P, T_K, om);
  for (int64_t s = 0; s < nsteps; ++s) {
    /* 1. B(dt/2) */
    for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * dt * QO_ACC * f[k];
    qo_aoa(t, P, dt, T_K, thermo, gamma0, seed, step0 + s, om, Q, Pm, a_block);
    /* 5.-7. forces at the new positions */
    qo_nm_forces(t, P, Pc, Q, f, NULL, use_cells);
    /* 8. B(dt/2) */
    for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * dt * QO_ACC * f[k];
  }
  free(om);
}

void qo_rpmd_steps(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                   double gamma0, uint64_t seed, int64_t step0, int64_t nsteps,
                   double *Q, double *Pm, double *f, int use_cells) {
  qo_rpmd_steps_ab(t, P, Pc, dt, T_K, thermo, gamma0, seed, step0, nsteps, Q, Pm, f, use_cells, 0);
}

/* NEXT-3  BCOCB: B(dt/2) C(dt/2) O(dt) C(dt/2) B(dt/2), C = cay(dt A)^(1/2) (see qo_aoa).
 * Pins (tests/test_oracle_bcocb.py): C^2 equals the Cayley matrix from a linear solve and C equals
 * scipy's matrix square root of it; det C = 1; the mode's harmonic energy is conserved exactly; C agrees
 * with the exact rotation to O((w dt)^3); time reversal; second order; w dt -> large stays bounded. */
void qo_rpmd_steps_bcocb(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                         double gamma0, uint64_t seed, int64_t step0, int64_t nsteps,
                         double *Q, double *Pm, double *f, int use_cells) {
  qo_rpmd_steps_ab(t, P, Pc, dt, T_K, thermo, gamma0, seed, step0, nsteps, Q, Pm, f, use_cells, 1);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-1  BAOAB-RESPA (Eq. 19): V = V_s + V_f (Eq. 18),
 *   Bs(n_alt dt/2) [ Bf(dt/2) A(dt/2) O(dt) A(dt/2) Bf(dt/2) ]^{n_alt} Bs(n_alt dt/2)
 * with V_f on all P beads and V_s on the Pc contracted beads (Eq. 20).
 * ff, fs: normal-mode forces of V_f and V_s at the current Q (both valid on entry and on exit).
 * `step0` counts INNER steps (one Philox step index per O block); n_outer outer steps are taken.
 * Pins (tests/test_oracle_respa.py): n_alt = 1 reproduces qo_rpmd_steps; V_s = 0 reproduces plain
 * BAOAB with dt; time reversal; second-order convergence to the single-step trajectory;
 * conservation of the ring-polymer Hamiltonian without thermostat.
 * ------------------------------------------------------------------------------------------ */
void qo_nm_forces_split(const qo_topology *t, int P, int Pc, const double *Q, double *ff, double *fs,
                        int use_cells) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *x = (double *)malloc(sizeof(double) * P * nd);
  double *Ff = (double *)calloc((size_t)(P * nd), sizeof(double));
  double *xc = (double *)malloc(sizeof(double) * Pc * nd);
  double *Fc = (double *)calloc((size_t)(Pc * nd), sizeof(double));
  if (ff) {
    qo_nm_to_beads(P, nd, Q, x);
    for (int i = 0; i < P; ++i) qo_force_fast(t, x + i * nd, Ff + i * nd);
    qo_beads_to_nm(P, nd, Ff, ff);
  }
  if (fs) {
    qo_contract(P, Pc, nd, Q, xc);
    for (int j = 0; j < Pc; ++j) {
      if (use_cells) qo_force_slow_cells(t, xc + j * nd, Fc + j * nd);
      else qo_force_slow_brute(t, xc + j * nd, Fc + j * nd);
    }
    qo_expand_force(P, Pc, nd, Fc, fs);
  }
  free(x); free(Ff); free(xc); free(Fc);
}

static void qo_rpmd_respa_steps_ab(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                                   double gamma0, uint64_t seed, int64_t step0, int64_t n_outer, int n_alt,
                                   double *Q, double *Pm, double *ff, double *fs, int use_cells, int a_block) {
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *om = (double *)malloc(sizeof(double) * P);
  qo_nm_freq(P, T_K, om);
  for (int64_t o = 0; o < n_outer; ++o) {
    /* Bs(n_alt dt/2) */
    for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * n_alt * dt * QO_ACC * fs[k];
    for (int j = 0; j < n_alt; ++j) {
      /* Bf(dt/2) A O A Bf(dt/2) */
      for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * dt * QO_ACC * ff[k];
      qo_aoa(t, P, dt, T_K, thermo, gamma0, seed, step0 + o * n_alt + j, om, Q, Pm, a_block);
      qo_nm_forces_split(t, P, Pc, Q, ff, NULL, use_cells);
      for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * dt * QO_ACC * ff[k];
    }
    /* Bs(n_alt dt/2) with V_s at the new positions */
    qo_nm_forces_split(t, P, Pc, Q, NULL, fs, use_cells);
    for (int64_t k = 0; k < P * nd; ++k) Pm[k] += 0.5 * n_alt * dt * QO_ACC * fs[k];
  }
  free(om);
}

void qo_rpmd_respa_steps(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                         double gamma0, uint64_t seed, int64_t step0, int64_t n_outer, int n_alt,
                         double *Q, double *Pm, double *ff, double *fs, int use_cells) {
  qo_rpmd_respa_steps_ab(t, P, Pc, dt, T_K, thermo, gamma0, seed, step0, n_outer, n_alt, Q, Pm, ff, fs, use_cells, 0);
}

/* RESPA with the BCOCB half-steps in the inner loop: Bs [Bf C O C Bf]^{n_alt} Bs (same pins as both parents:
 * n_alt = 1 reproduces qo_rpmd_steps_bcocb, tests/test_oracle_bcocb.py) */
void qo_rpmd_respa_steps_bcocb(const qo_topology *t, int P, int Pc, double dt, double T_K, int thermo,
                               double gamma0, uint64_t seed, int64_t step0, int64_t n_outer, int n_alt,
                               double *Q, double *Pm, double *ff, double *fs, int use_cells) {
  qo_rpmd_respa_steps_ab(t, P, Pc, dt, T_K, thermo, gamma0, seed, step0, n_outer, n_alt, Q, Pm, ff, fs, use_cells, 1);
}

/* ------------------------------------------------------------------------------------------
 * O10  QTB kernel (Eq. 13-14).
 * Theta(omega) = (hbar omega / 2) / tanh(beta hbar omega / 2), Theta(0) = kB T   (Eq. 14).
 * Pins: Theta -> kB T (classical) and hbar omega/2 (T -> 0); equals
 *       hbar omega [1/2 + 1/(exp(beta hbar omega) - 1)] (BASELINE.json north_star form).
 * ------------------------------------------------------------------------------------------ */
double qo_theta(double omega, double T_K) {
  double kT = QO_KB * T_K;
  if (omega == 0.0) return kT;
  double hw = QO_HBAR * fabs(omega);
  return 0.5 * hw / tanh(0.5 * hw / kT);
}

/* H_z(omega_j) = sqrt(2 m_z gamma_z(omega_j) Theta(omega_j) / dt), j = 0..n_seg, on the grid
 * omega_j = 2 pi j / (N_k dt), N_k = 2 n_seg; m_z = mass/418.4 so that H is in kcal/mol/A.
 * `classical` != 0 replaces Theta by kB T (hbar -> 0 limit, pin "adQTB classical limit"). */
void qo_qtb_filter(int n_seg, double dt, double T_K, double mass_amu, const double *gamma_z,
                   int classical, double *H) {
  int nk = 2 * n_seg;
  for (int j = 0; j <= n_seg; ++j) {
    double w = 2.0 * QO_PI * j / (nk * dt);
    double th = classical ? QO_KB * T_K : qo_theta(w, T_K);
    H[j] = sqrt(2.0 * (mass_amu / QO_ACC) * gamma_z[j] * th / dt);
  }
}

/* Kernel-correction hook (reading G11; PAPER.md:203 cites corrections "for finite timestep [33] and
 * non-zero friction [35]" without defining them): H_z(omega_j) <- kappa(omega_j) H_z(omega_j) with a
 * caller-supplied real factor kappa[j], j = 0..n_seg (amplitude factor: the noise PSD of Eq. 13 gets
 * kappa^2).  kappa == NULL is the identity.
 * Pins (tests/test_oracle_adqtb.py): kappa == 1 bit-identical; kappa = sqrt(kB T / Theta) gives the
 * classical kernel h[k != 0] = 0 and the white-noise BAOAB trajectory; F_c linear in a constant kappa. */
void qo_qtb_filter_kappa(int n_seg, double dt, double T_K, double mass_amu, const double *gamma_z,
                         int classical, const double *kappa, double *H) {
  qo_qtb_filter(n_seg, dt, T_K, mass_amu, gamma_z, classical, H);
  if (kappa)
    for (int j = 0; j <= n_seg; ++j) H[j] = kappa[j] * H[j];
}

/* h[k] = (1/N_k) sum_{j=0}^{N_k-1} H(omega_j) exp(+2 pi i j k / N_k), k = -n_seg..n_seg-1,
 * with H extended evenly (H_{N_k - j} = H_j): real and even.  Stored at h[k + n_seg].
 * Pins: DFT_{N_k}(h) = H; h even; Theta == kB T, gamma const  =>  h[k != 0] = 0. */
void qo_qtb_kernel(int n_seg, const double *H, double *h) {
  int nk = 2 * n_seg;
  for (int k = -n_seg; k < n_seg; ++k) {
    double s = 0.0;
    for (int j = 0; j < nk; ++j) {
      double Hj = (j <= n_seg) ? H[j] : H[nk - j];
      /* reduce j*k mod N_k in integers so the phase stays accurate */
      int64_t jk = ((int64_t)j * k) % nk; if (jk < 0) jk += nk;
      s += Hj * cos(2.0 * QO_PI * (double)jk / (double)nk);
    }
    h[k + n_seg] = s / nk;
  }
}

/* F_c[dof][n] = sum_{k=-n_seg}^{n_seg-1} h_z[k] r(dof, seg*n_seg + n - k + n_seg), n = 0..n_seg-1,
 * r(dof, s) = Philox normal of (atom, tag 4, step s) (readings G10, G17).  Direct sum.
 * h_types: [n_types][2 n_seg].  Fc: [3N][n_seg].
 * Pin: concatenated segments = one long direct convolution ("memory consistent between
 * segments"). */
void qo_qtb_colored_direct(const qo_topology *t, int n_seg, uint64_t seed, int64_t seg,
                           const double *h_types, double *Fc) {
  int nw = 3 * n_seg;
  double *r = (double *)malloc(sizeof(double) * 3 * nw);
  for (int a = 0; a < t->n_atoms; ++a) {
    for (int s = 0; s < nw; ++s) {
      double z[3];
      qo_normals3(seed, (uint32_t)a, 0u, 4u, (uint64_t)(seg * n_seg + s), z);
      r[s] = z[0]; r[nw + s] = z[1]; r[2 * nw + s] = z[2];
    }
    const double *h = h_types + (int64_t)t->type[a] * 2 * n_seg;
    for (int c = 0; c < 3; ++c)
      for (int n = 0; n < n_seg; ++n) {
        double acc = 0.0;
        for (int k = -n_seg; k < n_seg; ++k) acc += h[k + n_seg] * r[c * nw + n - k + n_seg];
        Fc[((int64_t)3 * a + c) * n_seg + n] = acc;
      }
  }
}

/* White-noise window of one atom (3 x 3 n_seg normals, component-major) for FFT-based variants
 * in the Python wrapper and for the PSD pin. */
void qo_qtb_white(uint64_t seed, int32_t atom, int64_t s0, int32_t count, double *r) {
  for (int s = 0; s < count; ++s) {
    double z[3];
    qo_normals3(seed, (uint32_t)atom, 0u, 4u, (uint64_t)(s0 + s), z);
    r[s] = z[0]; r[count + s] = z[1]; r[2 * count + s] = z[2];
  }
}

/* ------------------------------------------------------------------------------------------
 * O9  adQTB step = classical BAOAB carrying the coloured force (Eq. 12; l.199
 * "only replaces the white noise random forces").  P = 1.
 *   a = exp(-gamma0 dt), b = sqrt((1-a^2) dt / (2 gamma0))      (reading G16)
 *   v_seg[dof][n] = (p_before_O + p_after_O) / 2m               (reading G14)
 * x, p, F: [3N]; F = -grad V(x) valid on entry.  Fc, vseg: [3N][n_seg]; runs local steps
 * n0..n0+nsteps-1 of the current segment.
 * Pin: Theta == kB T  =>  identical to white-noise BAOAB driven by r(dof, n + n_seg).
 * ------------------------------------------------------------------------------------------ */
void qo_adqtb_steps(const qo_topology *t, double dt, double gamma0, int n_seg, int n0, int nsteps,
                    double *x, double *p, double *F, const double *Fc, double *vseg, int use_cells) {
  int N = t->n_atoms;
  int64_t nd = 3 * (int64_t)N;
  double a = exp(-gamma0 * dt), b = sqrt((1.0 - a * a) * dt / (2.0 * gamma0));
  for (int s = 0; s < nsteps; ++s) {
    int n = n0 + s;
    for (int64_t d = 0; d < nd; ++d) {
      double m = t->mass[t->type[d / 3]];
      p[d] += 0.5 * dt * QO_ACC * F[d];
      x[d] += 0.5 * dt * p[d] / m;
      double pn = a * p[d] + b * QO_ACC * Fc[d * n_seg + n];
      vseg[d * n_seg + n] = (p[d] + pn) / (2.0 * m);
      p[d] = pn;
      x[d] += 0.5 * dt * p[d] / m;
    }
    memset(F, 0, sizeof(double) * nd);
    qo_force_fast(t, x, F);
    if (use_cells) qo_force_slow_cells(t, x, F); else qo_force_slow_brute(t, x, F);
    for (int64_t d = 0; d < nd; ++d) p[d] += 0.5 * dt * QO_ACC * F[d];
  }
}

/* total force F = -grad(V_f + V_s)(x) of one replica; returns U. */
double qo_force_total(const qo_topology *t, const double *x, double *F, int use_cells) {
  memset(F, 0, sizeof(double) * 3 * (size_t)t->n_atoms);
  double u = qo_force_fast(t, x, F);
  u += use_cells ? qo_force_slow_cells(t, x, F) : qo_force_slow_brute(t, x, F);
  return u;
}

/* ------------------------------------------------------------------------------------------
 * O11  Segment spectra, per-type averages (Eq. 21-22), direct DFT.
 *   V_j = sum_{n<n_seg} v[n] exp(-2 pi i j n / N_k)  (zero-padded N_k-point DFT, reading G12)
 *   C_vv,i = (dt/n_seg) |V_j|^2,  Re C_vF,i = (dt/n_seg) Re(V_j conj(Phi_j))   (reading G13)
 * Cvv, CvF: [n_types][n_seg+1] = means over the DOFs of each type.
 * Pin: np.fft.rfft of the zero-padded segment; Parseval.
 * ------------------------------------------------------------------------------------------ */
void qo_qtb_spectra_direct(const qo_topology *t, int n_seg, double dt, const double *vseg,
                           const double *Fc, double *Cvv, double *CvF) {
  int nk = 2 * n_seg, nf = n_seg + 1;
  int64_t nd = 3 * (int64_t)t->n_atoms;
  double *cnt = (double *)calloc((size_t)t->n_types, sizeof(double));
  double *cs = (double *)malloc(sizeof(double) * nk), *sn = (double *)malloc(sizeof(double) * nk);
  for (int m = 0; m < nk; ++m) { cs[m] = cos(2.0 * QO_PI * m / nk); sn[m] = sin(2.0 * QO_PI * m / nk); }
  memset(Cvv, 0, sizeof(double) * t->n_types * nf);
  memset(CvF, 0, sizeof(double) * t->n_types * nf);
  for (int64_t d = 0; d < nd; ++d) {
    int z = t->type[d / 3];
    cnt[z] += 1.0;
    for (int j = 0; j < nf; ++j) {
      double vr = 0, vi = 0, fr = 0, fi = 0;
      for (int n = 0; n < n_seg; ++n) {
        int m = (int)(((int64_t)j * n) % nk);
        vr += vseg[d * n_seg + n] * cs[m]; vi -= vseg[d * n_seg + n] * sn[m];
        fr += Fc[d * n_seg + n] * cs[m];   fi -= Fc[d * n_seg + n] * sn[m];
      }
      Cvv[z * nf + j] += dt / n_seg * (vr * vr + vi * vi);
      CvF[z * nf + j] += dt / n_seg * (vr * fr + vi * fi);
    }
  }
  for (int z = 0; z < t->n_types; ++z) for (int j = 0; j < nf; ++j)
    if (cnt[z] > 0) { Cvv[z * nf + j] /= cnt[z]; CvF[z * nf + j] /= cnt[z]; }
  free(cnt); free(cs); free(sn);
}

/* SIMPLE adaptation (Eq. 23) with the scale-free rate of reading G15 and the
 * lower bound of PAPER.md:248:
 *   Delta_z = m_z gamma_z Cvv_z - Re CvF_z     (Eq. 21, m_z = mass/418.4)
 *   gamma_z <- max(gmin_frac gamma0, gamma_z - A gamma0 Delta_z / ||Delta_z||_2)
 * Pin: hand-computed toy case (tests/golden/adapt_toy.txt). */
void qo_qtb_adapt(int n_types, int n_seg, const double *mass_amu, double gamma0, double a_gamma,
                  double gmin_frac, const double *Cvv, const double *CvF, double *gamma) {
  int nf = n_seg + 1;
  double *dl = (double *)malloc(sizeof(double) * nf);
  for (int z = 0; z < n_types; ++z) {
    double nrm = 0.0;
    for (int j = 0; j < nf; ++j) {
      dl[j] = mass_amu[z] / QO_ACC * gamma[z * nf + j] * Cvv[z * nf + j] - CvF[z * nf + j];
      nrm += dl[j] * dl[j];
    }
    nrm = sqrt(nrm);
    if (nrm == 0.0) continue;
    for (int j = 0; j < nf; ++j) {
      double g = gamma[z * nf + j] - a_gamma * gamma0 * dl[j] / nrm;
      double gmin = gmin_frac * gamma0;
      gamma[z * nf + j] = g > gmin ? g : gmin;
    }
  }
  free(dl);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-2  RATIO adaptation (Eq. 24-26) for the types with tau[z] > 0:
 *   <C>_tau^(k) = <C>_tau^(k-1) w + C^(k) (1 - w),  w = exp(-N_seg dt / tau_z)          (Eq. 26)
 *   gamma_z(omega_j) = Re<C_vF,z>(omega_j) / (m_z <C_vv,z>(omega_j))                    (Eq. 25)
 *   gamma_z <- max(gamma_min, gamma_z)                                                  (l.248)
 * avv, avf: the running averages [n_types][n_seg+1], in/out.  Reading G24 (paper silent on k = 1):
 * the first segment initialises the averages with its own spectra (`first` != 0).  A bin whose
 * averaged C_vv is not positive keeps its gamma.  m_z in kcal/mol ps^2/A^2 as in O10/O11.
 * Types with tau[z] <= 0 are left untouched (SIMPLE, qo_qtb_adapt, handles them).
 * Pins (tests/test_oracle_ratio.py): closed form of the window recursion; Eq. 24 (a gamma with
 * Delta_FDT = 0 under the SIMPLE definition is a fixed point); the free-particle ratio (1 - a)/b.
 * ------------------------------------------------------------------------------------------ */
void qo_qtb_adapt_ratio(int n_types, int n_seg, const double *mass_amu, double gamma0, double gmin_frac,
                        double dt, const double *tau, int first, const double *Cvv, const double *CvF,
                        double *avv, double *avf, double *gamma) {
  int nf = n_seg + 1;
  double gmin = gmin_frac * gamma0;
  for (int z = 0; z < n_types; ++z) {
    if (!(tau[z] > 0.0)) continue;
    double w = first ? 0.0 : exp(-(double)n_seg * dt / tau[z]);
    for (int j = 0; j < nf; ++j) {
      int k = z * nf + j;
      avv[k] = avv[k] * w + Cvv[k] * (1.0 - w);
      avf[k] = avf[k] * w + CvF[k] * (1.0 - w);
      double den = mass_amu[z] / QO_ACC * avv[k];
      if (den > 0.0) {
        double g = avf[k] / den;
        gamma[k] = g > gmin ? g : gmin;
      }
    }
  }
}


/* ------------------------------------------------------------------------------------------
 * NEXT-5  PI-BAR free-energy estimator (Eq. 27-28).
 *   dF_AB = beta^-1 ln(Z_A/Z_B) = C + beta^-1 ln( <f(U_A - U_B + C)>_B / <f(U_B - U_A - C)>_A ),   (27)
 *   C = dF_AB + beta^-1 ln(n_B / n_A),   f(x) = 1 / (1 + exp(beta x)),                               (28)
 * "a self-consistent set of equations that is solved iteratively" (l.304).
 * Inputs are the stored series of bead-averaged potential differences (U of Eq. 3):
 *   wA[i] = U_B - U_A on the n_A configurations sampled in state A,
 *   wB[j] = U_A - U_B on the n_B configurations sampled in state B.
 * Reading G26 (paper silent): start from dF = 0; one iteration = Eq. 28 then Eq. 27; stop when
 * |dF_new - dF| <= tol or after max_iter iterations; returns the number of iterations done.
 * With U = V on a single bead this is the estimator of Appendix A (Eq. A1); with P = 1 it is BAR.
 * Pins (tests/test_oracle_pibar.py): U_B = U_A + c gives c exactly; the fixed point solves Bennett's
 * implicit equation sum_A f = sum_B f (root found with scipy.optimize.brentq); dF_BA = -dF_AB;
 * classical and finite-P quantum harmonic oscillators against their closed-form partition functions.
 * ------------------------------------------------------------------------------------------ */
static double qo_fermi(double beta, double x) { return 1.0 / (1.0 + exp(beta * x)); }

int qo_pibar(const double *wA, int64_t nA, const double *wB, int64_t nB, double beta, int max_iter,
             double tol, double *dF_out) {
  double dF = 0.0;
  int it = 0;
  while (it < max_iter) {
    double C = dF + log((double)nB / (double)nA) / beta;                /* Eq. 28 */
    double sB = 0.0, sA = 0.0;
    for (int64_t j = 0; j < nB; ++j) sB += qo_fermi(beta, wB[j] + C);   /* <f(U_A - U_B + C)>_B */
    for (int64_t i = 0; i < nA; ++i) sA += qo_fermi(beta, wA[i] - C);   /* <f(U_B - U_A - C)>_A */
    double dF_new = C + log((sB / (double)nB) / (sA / (double)nA)) / beta;   /* Eq. 27 */
    double change = fabs(dF_new - dF);
    dF = dF_new;
    ++it;
    if (change <= tol) break;
  }
  *dF_out = dF;
  return it;
}
