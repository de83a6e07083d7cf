// qhp_internal.cuh -- internal declarations of the B200 (sm_100a) Quantum-HP hot path.
// Shared by the translation units of libqhp.so only; nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/qhp.h"

// ---- physical constants (SURVEY.md §8(c) "Units and constants", CODATA 2018) ---------------
#define QHP_KB 1.987204258640832e-3    // kcal/mol/K
#define QHP_HBAR 1.5178728306651436e-2 // kcal/mol*ps
#define QHP_ACC 418.4                  // kcal/mol -> amu A^2/ps^2
#define QHP_COUL 332.063713            // kcal*A/(mol*e^2)
#define QHP_PI 3.14159265358979323846

#define QHP_MAX_P 32
#define QHP_MAX_TYPES 8
#define QHP_NPOLY 16   // degree-15 polynomials of the damped Coulomb kernel (pair_staged.cu): truncation ~1e-16 at alpha r_c = 1.8

// Philox stream tags
#define QHP_TAG_PILE 3u
#define QHP_TAG_QTB 4u

// One CTA of the integrator handles one tile = a run of whole molecules.
struct qhp_tile {
  int32_t a0, a1; // atoms [a0, a1)
  int32_t m0, m1; // molecules [m0, m1)
};

// Per-(type, mode) coefficients of the A and O blocks, laid out [type][mode][QHP_NCOEF].
#define QHP_NCOEF 6
// 0: cos(w dt/2)  1: sin/(m w)  2: -m w sin  3: c1 = exp(-g dt)  4: sqrt(m kB T ACC) c2  5: 1/m (unused for n>0)

struct qhp_dev_topology {
  int32_t *type;   // [N]
  int32_t *molid;  // [N] dense molecule index 0..n_mol-1
  int32_t *mol_atom_start;  // [n_mol+1]
  int32_t *mol_bond_start;  // [n_mol+1]
  int32_t *mol_angle_start; // [n_mol+1]
  int32_t *bond_idx;  double *bond_k, *bond_r0;   // sorted by molecule
  int32_t *angle_idx; double *angle_k, *angle_th0;
  double *mass;      // [nt]
  double *tether_k;  // [nt] (zeros when absent)
  qhp_tile *tiles;   // [n_tiles]
};

struct qhp_system {
  // ---- configuration (host) ----
  int N = 0, nt = 0, n_mol = 0, n_bonds = 0, n_angles = 0;
  int P = 1, Pc = 1;
  int a_block = 0;                         // 0: exact A(dt/2); 1: BCOCB half-step sqrt(cay(dt A))
  int n_alt = 1;                           // BAOAB-RESPA: inner steps per V_s kick (Eq. 19); 1 = plain BAOAB
  double dt = 0, T = 0;
  qhp_thermostat th{};
  double box[3]{}, inv_box[3]{};
  double r_cut = 0, alpha = 0, skin = 0;
  bool has_tether = false;
  cudaStream_t stream = nullptr;
  int device = 0;
  std::string err;

  // ---- host tables ----
  std::vector<double> mass, charge, lj_eps, lj_sigma;
  std::vector<double> T_P, T_Pc;      // normal-mode matrices T^(P) [i*P+n], T^(Pc)
  std::vector<double> omega;          // [P]

  // ---- device state ----
  qhp_dev_topology dt_{};
  int n_tiles = 0, tile_atoms = 0, tile_threads = 0;
  size_t int_smem = 0;
  bool int_mol1 = false;                   // P = 1 and molecules of <= 4 atoms: thread-per-molecule integrator
  double *Q = nullptr, *Pm = nullptr;      // [P][3N] normal modes
  double *coef = nullptr;                  // [nt][P][QHP_NCOEF]
  double *d_Tc = nullptr;                  // [Pc][Pc] T^(Pc) on the device
  int flag_idx = 0;                        // slot of d2max written by the last integrator pass
  double *pos4 = nullptr;                  // [Pc][N] double4 (x,y,z,type bits) in slot order
  double *Fs = nullptr;                    // [Pc][N][3] slow forces in slot order
  double *cent4 = nullptr;                 // [N] double4 (centroid xyz, molecule bits) in slot order
  double *cref = nullptr;                  // [3N] centroids at the last list build (atom order)
  double *pair_tab = nullptr;              // [nt*nt][4]: qq, 48 eps s^12, 24 eps s^6, (4 eps s^12, 4 eps s^6, shift) ...
  // cells and list
  int nc[3]{1, 1, 1}, ncell = 1;
  int32_t *cell_of = nullptr, *cell_count = nullptr, *cell_start = nullptr, *cell_cursor = nullptr;
  int32_t *cell_tmp = nullptr, *order = nullptr, *rank = nullptr;
  int32_t *cell_key = nullptr;             // [N] sub-cell Morton key of the atom inside its cell (internal slot order)
  int coop_blocks = 0;                     // resident CTAs of the fused (cooperative) cell kernel; 0 = four separate kernels
  int32_t *nbr = nullptr, *nbr_count = nullptr;
  int64_t nbr_stride = 0;
  // staged pair kernel (pair.cu): one CTA stages the 27-cell neighbourhood of a cell in shared
  // memory; the list then holds 16-bit indices into that staged array instead of slots
  bool staged_ok = false;                  // geometry allows it (>= 4 cells per dimension, polynomial fits)
  bool staged = false;                     // in use (decided at the synchronising list build)
  uint16_t *nbr16 = nullptr;               // [N][nbr_stride]
  int staged_cap = 0;                      // staged atoms that fit in shared memory
  int staged_warps = 0, staged_smem_max = 0; // CTA size in use, dynamic shared memory available
  bool staged_f32 = true;                  // the staged kernel keeps an 8-byte fp16 copy for the packed-half pre-test (else fp64 pre-test)
  double staged_thr = 0.0;                 // threshold of that pre-test (r_c^2 + its error bound, a half)
  int staged_split = 1;                    // CTAs per (cell, bead)
  // pruned per-bead rows + evaluation without pre-test (k_prune, k_pair_dense in pair_staged.cu)
  double prune_skin = 0.6;                 // A; <= 0: off (qhp_set_pair_prune); 0.6: best of the 0.3-1.0 sweep at C3 and C4
  bool dense = false;                      // in use (decided with `staged` at the synchronising list build)
  int dense_cap = 0;                       // staged atoms of k_pair_dense (two CTAs per SM)
  uint16_t *nbr16p = nullptr;              // [Pc][N][nbr_stride] pruned rows
  int32_t *nbr_count_p = nullptr;          // [Pc][N]
  int64_t nbr16p_stride = 0;               // stride the pruned table was allocated for
  double *pref4 = nullptr;                 // [Pc][N][4] bead positions at the last prune
  double *prune_part = nullptr;            // [Pc][PRUNE_CHECK_CTAS] displacement maxima of k_prune_check
  long long *pruned_at = nullptr;          // [Pc] rebuild count the pruned rows belong to (-1: none)
  int *prune_work = nullptr;               // [Pc] work counters of k_prune
  double polyS[QHP_NPOLY]{}, polyE[QHP_NPOLY]{};   // alpha^3 S(w), alpha E(w) in u = 2 r^2/rc^2 - 1
  unsigned long long *d2max = nullptr;     // [2] double bits, max |xc - cref|^2, double-buffered by step parity
  int64_t *counters = nullptr;             // [8] device: 0 rebuilds, 1 overflow flag, 2 max row count, 3 in-cutoff count, 6 skin-too-small flag
  double *red = nullptr;                   // scratch for reductions
  size_t red_len = 0;
  double *obs = nullptr;                   // [8] device observables
  double *stage_x = nullptr, *stage_p = nullptr;  // device staging of the *_host calls
  // adQTB
  int n_seg = 0;
  double *gamma = nullptr;   // [nt][n_seg+1]
  double *Hf = nullptr;      // [nt][n_seg+1] filter H_z
  double *hk = nullptr;      // [nt][2 n_seg] kernel h_z
  double *H4 = nullptr;      // [nt][4 n_seg][2] spectrum of the zero-padded shifted kernel
  // segment arrays F_c, v_seg: [n_groups][n_seg][12]: groups of 4 "segment slots" (atoms sorted by type, every
  // type padded to a multiple of 4), one 96-byte row (4 atoms x 3 components) per step: sector-exact per-step
  // access for the integrator, one contiguous n_seg x 96 B region per group for the per-segment FFT kernels
  double *Fc = nullptr, *vseg = nullptr;
  int32_t *seg_slot = nullptr;    // [N] atom -> segment slot
  int32_t *slot_atom = nullptr;   // [n_slots] segment slot -> atom (-1: padding)
  int n_slots = 0;
  double *tw = nullptr;      // twiddles exp(-2 pi i k / NT) [NT][2], NT = 4 n_seg
  std::vector<int> type_start;     // [nt+1] offsets into atoms_by_type
  int32_t *spec_cta = nullptr;     // [n_spec_cta][3] (type, first group, end group)
  int n_spec_cta = 0;
  std::vector<int> spec_cta_host;
  double *spec_part = nullptr;     // [n_spec_cta][2][n_seg+1]
  double *Cvv = nullptr, *CvF = nullptr; // [nt][n_seg+1]
  int64_t fc_segment = -1;
  double *ratio_tau = nullptr;             // [nt] ps, > 0: RATIO adaptation of that type (Eq. 24-26); NULL: SIMPLE for all
  double *ratio_avv = nullptr, *ratio_avf = nullptr;   // [nt][n_seg+1] exponential-window averages (Eq. 26)
  double *kappa = nullptr;                 // [n_seg+1] kernel-correction factor on H (reading G11); NULL: 1
  bool ratio_started = false;

  // ---- bead-sharded V_s (qhp_set_comm): this rank evaluates the contracted beads
  //      [rank Pc/world, (rank + 1) Pc/world) and the ranks all-gather F_s (bead-major: one contiguous block each) ----
  int shard_rank = 0, shard_world = 1;
  qhp_allgather_fn shard_allgather = nullptr;
  void *shard_ctx = nullptr;

  // ---- error flags seen without a synchronisation (qhp_step): async copy of `counters` into pinned memory + event ----
  int64_t *flags_host = nullptr;
  cudaEvent_t flags_ev = nullptr;
  bool flags_pending = false;

  // ---- CUDA graph of QHP_GRAPH_STEPS steps for small, launch-bound systems (qhp_step) ----
  cudaGraphExec_t graph_exec = nullptr;
  cudaStream_t graph_stream = nullptr;     // capture stream (the caller's may be the legacy default stream)
  long long *graph_step_base = nullptr;    // device: offset added to the step indices baked into the graph (Philox counters)
  int64_t graph_step0 = 0;                 // step index the graph was captured at
  int64_t graph_launches = 0;              // kernel launches inside one replay
  bool graph_capturing = false, graph_off = false;

  // ---- per-phase profiling (qhp_profile) ----
  bool prof = false;
  std::vector<cudaEvent_t> prof_ev;      // flat list of (begin, end) pairs
  std::vector<int> prof_kind;            // phase of each pair
  double prof_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // 0-4: phases of qhp_profile_read; 5-7: k_prune_check, k_prune, k_pair_dense
  int64_t prof_n[8] = {0, 0, 0, 0, 0, 0, 0, 0};

  // ---- run state (host) ----
  bool have_state = false;
  bool pending_kick = false;   // the final B(dt/2) of the last step has not been applied yet
  int64_t step = 0;
  int64_t n_launch = 0;        // kernels launched (for bench gpu_launches)
};

// ---- launch helpers implemented in the .cu files ----------------------------------------------
// nm_kernels.cu
int qhp_nm_to_modes(qhp_system *s, const double *xb, const double *pb);          // beads -> Q, Pm
int qhp_nm_to_beads(qhp_system *s, double *xb, double *pb);                      // Q, Pm -> beads
int qhp_nm_integrate(qhp_system *s, bool kick_prev, bool do_step, int64_t step); // fused pass
int qhp_nm_contract(qhp_system *s, bool rebuild_mode, bool force);               // Q -> pos4 (+ cent4, cref)
int qhp_nm_bead_forces(qhp_system *s, double *G);                                 // O7
int qhp_nm_observe(qhp_system *s);                                                // partial sums -> s->red
int qhp_nm_observe_final(qhp_system *s, int n_pair);                              // s->red -> s->obs
int qhp_nm_contracted_out(qhp_system *s, double *xc);
// cells.cu
int qhp_cells_rebuild(qhp_system *s, bool force);   // early-exits on device unless needed/forced
int qhp_cells_setup(qhp_system *s);                 // cooperative-launch capacity of the fused cell kernel
int qhp_cells_canonical_order(qhp_system *s, int32_t *order_out);   // parity hook: ties by atom index
int qhp_cells_export(qhp_system *s, int32_t *count, int32_t *nbr, int64_t cap, int64_t *total_host);
// pair.cu
int qhp_pair_forces(qhp_system *s, bool energy);     // pos4 -> Fs (+ U_s, count into obs/counters); bead-sharded if qhp_set_comm
int qhp_pair_forces_beads(qhp_system *s, bool energy, int bead0, int nbeads);   // the launch of one bead slice
int qhp_pair_setup(qhp_system *s);                   // polynomial tables, staged-kernel geometry
bool qhp_pair_staged_fit(qhp_system *s, long long region);  // CTA size / capacity for a neighbourhood size
int qhp_pair_dense_prepare(qhp_system *s, long long region); // pruned-row path: decide, (re)allocate, invalidate
void qhp_pair_dense_free(qhp_system *s);
int qhp_pair_prune_stats_impl(qhp_system *s, int64_t *out_host);
int qhp_pair_partials(const qhp_system *s);          // upper bound of per-CTA energy partials
// qtb.cu
int qhp_qtb_init(qhp_system *s);
int qhp_qtb_generate(qhp_system *s, int64_t seg);
int qhp_qtb_adapt(qhp_system *s);
int qhp_qtb_export_segment(qhp_system *s, const double *in, double *out);   // internal layout -> [3N][n_seg]
int qhp_fft_launch(double *data, int n, int64_t batch, int sign, const double *tw, int tw_n, cudaStream_t st);

#define QHP_CUDA_OK(s, call)                                                          \
  do {                                                                                \
    cudaError_t e_ = (call);                                                          \
    if (e_ != cudaSuccess) {                                                          \
      (s)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                  \
      return QHP_ECUDA;                                                               \
    }                                                                                 \
  } while (0)

#define QHP_LAUNCH_OK(s)                                                              \
  do {                                                                                \
    cudaError_t e_ = cudaGetLastError();                                              \
    if (e_ != cudaSuccess) {                                                          \
      (s)->err = std::string("kernel launch: ") + cudaGetErrorString(e_);             \
      return QHP_ECUDA;                                                               \
    }                                                                                 \
    (s)->n_launch++;                                                                  \
  } while (0)

// address of (segment slot s, component c, step n) in the segment arrays F_c / v_seg
__host__ __device__ __forceinline__ long long qhp_seg_addr(int slot, int n_seg, int n) {
  return ((long long)(slot >> 2) * n_seg + n) * 12 + (slot & 3) * 3;
}

// CUDA events around a phase (or one launch) on the library stream while qhp_profile is on
struct qhp_prof_scope {
  qhp_system *s; bool on;
  qhp_prof_scope(qhp_system *s_, int kind) : s(s_), on(s_->prof) {
    if (!on) return;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    s->prof_ev.push_back(a); s->prof_ev.push_back(b); s->prof_kind.push_back(kind);
    cudaEventRecord(a, s->stream);
    idx = s->prof_ev.size() - 1;
  }
  ~qhp_prof_scope() { if (on) cudaEventRecord(s->prof_ev[idx], s->stream); }
  size_t idx = 0;
};

void qhp_global_error(const char *msg);   // qhp_api.cu: error text of a call without a system handle (qhp_last_error(NULL))
