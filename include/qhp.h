/*
 * qhp.h -- C ABI of the B200-native Quantum-HP hot path (RPMD + adQTB MD step).
 *
 * What it computes is defined by /root/reference/PAPER.md (arXiv 2212.03137); citations are
 * "PAPER.md:<line>, Eq. n".  Readings of passages where the paper is silent (G1..G23) are in
 * DESIGN.md "Readings".  The force field (flexible 3-site water: harmonic bonds/angles,
 * Lennard-Jones, damped-shifted-force Coulomb) is BASELINE.json configs[0], not the paper's.
 *
 * Conventions
 *   units     Angstrom, ps, amu, kcal/mol, K, e.  Momenta amu*A/ps; forces kcal/mol/A.
 *   layouts   x_beads, p_beads, f_beads: fp64 [P][n_atoms][3], bead-major ("replicas",
 *             PAPER.md:32).  Momenta are bead momenta p_i = sqrt(P) sum_n T_in Pm_n (the map of
 *             Eq. 4).  Internally the state lives in scaled normal modes (Eq. 1-4).
 *   pointers  every pointer in qhp_topology / qhp_thermostat is a HOST pointer, deep-copied by
 *             qhp_create.  Array arguments of all other calls are DEVICE pointers on the device
 *             of the stream given to qhp_create, unless the function name ends in _host, in
 *             which case they are HOST pointers and the call copies synchronously.
 *   ownership the caller owns every buffer it passes; the library owns the qhp_system and all
 *             device state behind it until qhp_destroy.
 *   async     all calls enqueue work on the stream given at create time and return without
 *             synchronising, except qhp_create / qhp_destroy / qhp_set_state (builds the first
 *             neighbour list and sizes its storage) / *_host calls / qhp_check.
 *   errors    every call returns 0 (QHP_OK) or a negative qhp_status; text in qhp_last_error.
 *             No exceptions, no abort, no stdout.  There is no CPU fallback of any call.
 */
#ifndef QHP_H
#define QHP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  QHP_OK = 0,
  QHP_EINVAL = -1,  /* bad argument (P < 1, unsupported P, P_contract not in [1,P], box < 2 r_cut, ...) */
  QHP_ENOMEM = -2,  /* device or host allocation failed */
  QHP_ECUDA = -3,   /* CUDA error (sticky); text via qhp_last_error */
  QHP_ESTATE = -4   /* call out of order (step before set_state, adQTB restart inside a segment,
                       neighbour-list capacity overflow detected at a synchronising call) */
} qhp_status;

typedef struct qhp_system qhp_system; /* opaque */

/* Topology and force field (BASELINE.json configs[0]; V = V_s + V_f, Eq. 18).
 * Molecules must be contiguous in atom index (mol[] non-decreasing), bonds and angles join
 * atoms of one molecule, and a molecule has at most QHP_MAX_MOL_ATOMS atoms.  Atom pairs of the
 * same molecule are excluded from V_s. */
#define QHP_MAX_MOL_ATOMS 48
typedef struct {
  int32_t n_atoms, n_types, n_bonds, n_angles;
  const int32_t *type;     /* [n_atoms] atom type z (adQTB averages per type)     */
  const int32_t *mol;      /* [n_atoms] molecule id                                            */
  const double *mass;      /* [n_types] amu                                                    */
  const double *charge;    /* [n_types] e                                                      */
  const double *lj_eps;    /* [n_types] kcal/mol (0 => no LJ); Lorentz-Berthelot mixing        */
  const double *lj_sigma;  /* [n_types] Angstrom                                               */
  const double *tether_k;  /* [n_types] or NULL: extra V_f term 1/2 k |x|^2 (harmonic pins)    */
  const int32_t *bond_idx; /* [n_bonds][2]                                                     */
  const double *bond_k;    /* [n_bonds] kcal/mol/A^2, V = 1/2 k (r - r0)^2                     */
  const double *bond_r0;   /* [n_bonds] A                                                      */
  const int32_t *angle_idx;/* [n_angles][3] (end, centre, end)                                 */
  const double *angle_k;   /* [n_angles] kcal/mol/rad^2, V = 1/2 k (th - th0)^2                */
  const double *angle_th0; /* [n_angles] rad                                                   */
  double box[3];           /* orthorhombic periodic box, A; every edge >= 2 r_cut              */
  double r_cut;            /* V_s cutoff (LJ shifted, DSF Coulomb), A                          */
  double dsf_alpha;        /* DSF damping, 1/A                                                 */
  double skin;             /* neighbour-list skin, A: r_list = r_cut + skin     */
} qhp_topology;

typedef enum { QHP_THERMO_NONE = 0, QHP_THERMO_PILE = 1, QHP_THERMO_ADQTB = 2 } qhp_thermo_kind;

typedef struct {
  int32_t kind;          /* qhp_thermo_kind                                                     */
  double gamma0;         /* 1/ps: PILE centroid friction / adQTB gamma_0 (Eq. 12)*/
  uint64_t seed;         /* Philox4x32-10 key                                                   */
  int32_t n_seg;         /* adQTB: steps per noise segment, a power of two in [8, 2048]         */
                         /* (the 4 n_seg-point transform of the noise lives in    */
                         /* shared memory: 8192 points = 128 KB is the largest that fits)       */
  double a_gamma;        /* adQTB: adaptation rate A (Eq. 23, reading G15); 0 = no adaptation   */
  double gamma_min_frac; /* adQTB: gamma_z >= gamma_min_frac * gamma0; 0.01      */
  int32_t classical;     /* adQTB: != 0 replaces Theta(omega) by kB T (test hook, hbar -> 0)    */
} qhp_thermostat;

/* Create a system of P beads with V_s evaluated on P_contract <= P contracted beads (ring-polymer
 * contraction, Eq. 20) and V_f on all P.  dt in ps, T in K.  Supported P:
 * 1,2,3,4,5,6,8,12,16,24,32.  adQTB requires P = 1.  cuda_stream is a cudaStream_t (NULL = legacy default
 * stream). */
int qhp_create(const qhp_topology *top, int P, int P_contract, double dt_ps, double T_K,
               const qhp_thermostat *thermo, void *cuda_stream, qhp_system **out);
int qhp_destroy(qhp_system *sys);

/* Load bead positions / momenta (device [P][n_atoms][3]); transforms to normal modes (Eq. 4
 * inverted), builds cells + neighbour list on the centroids and evaluates the
 * forces.  step0 = index of the next step: Philox streams are functions of (seed, atom, mode,
 * step), so get_state -> set_state resumes bit-identically up to the summation order of the freshly built
 * neighbour list.  adQTB: step0 % n_seg == 0; the adapted gamma_z travels through qhp_adqtb_gamma /
 * qhp_adqtb_set_gamma. */
int qhp_set_state(qhp_system *sys, const double *x_beads, const double *p_beads, int64_t step0);
int qhp_get_state(qhp_system *sys, double *x_beads, double *p_beads, int64_t *step_host);
int qhp_set_state_host(qhp_system *sys, const double *x_beads, const double *p_beads, int64_t step0);
int qhp_get_state_host(qhp_system *sys, double *x_beads, double *p_beads, int64_t *step_host);

/* Advance nsteps of B A O A B in normal modes (Eq. 16-17): exact free
 * ring-polymer A blocks, PILE/TRPMD O block gamma_n = max(gamma0, omega_n) (l.146), or, for
 * adQTB, classical BAOAB whose O block carries the coloured force (Eq. 12-14, l.199), with the
 * segment generation (l.203-209) and gamma_z(omega) adaptation (Eq. 21-23, l.248) at segment
 * boundaries.  Enqueues its work and returns; never waits for the device.  Small systems (n_atoms <= 32768, n_alt = 1,
 * no qhp_set_comm, profiling off) are launch-bound: longer calls replay 32 steps at a time from a CUDA graph captured
 * once per state (same kernels and arguments; the Philox step index and the adQTB segment position are taken from
 * device memory; an adQTB replay never crosses a segment boundary): the trajectory is bit-identical to plain
 * launches, qhp_counters counts the replayed kernels.  The sticky error flags of the device
 * (list-row overflow, staged neighbourhood outgrew shared memory, skin smaller than the bead spread: qhp_counters
 * [5]) are copied to pinned memory behind the work of every call and every 256 steps of a long one, and looked at
 * without waiting when qhp_step is entered again or reaches the next 256-step mark: QHP_ESTATE then (text in
 * qhp_last_error); qhp_check reports them at once. */
int qhp_step(qhp_system *sys, int64_t nsteps);

/* BAOAB-RESPA (Eq. 19): Bs(n_alt dt/2) [Bf(dt/2) A O A Bf(dt/2)]^n_alt Bs(n_alt dt/2)
 * with V_f (bonds, angles, tethers; all P beads) in Bf and V_s (LJ + DSF Coulomb; P_contract beads) in
 * Bs.  qhp_step keeps counting INNER steps of dt (one Philox index per O block) and then accepts
 * multiples of n_alt only; V_s and the neighbour objects are evaluated once per n_alt inner steps.
 * n_alt = 1 (default) is plain B A O A B.  Call it at a multiple of n_alt steps (the closing kicks of the
 * last step are applied first, with the n_alt they were taken under); not with adQTB. */
int qhp_set_respa(qhp_system *sys, int n_alt);

/* Contraction variant (reading G3; Eq. 20).  QHP_CONTRACT_LITERAL (default): the
 * P' lowest normal-mode amplitudes of the full polymer are fed unchanged into the P'-bead transform.
 * QHP_CONTRACT_TRIG: the contracted beads are the band-limited (Fourier) interpolant of the P beads at P'
 * points, which differs for even P' < P only: the Nyquist mode of the contracted polymer gets sqrt(2) times
 * the amplitude of the cos member of the degenerate pair it is fed from (the sin partner vanishes at the
 * contracted points); positions and the chain-rule force projection change together.  Call before
 * qhp_set_state (QHP_ESTATE afterwards). */
#define QHP_CONTRACT_LITERAL 0
#define QHP_CONTRACT_TRIG 1
int qhp_set_contraction(qhp_system *sys, int variant);

/* Pruned per-bead rows of the staged pair kernel (an acceleration structure of R8; the centroid
 * table of R7 -- the list the paper describes and the oracle is compared with -- is unchanged).  With
 * prune_skin > 0 (default 0.6 A; must be < the list skin) every contracted bead keeps a second table holding the
 * entries of the centroid table within r_cut + prune_skin of the bead's own positions; V_s is then evaluated on
 * those rows without a per-step pre-test.  A bead's rows are renewed on the device, without a host round trip,
 * when one of its atoms has moved more than prune_skin / 2 since they were made or the centroid table was
 * rebuilt, so the evaluated pair set always contains every pair inside r_cut: forces equal those of the unpruned
 * path up to the summation order.  Costs 2 B x P_contract x N x row stride of device memory.  prune_skin <= 0:
 * off (every step walks the centroid table with the packed-half pre-test).  Before qhp_set_state
 * (QHP_ESTATE afterwards). */
int qhp_set_pair_prune(qhp_system *sys, double prune_skin);
/* Parity hook of the pruned rows.  Makes the rows current for the present state exactly as a step does (displacement
 * check, prune if due), evaluates V_s through them and reports, out_host[4] (HOST): [0] 1 if the pruned-row path serves
 * this system (else the other entries are 0), [1] number of prunes so far (summed over the contracted beads; a step
 * without a prune leaves it unchanged), [2] entries in the pruned rows, [3] ordered pair-beads of those rows that pass
 * the fp64 test r^2 < r_cut^2 -- equal to qhp_counters' pair_beads_in_cutoff (centroid table) iff no pair inside the
 * cutoff is missing.  Synchronises.  After qhp_set_state. */
int qhp_pair_prune_stats(qhp_system *sys, int64_t *out_host);

/* A block of the splitting: QHP_ABLOCK_EXACT (default) = exact harmonic evolution of the
 * fluctuation modes over dt/2 (Eq. 17); QHP_ABLOCK_CAYLEY = the BCOCB variant, whose half-step is the
 * square root of the Cayley transform of the free ring-polymer generator,
 *   (q, p) -> (1 + (w dt/2)^2)^(-1/2) (q + dt/(2m) p, p - m w^2 dt/2 q)      (reading G25),
 * stable for any w dt.  The centroid and P = 1 are unchanged.  May be called at any step. */
#define QHP_ABLOCK_EXACT 0
#define QHP_ABLOCK_CAYLEY 1
int qhp_set_a_block(qhp_system *sys, int kind);

/* Bead-parallel evaluation of V_s over several processes, one GPU each (Sec. III.C: the beads of
 * the -- contracted -- ring polymer are distributed over the ranks of a "polymer" communicator, each rank evaluates
 * the forces of its beads, the forces are gathered and then projected on the normal modes, l.192, l.195).  Every rank
 * holds the whole system and runs the same qhp_* calls (the integrator pass is replicated, so the copies stay
 * bit-identical); after qhp_set_comm(sys, rank, world, fn, ctx) the pair kernel of rank r evaluates the contracted
 * beads [r P'/world, (r + 1) P'/world) only, and the library calls
 *     fn(ctx, Fs, bytes_per_rank, rank, world, cuda_stream)
 * once per V_s evaluation: an IN-PLACE all-gather of the DEVICE buffer Fs (world consecutive blocks of bytes_per_rank
 * bytes, block r valid on rank r on entry, all blocks valid on every rank on return), enqueued on cuda_stream (the
 * stream of qhp_create); return 0 on success.  The caller owns the communicator (NCCL all-gather over NVLink in
 * the Python binding: torch.distributed.all_gather_into_tensor).  world must divide P_contract; world = 1 (or fn =
 * NULL) restores the single-process path.  Observables and the counters hook evaluate every bead locally.  Call before
 * qhp_set_state.  QHP_EINVAL for rank/world out of range or world not dividing P_contract. */
typedef int (*qhp_allgather_fn)(void *ctx, void *device_buf, size_t bytes_per_rank, int rank, int world, void *cuda_stream);
int qhp_set_comm(qhp_system *sys, int rank, int world, qhp_allgather_fn fn, void *ctx);
/* Test hook of the bead slicing: overwrites the slow forces F_s with NaN, then evaluates them in n_slices bead
 * slices, one launch after the other (the launches ranks 0..n_slices-1 would make); F_s, hence qhp_forces, must
 * afterwards equal the unsliced result bit for bit.  n_slices must divide P_contract. */
int qhp_pair_slices(qhp_system *sys, int n_slices);

/* Bead-space forces at the current positions, device [P][n_atoms][3]:
 * G_i = -grad V_f(x_i) + (P/P') sum_j C_ji (-grad V_s(xc_j))  (Eq. 10-11 and chain rule on Eq. 20). */
int qhp_forces(qhp_system *sys, double *f_beads);

/* out[0] = K_CV centroid-virial kinetic energy, out[1] = U = (1/P) sum V_f + (1/P') sum V_s
 * (Eq. 6, Eq. 20), out[2] = K_nm = sum Pm^2/2m, out[3] = T_inst = 2 K_nm/(3 N P kB);
 * kcal/mol, K.  n_out <= 4 values are written. */
int qhp_observables(qhp_system *sys, double *out, int n_out);
int qhp_observables_host(qhp_system *sys, double *out, int n_out);

/* ---- parity hooks (device pointers) ---------------------------------------------------- */
/* Canonical neighbour objects of the CURRENT centroids (rebuilds them): cell_of[n_atoms],
 * order[n_atoms] (atoms stably sorted by cell), cell_start[ncell+1], n_cells3[3].
 * Any pointer may be NULL. */
int qhp_neighbor_lists(qhp_system *sys, int32_t *cell_of, int32_t *order, int32_t *cell_start,
                       int32_t *n_cells3);
/* Pair list of the current centroids in ATOM indices: count[n_atoms] and, if nbr != NULL,
 * nbr[start(i) .. start(i)+count[i]) with start = exclusive prefix sum of count; entries are
 * all j != i of another molecule with centroid distance^2 < r_list^2 (order unspecified).
 * total_host (HOST pointer, may be NULL) receives sum(count) (synchronises). */
int qhp_pair_list(qhp_system *sys, int32_t *count, int32_t *nbr, int64_t cap, int64_t *total_host);
/* Contracted bead positions xc [P_contract][n_atoms][3] (Eq. 20) of the current state. */
int qhp_contracted(qhp_system *sys, double *xc);
/* adQTB: gamma_z(omega_j) [n_types][n_seg+1]; coloured force segment Fc and recorded
 * velocities vseg, both [3 n_atoms][n_seg] (NULL to skip). */
int qhp_adqtb_gamma(qhp_system *sys, double *gamma);
/* adQTB restart: load gamma_z(omega_j) [n_types][n_seg+1] (DEVICE pointer, values > 0) as written by qhp_adqtb_gamma
 * of an earlier run, so that create -> qhp_adqtb_set_gamma -> qhp_set_state(x, p, step0) at a segment boundary
 * continues an adapted run (the adaptation takes ps to 100s of ps) instead of restarting from gamma_0.
 * Allowed before qhp_set_state, or at a segment boundary before the first step of the segment (QHP_ESTATE
 * otherwise: the segment's coloured force has been generated with the old gamma).  Not restored: the RATIO
 * window averages (Eq. 26; the first segment after a restart re-initialises them) -- kappa is an input the caller
 * sets again. */
int qhp_adqtb_set_gamma(qhp_system *sys, const double *gamma);
/* adQTB: RATIO adaptation (Eq. 24-26) for the atom types with tau_ps[z] > 0:
 * gamma_z = Re<C_vF,z> / (m_z <C_vv,z>) from exponential-window averages of the segment spectra with
 * time constant tau_ps[z] (the first segment after this call initialises them); the other types keep
 * the SIMPLE rule (Eq. 23, thermostat a_gamma).  tau_ps: HOST pointer [n_types], or NULL for SIMPLE on
 * every type.  Synchronises. */
int qhp_adqtb_ratio(qhp_system *sys, const double *tau_ps);
/* adQTB: kernel-correction hook (PAPER.md:203 cites corrections of the QTB kernel "for finite timestep"
 * and "non-zero friction" without defining them; SURVEY reading G11): the filter of Eq. 13-14 becomes
 * H_z(omega_j) = kappa[j] sqrt(2 m_z gamma_z(omega_j) Theta(omega_j) / dt), omega_j = pi j / (n_seg dt),
 * j = 0..n_seg, the same factor for every type (an AMPLITUDE factor: the noise PSD gets kappa^2).  It
 * takes effect from the next noise generation (the next segment boundary, or the first step after
 * qhp_set_state).  kappa: HOST pointer [n_seg+1], finite and >= 0 (else QHP_EINVAL); NULL restores the
 * identity.  The caller keeps the buffer; the values are copied.  Synchronises. */
int qhp_adqtb_kappa(qhp_system *sys, const double *kappa);
int qhp_adqtb_segment(qhp_system *sys, double *Fc, double *vseg);
/* Counters for measurement: out_host[0] = neighbour-list rebuilds so far, [1] = list entries,
 * [2] = pair-bead interactions inside r_cut at the current positions (full list, both
 * directions), [3] = list capacity, [4] = kernels launched so far, [5] = error flags (bit 0 list
 * overflow, bit 1 skin < 2 x bead spread, bit 2 staged neighbourhood outgrew shared memory),
 * [6] = 1 if the shared-memory staged pair kernel serves this system (0: generic kernel),
 * [7] = warps per CTA of the staged kernel.  n_out <= 8.  HOST pointer; synchronises. */
int qhp_counters(qhp_system *sys, int64_t *out_host, int n_out);
/* Per-phase device timing with CUDA events recorded on the library stream inside qhp_step:
 * qhp_profile(sys, 1) starts recording (and clears the sums), qhp_profile(sys, 0) stops.
 * qhp_profile_read synchronises and writes ms_host[0..4] = summed milliseconds of
 * {integrator pass, neighbour rebuild chain, pair forces, adQTB segment generation (Q2-Q4),
 * adQTB spectra + adaptation (Q5-Q7)} and n_host[0..4] = number of timed intervals of each.
 * HOST pointers. */
int qhp_profile(qhp_system *sys, int enable);
int qhp_profile_read(qhp_system *sys, double *ms_host, int64_t *n_host);
/* The pair-force phase launch by launch, from the same recording: ms_host[0..2], n_host[0..2] = {k_prune_check,
 * k_prune, k_pair_dense} (all 0 when the pruned-row path does not serve the system).  HOST pointers; synchronises. */
int qhp_profile_read_pair(qhp_system *sys, double *ms_host, int64_t *n_host);
/* Synchronise the stream and report sticky CUDA / overflow errors. */
int qhp_check(qhp_system *sys);
const char *qhp_last_error(const qhp_system *sys); /* sys may be NULL: last error of a call without a handle
                                                     * (qhp_create, qhp_pibar_noalloc) */

/* ---- stand-alone primitives of the path (device pointers), for parity tests ------------- */
/* Philox4x32-10 words and the three Box-Muller normals of counter (atom0+i, mode | tag<<24,
 * step) for i < n: words [n][4] uint32 (may be NULL), z [n][3] (may be NULL). */
int qhp_philox_normals(uint64_t seed, uint32_t atom0, uint32_t mode, uint32_t tag, uint64_t step,
                       int64_t n, uint32_t *words, double *z, void *cuda_stream);
/* Batched complex fp64 FFT of length n (power of two, 8..8192) by the shared-memory Stockham
 * kernel used for the QTB noise and spectra: data [batch][n][2], in place; sign = -1 forward,
 * +1 inverse (unnormalised). */
int qhp_fft_c2c(double *data, int n, int64_t batch, int sign, void *cuda_stream);
/* DFMA throughput probe: runs iters fused multiply-adds per thread on grid x block threads and
 * writes one double per thread to sink (device, grid*block doubles). */
int qhp_dfma_probe(double *sink, int grid, int block, int64_t iters, void *cuda_stream);

/* ---- post-processing of stored potential-energy series ---------------------------------- */
/* PI-BAR free-energy difference dF_AB = (1/beta) ln(Z_A/Z_B) (Eq. 27-28):
 *   dF = C + (1/beta) ln( <f(U_A - U_B + C)>_B / <f(U_B - U_A - C)>_A ),  C = dF + (1/beta) ln(n_B/n_A),
 *   f(x) = 1/(1 + exp(beta x)), iterated from dF = 0 until |change| <= tol or max_iter iterations (G26).
 * wA (device, n_A doubles) = U_B - U_A on the configurations sampled in state A, wB (device, n_B) =
 * U_A - U_B on those sampled in state B, U the bead-averaged potential of Eq. 3 (qhp_observables out[1]);
 * with a single bead's V it is the estimator of Appendix A, with P = 1 classical BAR.  beta in mol/kcal.
 * Runs on cuda_stream and synchronises it; dF_host (kcal/mol) and iters_host (may be NULL) are host
 * pointers.  The inputs are not modified.  QHP_EINVAL for empty series or beta <= 0. */
int qhp_pibar(const double *wA, int64_t n_A, const double *wB, int64_t n_B, double beta, int max_iter,
              double tol, void *cuda_stream, double *dF_host, int *iters_host);

/* The same estimator for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc).  qhp_pibar allocates and frees its per-CTA partial sums on
 * every call and copies the result to the host; this entry point calls no cudaMalloc, cudaFree, memcpy or
 * allocating library routine and does NOT synchronise: it enqueues one cooperative kernel on cuda_stream.
 *   scratch   the per-CTA partial sums live in a file-scope static __device__ array of the library
 *             (QHP_PIBAR_NOALLOC_SCRATCH_BYTES = 16 KiB, held by every GPU that loads the library until
 *             exit): room for QHP_PIBAR_NOALLOC_MAX_CTAS CTAs.
 *   limit     n_A, n_B <= QHP_PIBAR_NOALLOC_MAX_N (= MAX_CTAS CTAs x 256 threads x 64 samples per thread and
 *             iteration); longer series, or a device whose grid would need more CTAs than the array holds,
 *             are rejected with QHP_EINVAL and a text in qhp_last_error(NULL).  Use qhp_pibar for those.
 *   out_dev   DEVICE pointer, 2 doubles, caller-owned: out_dev[0] = dF (kcal/mol), out_dev[1] = number of
 *             iterations; valid once the work enqueued on cuda_stream has finished.
 *   sharing   every call on a device uses the same array and finds the previous call's partial sums in it.
 *             Nothing has to start at zero: each iteration writes all of its partial sums before the grid
 *             barrier that precedes their reads.  Calls that overlap on the GPU (two streams, two host
 *             threads, two graphs in flight) RACE on the array: serialise them (one stream, or events).
 *   set-up    the first call on each device resolves the array's device address (cudaGetSymbolAddress with
 *             that device current) and the launch geometry; make that first call outside stream capture.
 * Same arguments, arithmetic, grid and summation order as qhp_pibar otherwise: the two agree bit for bit. */
#define QHP_PIBAR_NOALLOC_MAX_CTAS 512
#define QHP_PIBAR_NOALLOC_SCRATCH_BYTES (4 * QHP_PIBAR_NOALLOC_MAX_CTAS * 8)
#define QHP_PIBAR_NOALLOC_MAX_N (QHP_PIBAR_NOALLOC_MAX_CTAS * 256 * 64)
int qhp_pibar_noalloc(const double *wA, int64_t n_A, const double *wB, int64_t n_B, double beta, int max_iter,
                      double tol, void *cuda_stream, double *out_dev);

#ifdef __cplusplus
}
#endif
#endif /* QHP_H */
