"""CPU oracle for the Quantum-HP hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It wraps `oracle/qhp_oracle.c` (plain C, fp64, single thread)
with ctypes and adds numpy pieces whose only library primitive is `numpy.fft` (used as "the
DFT", validated against the direct sums of the C file in tests/test_oracle_adqtb.py).

It never imports `paper_2212_03137_b200` and shares no code with it.
Citations: "PAPER.md:<line>" = /root/reference/PAPER.md; O1..O11 / G1..G23 = SURVEY.md §8(c),
restated in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qhp_oracle.c")
_LIB = os.path.join(_HERE, "libqhp_oracle.so")

KB = 1.987204258640832e-3
HBAR = 1.5178728306651436e-2
ACC = 418.4


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc -O2, no implicit FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Top(C.Structure):
    _fields_ = [("n_atoms", C.c_int32), ("n_types", C.c_int32), ("n_bonds", C.c_int32),
                ("n_angles", C.c_int32),
                ("type", C.c_void_p), ("mol", C.c_void_p),
                ("mass", C.c_void_p), ("charge", C.c_void_p), ("lj_eps", C.c_void_p),
                ("lj_sigma", C.c_void_p), ("tether_k", C.c_void_p),
                ("bond_idx", C.c_void_p), ("bond_k", C.c_void_p), ("bond_r0", C.c_void_p),
                ("angle_idx", C.c_void_p), ("angle_k", C.c_void_p), ("angle_th0", C.c_void_p),
                ("box", C.c_double * 3),
                ("r_cut", C.c_double), ("dsf_alpha", C.c_double), ("skin", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.qo_theta.restype = C.c_double
        _lib.qo_theta.argtypes = [C.c_double, C.c_double]
        for name in ("qo_force_fast", "qo_force_slow_brute", "qo_force_slow_cells"):
            getattr(_lib, name).restype = C.c_double
        _lib.qo_force_total.restype = C.c_double
        _lib.qo_pairs_brute.restype = C.c_int64
        _lib.qo_neighbours_of.restype = C.c_int32
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Topology:
    """Keeps the numpy arrays alive and exposes the C struct."""

    def __init__(self, top: dict):
        self.n_atoms = int(top["n_atoms"])
        self.n_types = int(top["n_types"])
        self._keep = {}
        t = _Top()
        t.n_atoms, t.n_types = self.n_atoms, self.n_types
        t.n_bonds, t.n_angles = int(top["n_bonds"]), int(top["n_angles"])
        for k in ("type", "mol", "bond_idx", "angle_idx"):
            self._keep[k] = np.ascontiguousarray(top[k], dtype=np.int32)
            setattr(t, k, _p(self._keep[k]))
        for k in ("mass", "charge", "lj_eps", "lj_sigma", "bond_k", "bond_r0", "angle_k", "angle_th0"):
            self._keep[k] = _f64(top[k])
            setattr(t, k, _p(self._keep[k]))
        if top.get("tether_k") is not None:
            self._keep["tether_k"] = _f64(top["tether_k"])
            t.tether_k = _p(self._keep["tether_k"])
        else:
            t.tether_k = None
        for d in range(3):
            t.box[d] = float(top["box"][d])
        t.r_cut, t.dsf_alpha, t.skin = float(top["r_cut"]), float(top["dsf_alpha"]), float(top["skin"])
        self.c = t
        self.type = self._keep["type"]
        self.mol = self._keep["mol"]
        self.mass = self._keep["mass"]
        self.box = np.array([t.box[0], t.box[1], t.box[2]])
        self.r_cut, self.skin = t.r_cut, t.skin

    @property
    def ref(self):
        return C.byref(self.c)

    @property
    def use_cells(self) -> int:
        return int(self.n_atoms > 3000)


# ---------------------------------------------------------------- Philox / normals (O6)
def philox4x32_10(ctr, key) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().qo_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def normals3(seed: int, atom: int, mode: int, tag: int, step: int) -> np.ndarray:
    z = np.empty(3)
    lib().qo_normals3(C.c_uint64(seed), C.c_uint32(atom), C.c_uint32(mode), C.c_uint32(tag),
                      C.c_uint64(step), _p(z))
    return z


# ---------------------------------------------------------------- normal modes (O1, O2)
def nm_matrix(P: int) -> np.ndarray:
    T = np.empty((P, P))
    lib().qo_nm_matrix(C.c_int(P), _p(T))
    return T


def nm_freq(P: int, T_K: float) -> np.ndarray:
    w = np.empty(P)
    lib().qo_nm_freq(C.c_int(P), C.c_double(T_K), _p(w))
    return w


def beads_to_nm(x: np.ndarray) -> np.ndarray:
    """x [P][...] -> Q [P][...]  (Q_n = (1/sqrt P) sum_i T[i][n] x_i)."""
    x = _f64(x)
    P = x.shape[0]
    Q = np.empty_like(x)
    lib().qo_beads_to_nm(C.c_int(P), C.c_int64(x[0].size), _p(x), _p(Q))
    return Q


def nm_to_beads(Q: np.ndarray) -> np.ndarray:
    Q = _f64(Q)
    P = Q.shape[0]
    x = np.empty_like(Q)
    lib().qo_nm_to_beads(C.c_int(P), C.c_int64(Q[0].size), _p(Q), _p(x))
    return x


def contract(Q: np.ndarray, Pc: int) -> np.ndarray:
    """Eq. 20: contracted beads [Pc][...] from the NM amplitudes Q [P][...]."""
    Q = _f64(Q)
    xc = np.empty((Pc,) + Q.shape[1:])
    lib().qo_contract(C.c_int(Q.shape[0]), C.c_int(Pc), C.c_int64(Q[0].size), _p(Q), _p(xc))
    return xc


def expand_force(Fc: np.ndarray, P: int) -> np.ndarray:
    Fc = _f64(Fc)
    fs = np.empty((P,) + Fc.shape[1:])
    lib().qo_expand_force(C.c_int(P), C.c_int(Fc.shape[0]), C.c_int64(Fc[0].size), _p(Fc), _p(fs))
    return fs


def contraction_matrix(P: int, Pc: int) -> np.ndarray:
    """C = (sqrt Pc / sqrt P) T^(Pc) [I 0] T^(P)^T obtained by contracting unit bead vectors."""
    C_ = np.empty((Pc, P))
    for i in range(P):
        e = np.zeros((P, 1))
        e[i, 0] = 1.0
        C_[:, i] = contract(beads_to_nm(e), Pc)[:, 0]
    return C_


# ---------------------------------------------------------------- forces (O3, O7)
def force_fast(top: Topology, x: np.ndarray):
    x = _f64(x)
    F = np.zeros_like(x)
    u = lib().qo_force_fast(top.ref, _p(x), _p(F))
    return u, F


def force_slow(top: Topology, x: np.ndarray, cells: bool = False):
    x = _f64(x)
    F = np.zeros_like(x)
    fn = lib().qo_force_slow_cells if cells else lib().qo_force_slow_brute
    u = fn(top.ref, _p(x), _p(F))
    return u, F


def force_total(top: Topology, x: np.ndarray, cells: bool | None = None):
    x = _f64(x)
    F = np.zeros_like(x)
    uc = top.use_cells if cells is None else int(cells)
    u = lib().qo_force_total(top.ref, _p(x), _p(F), C.c_int(uc))
    return u, F


def nm_forces(top: Topology, P: int, Pc: int, Q: np.ndarray, cells: bool | None = None):
    """NM forces f_n(Q) [P][N][3] and (U_f, U_s)."""
    Q = _f64(Q)
    f = np.empty_like(Q)
    e = np.empty(2)
    uc = top.use_cells if cells is None else int(cells)
    lib().qo_nm_forces(top.ref, C.c_int(P), C.c_int(Pc), _p(Q), _p(f), _p(e), C.c_int(uc))
    return f, e


def bead_forces(top: Topology, P: int, Pc: int, x_beads: np.ndarray, cells: bool | None = None):
    """O7: G_i = F^f_i + (P/Pc) sum_j C[j][i] Fc_j, [P][N][3]."""
    x = _f64(x_beads)
    G = np.empty_like(x)
    uc = top.use_cells if cells is None else int(cells)
    lib().qo_bead_forces(top.ref, C.c_int(P), C.c_int(Pc), _p(x), _p(G), C.c_int(uc))
    return G


def observables(top: Topology, P: int, Pc: int, T_K: float, Q, Pm, cells: bool | None = None):
    Q, Pm = _f64(Q), _f64(Pm)
    out = np.empty(4)
    uc = top.use_cells if cells is None else int(cells)
    lib().qo_observables(top.ref, C.c_int(P), C.c_int(Pc), C.c_double(T_K), _p(Q), _p(Pm), _p(out),
                         C.c_int(uc))
    return out


# ---------------------------------------------------------------- neighbour objects (O4)
def cells(top: Topology, centroids: np.ndarray):
    c = _f64(centroids)
    nc = np.zeros(3, np.int32)
    N = top.n_atoms
    rl = top.r_cut + top.skin
    ncell = int(np.prod(np.maximum(1, np.floor(top.box / rl)).astype(int)))
    cell_of = np.empty(N, np.int32)
    order = np.empty(N, np.int32)
    cell_start = np.empty(ncell + 1, np.int32)
    lib().qo_cells(top.ref, _p(c), _p(nc), _p(cell_of), _p(order), _p(cell_start))
    return nc, cell_of, order, cell_start


def pairs_brute(top: Topology, centroids: np.ndarray) -> np.ndarray:
    c = _f64(centroids)
    n = lib().qo_pairs_brute(top.ref, _p(c), None, C.c_int64(0))
    pairs = np.empty((n, 2), np.int32)
    lib().qo_pairs_brute(top.ref, _p(c), _p(pairs), C.c_int64(n))
    return pairs


def neighbours_of(top: Topology, centroids: np.ndarray, i: int) -> np.ndarray:
    c = _f64(centroids)
    nb = np.empty(4096, np.int32)
    n = lib().qo_neighbours_of(top.ref, _p(c), C.c_int32(i), _p(nb), C.c_int32(nb.size))
    assert n <= nb.size
    return nb[:n].copy()


# ---------------------------------------------------------------- RPMD driver (O5)
class Rpmd:
    """State in normal modes; `step(n)` = n x B A O A B (Eq. 16-17)."""

    def __init__(self, top: Topology, P: int, Pc: int, dt_ps: float, T_K: float, thermo: str,
                 gamma0: float, seed: int, cells: bool | None = None, a_block: str = "exact"):
        self.top, self.P, self.Pc, self.dt, self.T = top, P, Pc, dt_ps, T_K
        self.a_block = {"exact": 0, "cayley": 1}[a_block]       # "cayley": BCOCB
        self.thermo = {"none": 0, "pile": 1}[thermo]
        self.gamma0, self.seed = gamma0, seed
        self.uc = top.use_cells if cells is None else int(cells)
        self.step_index = 0

    def set_state(self, x_beads, p_beads, step0: int = 0):
        self.Q = beads_to_nm(x_beads)
        self.Pm = beads_to_nm(p_beads)
        self.f, _ = nm_forces(self.top, self.P, self.Pc, self.Q, self.uc)
        self.step_index = step0

    def step(self, n: int):
        fn = lib().qo_rpmd_steps_bcocb if self.a_block else lib().qo_rpmd_steps
        fn(self.top.ref, C.c_int(self.P), C.c_int(self.Pc), C.c_double(self.dt),
           C.c_double(self.T), C.c_int(self.thermo), C.c_double(self.gamma0),
           C.c_uint64(self.seed), C.c_int64(self.step_index), C.c_int64(n),
           _p(self.Q), _p(self.Pm), _p(self.f), C.c_int(self.uc))
        self.step_index += n

    def get_state(self):
        return nm_to_beads(self.Q), nm_to_beads(self.Pm)

    def forces(self):
        return nm_to_beads(self.f)          # G_i = sqrt(P) sum_n T[i][n] f_n  (O7)

    def observables(self):
        return observables(self.top, self.P, self.Pc, self.T, self.Q, self.Pm, self.uc)


def set_contraction_variant(v: int):
    """0 = literal Eq. 20 (default); 1 = trigonometric interpolation (sqrt 2 on the Nyquist mode of an even P').
    Process-wide switch of the oracle: reset it to 0 after use."""
    lib().qo_set_contraction_variant(C.c_int(int(v)))


def nm_forces_split(top: Topology, P: int, Pc: int, Q: np.ndarray, cells: bool | None = None):
    """Normal-mode forces of V_f and V_s separately (Eq. 18; used by the RESPA stepper)."""
    Q = _f64(Q)
    ff, fs = np.empty_like(Q), np.empty_like(Q)
    uc = top.use_cells if cells is None else int(cells)
    lib().qo_nm_forces_split(top.ref, C.c_int(P), C.c_int(Pc), _p(Q), _p(ff), _p(fs), C.c_int(uc))
    return ff, fs


class RpmdRespa(Rpmd):
    """BAOAB-RESPA (Eq. 19): `step(n)` advances n INNER steps of dt, n a multiple of
    n_alt; V_s (on the Pc contracted beads) kicks with n_alt*dt/2 around every n_alt inner steps."""

    def __init__(self, top, P, Pc, dt_ps, T_K, thermo, gamma0, seed, n_alt: int, cells=None, a_block="exact"):
        super().__init__(top, P, Pc, dt_ps, T_K, thermo, gamma0, seed, cells, a_block)
        self.n_alt = int(n_alt)

    def set_state(self, x_beads, p_beads, step0: int = 0):
        self.Q = beads_to_nm(x_beads)
        self.Pm = beads_to_nm(p_beads)
        self.ff, self.fs = nm_forces_split(self.top, self.P, self.Pc, self.Q, self.uc)
        self.step_index = step0

    @property
    def f(self):
        return self.ff + self.fs

    def step(self, n: int):
        assert n % self.n_alt == 0
        fn = lib().qo_rpmd_respa_steps_bcocb if self.a_block else lib().qo_rpmd_respa_steps
        fn(self.top.ref, C.c_int(self.P), C.c_int(self.Pc), C.c_double(self.dt),
           C.c_double(self.T), C.c_int(self.thermo), C.c_double(self.gamma0),
           C.c_uint64(self.seed), C.c_int64(self.step_index), C.c_int64(n // self.n_alt),
           C.c_int(self.n_alt), _p(self.Q), _p(self.Pm), _p(self.ff), _p(self.fs),
           C.c_int(self.uc))
        self.step_index += n


# ---------------------------------------------------------------- adQTB (O9-O11)
def theta(omega, T_K: float):
    return np.vectorize(lambda w: lib().qo_theta(float(w), float(T_K)))(omega)


def qtb_filter(n_seg: int, dt: float, T_K: float, mass_amu: float, gamma_z: np.ndarray,
               classical: bool = False, kappa=None) -> np.ndarray:
    """kappa: optional amplitude factor kappa(omega_j), j = 0..n_seg, on H (reading G11)."""
    g = _f64(gamma_z)
    H = np.empty(n_seg + 1)
    if kappa is None:
        lib().qo_qtb_filter(C.c_int(n_seg), C.c_double(dt), C.c_double(T_K), C.c_double(mass_amu),
                            _p(g), C.c_int(int(classical)), _p(H))
    else:
        k = _f64(kappa)
        assert k.shape == (n_seg + 1,)
        lib().qo_qtb_filter_kappa(C.c_int(n_seg), C.c_double(dt), C.c_double(T_K), C.c_double(mass_amu),
                                  _p(g), C.c_int(int(classical)), _p(k), _p(H))
    return H


def qtb_kernel(H: np.ndarray) -> np.ndarray:
    """h[k + n_seg], k = -n_seg..n_seg-1 (direct inverse DFT of the evenly extended H)."""
    H = _f64(H)
    n_seg = H.size - 1
    h = np.empty(2 * n_seg)
    lib().qo_qtb_kernel(C.c_int(n_seg), _p(H), _p(h))
    return h


def qtb_white(seed: int, atom: int, s0: int, count: int) -> np.ndarray:
    r = np.empty((3, count))
    lib().qo_qtb_white(C.c_uint64(seed), C.c_int32(atom), C.c_int64(s0), C.c_int32(count), _p(r))
    return r


def qtb_colored_direct(top: Topology, n_seg: int, seed: int, seg: int, h_types: np.ndarray):
    h = _f64(h_types)
    Fc = np.empty((3 * top.n_atoms, n_seg))
    lib().qo_qtb_colored_direct(top.ref, C.c_int(n_seg), C.c_uint64(seed), C.c_int64(seg), _p(h), _p(Fc))
    return Fc


def qtb_colored_fft(top: Topology, n_seg: int, seed: int, seg: int, h_types: np.ndarray, atoms=None):
    """Same definition as `qtb_colored_direct`, the sum evaluated with numpy.fft as the DFT
    (linear convolution through zero-padding to 4 n_seg).  Validated against the direct sum.
    `atoms` (optional): only these atoms, rows returned in that order ([3 len(atoms)][n_seg]) --
    lets the tests sample boxes too large to do in full."""
    nfft = 4 * n_seg
    atom_list = range(top.n_atoms) if atoms is None else [int(a) for a in atoms]
    Fc = np.empty((3 * len(atom_list), n_seg))
    hk = []
    for z in range(top.n_types):
        buf = np.zeros(nfft)
        buf[:2 * n_seg] = h_types[z]          # buf[m] = h[m - n_seg]
        hk.append(np.fft.rfft(buf))
    for row, a in enumerate(atom_list):
        r = qtb_white(seed, a, seg * n_seg, 3 * n_seg)
        y = np.fft.irfft(np.fft.rfft(r, n=nfft, axis=1) * hk[top.type[a]][None, :], n=nfft, axis=1)
        # y[m] = sum_k h[k] r[m - n_seg - k]  =>  F_c[n] = y[n + 2 n_seg]
        Fc[3 * row:3 * row + 3] = y[:, 2 * n_seg:3 * n_seg]
    return Fc


def qtb_spectra_direct(top: Topology, n_seg: int, dt: float, vseg, Fc):
    vseg, Fc = _f64(vseg), _f64(Fc)
    Cvv = np.empty((top.n_types, n_seg + 1))
    CvF = np.empty((top.n_types, n_seg + 1))
    lib().qo_qtb_spectra_direct(top.ref, C.c_int(n_seg), C.c_double(dt), _p(vseg), _p(Fc), _p(Cvv), _p(CvF))
    return Cvv, CvF


def qtb_spectra_fft(top: Topology, n_seg: int, dt: float, vseg, Fc):
    """Eq. 22 with numpy.fft.rfft (zero-padded to N_k = 2 n_seg) as the DFT."""
    V = np.fft.rfft(vseg, n=2 * n_seg, axis=1)
    Ph = np.fft.rfft(Fc, n=2 * n_seg, axis=1)
    cvv = dt / n_seg * np.abs(V) ** 2
    cvf = dt / n_seg * (V * np.conj(Ph)).real
    tdof = np.repeat(top.type, 3)
    Cvv = np.stack([cvv[tdof == z].mean(axis=0) for z in range(top.n_types)])
    CvF = np.stack([cvf[tdof == z].mean(axis=0) for z in range(top.n_types)])
    return Cvv, CvF


def qtb_adapt(top: Topology, n_seg: int, gamma0: float, a_gamma: float, gmin_frac: float,
              Cvv, CvF, gamma):
    g = _f64(gamma).copy()
    Cvv, CvF = _f64(Cvv), _f64(CvF)
    lib().qo_qtb_adapt(C.c_int(top.n_types), C.c_int(n_seg), _p(top.mass), C.c_double(gamma0),
                       C.c_double(a_gamma), C.c_double(gmin_frac), _p(Cvv), _p(CvF), _p(g))
    return g


def qtb_adapt_ratio(top: Topology, n_seg: int, gamma0: float, gmin_frac: float, dt: float, tau, first: bool,
                    Cvv, CvF, avv, avf, gamma):
    """RATIO adaptation (Eq. 24-26) of the types with tau[z] > 0; returns (gamma, avv, avf) copies."""
    g, av, af = _f64(gamma).copy(), _f64(avv).copy(), _f64(avf).copy()
    Cvv, CvF, tau = _f64(Cvv), _f64(CvF), _f64(tau)
    lib().qo_qtb_adapt_ratio(C.c_int(top.n_types), C.c_int(n_seg), _p(top.mass), C.c_double(gamma0),
                             C.c_double(gmin_frac), C.c_double(dt), _p(tau), C.c_int(int(first)), _p(Cvv), _p(CvF),
                             _p(av), _p(af), _p(g))
    return g, av, af


class Adqtb:
    """adQTB driver: segments of n_seg steps, noise generated at segment start
    (l.203-209), spectra + SIMPLE adaptation at segment end (l.213-232, 248)."""

    def __init__(self, top: Topology, dt_ps: float, T_K: float, gamma0: float, seed: int,
                 n_seg: int, a_gamma: float, gmin_frac: float = 0.01, classical: bool = False,
                 direct: bool = False, cells: bool | None = None, ratio_tau=None):
        self.top, self.dt, self.T, self.gamma0, self.seed = top, dt_ps, T_K, gamma0, seed
        self.n_seg, self.a_gamma, self.gmin_frac = n_seg, a_gamma, gmin_frac
        self.classical, self.direct = classical, direct
        self.uc = top.use_cells if cells is None else int(cells)
        self.gamma = np.full((top.n_types, n_seg + 1), gamma0)
        self.step_index = 0
        self.Fc = None
        self.vseg = np.zeros((3 * top.n_atoms, n_seg))
        self.history = []           # (Cvv, CvF, gamma_after) per finished segment
        # RATIO adaptation (Eq. 24-26) for the types with ratio_tau[z] > 0 ps, SIMPLE (Eq. 23) for the others
        self.ratio_tau = None if ratio_tau is None else np.asarray(ratio_tau, float)
        self.avv = np.zeros((top.n_types, n_seg + 1))
        self.avf = np.zeros((top.n_types, n_seg + 1))
        self.ratio_started = False
        self.kappa = None           # kernel-correction factor kappa(omega_j) [n_seg + 1] (reading G11), None = 1

    def set_state(self, x, p, step0: int = 0):
        assert step0 % self.n_seg == 0
        self.x = _f64(x).reshape(-1).copy()
        self.p = _f64(p).reshape(-1).copy()
        self.F = np.empty_like(self.x)
        lib().qo_force_total(self.top.ref, _p(self.x), _p(self.F), C.c_int(self.uc))
        self.step_index = step0
        self.Fc = None

    def kernels(self):
        return np.stack([qtb_kernel(qtb_filter(self.n_seg, self.dt, self.T, self.top.mass[z],
                                               self.gamma[z], self.classical, self.kappa))
                         for z in range(self.top.n_types)])

    def _new_segment(self):
        seg = self.step_index // self.n_seg
        fn = qtb_colored_direct if self.direct else qtb_colored_fft
        self.Fc = fn(self.top, self.n_seg, self.seed, seg, self.kernels())

    def step(self, n: int):
        while n > 0:
            n0 = self.step_index % self.n_seg
            if n0 == 0 and (self.Fc is None or self._seg_of_Fc != self.step_index // self.n_seg):
                self._new_segment()
                self._seg_of_Fc = self.step_index // self.n_seg
            m = min(n, self.n_seg - n0)
            lib().qo_adqtb_steps(self.top.ref, C.c_double(self.dt), C.c_double(self.gamma0),
                                 C.c_int(self.n_seg), C.c_int(n0), C.c_int(m), _p(self.x), _p(self.p),
                                 _p(self.F), _p(self.Fc), _p(self.vseg), C.c_int(self.uc))
            self.step_index += m
            n -= m
            if self.step_index % self.n_seg == 0:
                fn = qtb_spectra_direct if self.direct else qtb_spectra_fft
                Cvv, CvF = fn(self.top, self.n_seg, self.dt, self.vseg, self.Fc)
                g_simple = qtb_adapt(self.top, self.n_seg, self.gamma0, self.a_gamma,
                                     self.gmin_frac, Cvv, CvF, self.gamma)
                if self.ratio_tau is not None and (self.ratio_tau > 0).any():
                    g_ratio, self.avv, self.avf = qtb_adapt_ratio(
                        self.top, self.n_seg, self.gamma0, self.gmin_frac, self.dt, self.ratio_tau,
                        not self.ratio_started, Cvv, CvF, self.avv, self.avf, self.gamma)
                    self.ratio_started = True
                    for z in range(self.top.n_types):
                        if self.ratio_tau[z] > 0:
                            g_simple[z] = g_ratio[z]
                self.gamma = g_simple
                self.history.append((Cvv, CvF, self.gamma.copy()))

    def get_state(self):
        N = self.top.n_atoms
        return self.x.reshape(1, N, 3).copy(), self.p.reshape(1, N, 3).copy()


# ---------------------------------------------------------------- PI-BAR (NEXT-5, Eq. 27-28)
def pibar(wA, wB, beta: float, max_iter: int = 1000, tol: float = 1e-13):
    """dF_AB = (1/beta) ln(Z_A/Z_B) from wA = U_B - U_A on samples of A and wB = U_A - U_B on samples of B
    (Eq. 27-28, solved by fixed-point iteration).  Returns (dF, iterations)."""
    wA, wB = _f64(wA), _f64(wB)
    out = C.c_double(0.0)
    fn = lib().qo_pibar
    fn.restype = C.c_int
    it = fn(_p(wA), C.c_int64(wA.size), _p(wB), C.c_int64(wB.size), C.c_double(beta), C.c_int(max_iter),
            C.c_double(tol), C.byref(out))
    return out.value, it
