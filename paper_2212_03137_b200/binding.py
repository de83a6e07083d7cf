"""ctypes binding of include/qhp.h.  Marshals torch CUDA tensors / numpy topology arrays into the
C ABI; holds no arithmetic of the method.  Fails loudly if libqhp.so is missing."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("QHP_LIB") or os.path.join(_HERE, "libqhp.so")   # QHP_LIB: another build of the same library

QHP_THERMO_NONE, QHP_THERMO_PILE, QHP_THERMO_ADQTB = 0, 1, 2
_STATUS = {0: "QHP_OK", -1: "QHP_EINVAL", -2: "QHP_ENOMEM", -3: "QHP_ECUDA", -4: "QHP_ESTATE"}

# every symbol include/qhp.h declares (tests check that the library exports them all)
SYMBOLS = ["qhp_create", "qhp_destroy", "qhp_set_respa", "qhp_set_a_block", "qhp_set_contraction", "qhp_set_state", "qhp_get_state", "qhp_set_state_host",
           "qhp_get_state_host", "qhp_step", "qhp_forces", "qhp_observables", "qhp_observables_host",
           "qhp_neighbor_lists", "qhp_pair_list", "qhp_contracted", "qhp_adqtb_gamma", "qhp_adqtb_ratio", "qhp_adqtb_kappa",
           "qhp_adqtb_segment", "qhp_counters", "qhp_profile", "qhp_profile_read", "qhp_check", "qhp_last_error", "qhp_philox_normals",
           "qhp_fft_c2c", "qhp_dfma_probe", "qhp_pibar", "qhp_pibar_noalloc", "qhp_set_comm", "qhp_pair_slices", "qhp_set_pair_prune", "qhp_pair_prune_stats", "qhp_profile_read_pair", "qhp_adqtb_set_gamma"]


# int fn(void *ctx, void *device_buf, size_t bytes_per_rank, int rank, int world, void *cuda_stream)  (include/qhp.h)
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_int, C.c_int, C.c_void_p)


def allgather_inplace(buf, rank: int, world: int, group=None):
    """In-place all-gather of a flat tensor of `world` equal blocks (block `rank` valid on entry) over
    torch.distributed: NCCL for CUDA tensors (the data-path collective of the bead-sharded V_s), gloo for the
    host-side tests.  Argument marshalling only."""
    import torch.distributed as dist
    n = buf.numel() // world
    dist.all_gather_into_tensor(buf, buf[rank * n:(rank + 1) * n].clone(), group=group)
    return buf


class _DevMem:
    """A raw device allocation of the library seen through __cuda_array_interface__ (no copy)."""

    def __init__(self, ptr: int, n: int):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False), "version": 2}


def _wrap_device_f64(ptr: int, n: int):
    return _torch().as_tensor(_DevMem(ptr, n), device="cuda")


class QhpError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_STATUS.get(code, code)}: {text}")
        self.code = code


class _Topology(C.Structure):
    _fields_ = [("n_atoms", C.c_int32), ("n_types", C.c_int32), ("n_bonds", C.c_int32), ("n_angles", C.c_int32),
                ("type", C.c_void_p), ("mol", C.c_void_p), ("mass", C.c_void_p), ("charge", C.c_void_p),
                ("lj_eps", C.c_void_p), ("lj_sigma", C.c_void_p), ("tether_k", C.c_void_p),
                ("bond_idx", C.c_void_p), ("bond_k", C.c_void_p), ("bond_r0", C.c_void_p),
                ("angle_idx", C.c_void_p), ("angle_k", C.c_void_p), ("angle_th0", C.c_void_p),
                ("box", C.c_double * 3), ("r_cut", C.c_double), ("dsf_alpha", C.c_double), ("skin", C.c_double)]


class _Thermostat(C.Structure):
    _fields_ = [("kind", C.c_int32), ("gamma0", C.c_double), ("seed", C.c_uint64), ("n_seg", C.c_int32),
                ("a_gamma", C.c_double), ("gamma_min_frac", C.c_double), ("classical", C.c_int32)]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libqhp.so (built by `python -m paper_2212_03137_b200.build`).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2212_03137_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
        L.qhp_create.argtypes = [C.POINTER(_Topology), i32, i32, dbl, dbl, C.POINTER(_Thermostat), vp, C.POINTER(vp)]
        L.qhp_destroy.argtypes = [vp]
        L.qhp_set_state.argtypes = [vp, vp, vp, i64]
        L.qhp_get_state.argtypes = [vp, vp, vp, C.POINTER(i64)]
        L.qhp_set_state_host.argtypes = [vp, vp, vp, i64]
        L.qhp_get_state_host.argtypes = [vp, vp, vp, C.POINTER(i64)]
        L.qhp_step.argtypes = [vp, i64]
        L.qhp_set_respa.argtypes = [vp, i32]
        L.qhp_set_a_block.argtypes = [vp, i32]
        L.qhp_set_contraction.argtypes = [vp, i32]
        L.qhp_forces.argtypes = [vp, vp]
        L.qhp_set_comm.argtypes = [vp, i32, i32, ALLGATHER_FN, vp]
        L.qhp_pair_slices.argtypes = [vp, i32]
        L.qhp_observables.argtypes = [vp, vp, i32]
        L.qhp_observables_host.argtypes = [vp, vp, i32]
        L.qhp_neighbor_lists.argtypes = [vp, vp, vp, vp, vp]
        L.qhp_pair_list.argtypes = [vp, vp, vp, i64, C.POINTER(i64)]
        L.qhp_contracted.argtypes = [vp, vp]
        L.qhp_adqtb_gamma.argtypes = [vp, vp]
        L.qhp_adqtb_ratio.argtypes = [vp, vp]
        L.qhp_adqtb_kappa.argtypes = [vp, vp]
        L.qhp_adqtb_segment.argtypes = [vp, vp, vp]
        L.qhp_counters.argtypes = [vp, C.POINTER(i64), i32]
        L.qhp_check.argtypes = [vp]
        L.qhp_profile.argtypes = [vp, i32]
        L.qhp_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
        L.qhp_last_error.argtypes = [vp]
        L.qhp_last_error.restype = C.c_char_p
        L.qhp_philox_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, i64, vp, vp, vp]
        L.qhp_fft_c2c.argtypes = [vp, i32, i64, i32, vp]
        L.qhp_dfma_probe.argtypes = [vp, i32, i32, i64, vp]
        L.qhp_pibar.argtypes = [vp, i64, vp, i64, C.c_double, i32, C.c_double, vp, C.POINTER(C.c_double), C.POINTER(i32)]
        L.qhp_set_pair_prune.argtypes = [vp, C.c_double]
        L.qhp_pair_prune_stats.argtypes = [vp, C.POINTER(C.c_int64)]
        L.qhp_adqtb_set_gamma.argtypes = [vp, vp]
        L.qhp_profile_read_pair.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.qhp_pibar_noalloc.argtypes = [vp, i64, vp, i64, C.c_double, i32, C.c_double, vp, vp]
        for name in SYMBOLS:
            if name != "qhp_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2212_03137_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream=None):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _chk_dev(t, dtype, numel=None, name="tensor"):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")


class System:
    """One qhp_system.  Methods mirror the C ABI (qhp_<name>)."""

    def __init__(self, top: dict, P: int, P_contract: int, dt_ps: float, T_K: float, thermostat: str | int = "none",
                 gamma0: float = 1.0, seed: int = 0, n_seg: int = 0, a_gamma: float = 0.0,
                 gamma_min_frac: float = 0.01, classical: bool = False, stream=None):
        torch = _torch()
        self._h = C.c_void_p()
        self._L = lib()
        kinds = {"none": 0, "pile": 1, "adqtb": 2}
        kind = kinds[thermostat] if isinstance(thermostat, str) else int(thermostat)
        keep = {}
        t = _Topology()
        t.n_atoms, t.n_types = int(top["n_atoms"]), int(top["n_types"])
        t.n_bonds, t.n_angles = int(top["n_bonds"]), int(top["n_angles"])
        for k in ("type", "mol", "bond_idx", "angle_idx"):
            keep[k] = np.ascontiguousarray(top[k], dtype=np.int32)
            setattr(t, k, keep[k].ctypes.data_as(C.c_void_p))
        for k in ("mass", "charge", "lj_eps", "lj_sigma", "bond_k", "bond_r0", "angle_k", "angle_th0"):
            keep[k] = np.ascontiguousarray(top[k], dtype=np.float64)
            setattr(t, k, keep[k].ctypes.data_as(C.c_void_p))
        if top.get("tether_k") is not None:
            keep["tether_k"] = np.ascontiguousarray(top["tether_k"], dtype=np.float64)
            t.tether_k = keep["tether_k"].ctypes.data_as(C.c_void_p)
        for d in range(3):
            t.box[d] = float(top["box"][d])
        t.r_cut, t.dsf_alpha, t.skin = float(top["r_cut"]), float(top["dsf_alpha"]), float(top["skin"])
        th = _Thermostat(kind, float(gamma0), int(seed), int(n_seg), float(a_gamma), float(gamma_min_frac),
                         int(bool(classical)))
        self.stream = torch.cuda.current_stream() if stream is None else stream
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.N, self.P, self.Pc, self.n_types, self.n_seg = t.n_atoms, int(P), int(P_contract), t.n_types, int(n_seg)
        rc = self._L.qhp_create(C.byref(t), int(P), int(P_contract), float(dt_ps), float(T_K), C.byref(th),
                                C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc != 0:
            raise QhpError(rc, (self._L.qhp_last_error(None) or b"").decode())

    # -- helpers
    def _ok(self, rc):
        if rc != 0:
            raise QhpError(rc, (self._L.qhp_last_error(self._h) or b"").decode())

    def _empty(self, shape, dtype=None):
        torch = _torch()
        return torch.empty(shape, dtype=dtype or torch.float64, device=self.device)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._L.qhp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- C ABI
    def set_state(self, x_beads, p_beads, step0: int = 0):
        torch = _torch()
        n = self.P * self.N * 3
        _chk_dev(x_beads, torch.float64, n, "x_beads")
        _chk_dev(p_beads, torch.float64, n, "p_beads")
        self._ok(self._L.qhp_set_state(self._h, _ptr(x_beads), _ptr(p_beads), int(step0)))

    def get_state(self):
        x, p = self._empty((self.P, self.N, 3)), self._empty((self.P, self.N, 3))
        step = C.c_int64()
        self._ok(self._L.qhp_get_state(self._h, _ptr(x), _ptr(p), C.byref(step)))
        return x, p, step.value

    def set_state_host(self, x_host, p_host, step0: int = 0):
        """x_host, p_host: CPU tensors / numpy arrays [P][N][3] fp64 (pinned for full PCIe speed)."""
        self._ok(self._L.qhp_set_state_host(self._h, _host_ptr(x_host, self.P * self.N * 3),
                                            _host_ptr(p_host, self.P * self.N * 3), int(step0)))

    def get_state_host(self, x_host, p_host):
        step = C.c_int64()
        self._ok(self._L.qhp_get_state_host(self._h, _host_ptr(x_host, self.P * self.N * 3),
                                            _host_ptr(p_host, self.P * self.N * 3), C.byref(step)))
        return step.value

    def adqtb_ratio(self, tau_ps):
        """tau_ps: per-type time constants in ps (> 0: RATIO, <= 0: SIMPLE), or None."""
        if tau_ps is None:
            self._ok(self._L.qhp_adqtb_ratio(self._h, None))
            return
        tau = np.ascontiguousarray(tau_ps, dtype=np.float64)
        if tau.size != self.n_types:
            raise ValueError("tau_ps: one value per atom type")
        self._ok(self._L.qhp_adqtb_ratio(self._h, tau.ctypes.data_as(C.c_void_p)))

    def adqtb_kappa(self, kappa):
        """kappa: kernel-correction factor kappa(omega_j), j = 0..n_seg, on the noise filter H (reading G11), or None."""
        if kappa is None:
            self._ok(self._L.qhp_adqtb_kappa(self._h, None))
            return
        k = np.ascontiguousarray(kappa, dtype=np.float64)
        if k.shape != (self.n_seg + 1,):
            raise ValueError("kappa: one value per frequency omega_j, j = 0..n_seg")
        self._ok(self._L.qhp_adqtb_kappa(self._h, k.ctypes.data_as(C.c_void_p)))

    def set_comm(self, rank: int, world: int, group=None):
        """Bead-sharded V_s over `world` processes: this rank evaluates P'/world contracted beads,
        the slow forces are all-gathered through torch.distributed (NCCL) on the library's stream.  Before set_state."""
        torch = _torch()
        if world <= 1:
            self._ok(self._L.qhp_set_comm(self._h, 0, 1, ALLGATHER_FN(0), None))
            self._comm_cb = None
            return
        stream = self.stream

        def cb(ctx, ptr, nbytes, rk, wd, cuda_stream):
            try:
                n = nbytes * wd // 8
                buf = _wrap_device_f64(ptr, n)
                with torch.cuda.stream(stream):
                    allgather_inplace(buf, rk, wd, group)
                return 0
            except Exception:
                return 1
        self._comm_cb = ALLGATHER_FN(cb)          # keep the callback alive as long as the system
        self._ok(self._L.qhp_set_comm(self._h, int(rank), int(world), self._comm_cb, None))

    def pair_slices(self, n_slices: int):
        """Test hook: F_s re-evaluated in n_slices bead slices (include/qhp.h)."""
        self._ok(self._L.qhp_pair_slices(self._h, int(n_slices)))

    def set_respa(self, n_alt: int):
        self._ok(self._L.qhp_set_respa(self._h, int(n_alt)))

    def set_contraction(self, variant: str):
        """"literal" (default, Eq. 20 as printed) or "trig" (Fourier interpolation; reading G3); before set_state."""
        self._ok(self._L.qhp_set_contraction(self._h, {"literal": 0, "trig": 1}[variant]))

    def set_pair_prune(self, prune_skin: float):
        """Pruned per-bead rows of the staged pair kernel (include/qhp.h): prune_skin in A (default 0.6), <= 0 off.
        Before set_state."""
        self._ok(self._L.qhp_set_pair_prune(self._h, float(prune_skin)))

    def pair_prune_stats(self) -> dict:
        """Parity hook (include/qhp.h qhp_pair_prune_stats)."""
        out = (C.c_int64 * 4)()
        self._ok(self._L.qhp_pair_prune_stats(self._h, out))
        return dict(zip(["active", "prunes", "entries", "pair_beads_in_cutoff"], [int(v) for v in out]))

    def set_a_block(self, kind: str):
        """"exact" (default) or "cayley" = BCOCB."""
        self._ok(self._L.qhp_set_a_block(self._h, {"exact": 0, "cayley": 1}[kind]))

    def step(self, nsteps: int):
        self._ok(self._L.qhp_step(self._h, int(nsteps)))

    def forces(self):
        f = self._empty((self.P, self.N, 3))
        self._ok(self._L.qhp_forces(self._h, _ptr(f)))
        return f

    def observables(self):
        out = self._empty((4,))
        self._ok(self._L.qhp_observables(self._h, _ptr(out), 4))
        return out

    def observables_host(self) -> np.ndarray:
        out = np.empty(4)
        self._ok(self._L.qhp_observables_host(self._h, out.ctypes.data_as(C.c_void_p), 4))
        return out

    def neighbor_lists(self):
        torch = _torch()
        nc = self._empty((3,), torch.int32)
        cell_of, order = self._empty((self.N,), torch.int32), self._empty((self.N,), torch.int32)
        # ncell is not known before the call: size cell_start generously from the box, then trim
        self._ok(self._L.qhp_neighbor_lists(self._h, _ptr(cell_of), _ptr(order), None, _ptr(nc)))
        ncell = int(nc.prod().item())
        cell_start = self._empty((ncell + 1,), torch.int32)
        self._ok(self._L.qhp_neighbor_lists(self._h, None, None, _ptr(cell_start), None))
        return nc, cell_of, order, cell_start

    def pair_list(self):
        torch = _torch()
        count = self._empty((self.N,), torch.int32)
        total = C.c_int64()
        self._ok(self._L.qhp_pair_list(self._h, _ptr(count), None, 0, C.byref(total)))
        nbr = self._empty((max(total.value, 1),), torch.int32)
        self._ok(self._L.qhp_pair_list(self._h, _ptr(count), _ptr(nbr), total.value, C.byref(total)))
        return count, nbr[:total.value]

    def contracted(self):
        xc = self._empty((self.Pc, self.N, 3))
        self._ok(self._L.qhp_contracted(self._h, _ptr(xc)))
        return xc

    def adqtb_gamma(self):
        g = self._empty((self.n_types, self.n_seg + 1))
        self._ok(self._L.qhp_adqtb_gamma(self._h, _ptr(g)))
        return g

    def adqtb_set_gamma(self, gamma):
        """Restart of an adapted adQTB run: gamma [n_types][n_seg+1] (CUDA fp64) as returned by adqtb_gamma."""
        torch = _torch()
        _chk_dev(gamma, torch.float64, self.n_types * (self.n_seg + 1), "gamma")
        self._ok(self._L.qhp_adqtb_set_gamma(self._h, _ptr(gamma)))

    def adqtb_segment(self, want_fc=True, want_v=True):
        Fc = self._empty((3 * self.N, self.n_seg)) if want_fc else None
        v = self._empty((3 * self.N, self.n_seg)) if want_v else None
        self._ok(self._L.qhp_adqtb_segment(self._h, _ptr(Fc), _ptr(v)))
        return Fc, v

    def counters(self) -> dict:
        out = (C.c_int64 * 8)()
        self._ok(self._L.qhp_counters(self._h, out, 8))
        keys = ["rebuilds", "list_entries", "pair_beads_in_cutoff", "list_capacity", "launches", "overflow",
                "staged", "staged_warps"]
        return dict(zip(keys, [int(v) for v in out]))

    def check(self):
        self._ok(self._L.qhp_check(self._h))

    def profile(self, enable: bool):
        self._ok(self._L.qhp_profile(self._h, int(bool(enable))))

    def profile_read_pair(self) -> dict:
        ms, n = (C.c_double * 3)(), (C.c_int64 * 3)()
        self._ok(self._L.qhp_profile_read_pair(self._h, ms, n))
        keys = ["k_prune_check", "k_prune", "k_pair_dense"]
        return {k: dict(ms=float(ms[i]), n=int(n[i])) for i, k in enumerate(keys)}

    def profile_read(self) -> dict:
        ms, n = (C.c_double * 5)(), (C.c_int64 * 5)()
        self._ok(self._L.qhp_profile_read(self._h, ms, n))
        keys = ["integrate", "rebuild", "pair", "qtb_generate", "qtb_adapt"]
        return {k: dict(ms=float(ms[i]), n=int(n[i])) for i, k in enumerate(keys)}


def _host_ptr(a, numel):
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != numel:
            raise TypeError("expected a contiguous CPU float64 tensor of the state's size")
        return C.c_void_p(a.data_ptr())
    a = np.asarray(a)
    if a.dtype != np.float64 or not a.flags.c_contiguous or a.size != numel:
        raise TypeError("expected a contiguous float64 array of the state's size")
    return a.ctypes.data_as(C.c_void_p)


# ---- stand-alone primitives --------------------------------------------------------------------
def qhp_philox_normals(seed: int, atom0: int, mode: int, tag: int, step: int, n: int, stream=None):
    torch = _torch()
    words = torch.empty((n, 4), dtype=torch.int32, device="cuda")
    z = torch.empty((n, 3), dtype=torch.float64, device="cuda")
    rc = lib().qhp_philox_normals(int(seed), int(atom0), int(mode), int(tag), int(step), int(n), _ptr(words), _ptr(z),
                                  _stream_ptr(stream))
    if rc:
        raise QhpError(rc, "qhp_philox_normals")
    return words, z


def qhp_fft_c2c(data, sign: int, stream=None):
    """data: CUDA tensor [batch][n][2] fp64 (or complex128 [batch][n]); transformed in place."""
    torch = _torch()
    view = torch.view_as_real(data) if data.is_complex() else data
    _chk_dev(view, torch.float64, None, "data")
    batch, n = view.shape[0], view.shape[1]
    rc = lib().qhp_fft_c2c(_ptr(view), int(n), int(batch), int(sign), _stream_ptr(stream))
    if rc:
        raise QhpError(rc, "qhp_fft_c2c")
    return data


def qhp_dfma_probe(grid: int, block: int, iters: int, stream=None):
    torch = _torch()
    sink = torch.empty(grid * block, dtype=torch.float64, device="cuda")
    rc = lib().qhp_dfma_probe(_ptr(sink), int(grid), int(block), int(iters), _stream_ptr(stream))
    if rc:
        raise QhpError(rc, "qhp_dfma_probe")
    return sink


def qhp_pibar(wA, wB, beta: float, max_iter: int = 1000, tol: float = 1e-13, stream=None):
    """PI-BAR (Eq. 27-28) on device series wA = U_B - U_A (samples of A), wB = U_A - U_B (samples
    of B); returns (dF, iterations)."""
    torch = _torch()
    _chk_dev(wA, torch.float64, None, "wA")
    _chk_dev(wB, torch.float64, None, "wB")
    dF, it = C.c_double(0.0), C.c_int32(0)
    rc = lib().qhp_pibar(_ptr(wA), int(wA.numel()), _ptr(wB), int(wB.numel()), float(beta), int(max_iter), float(tol),
                         _stream_ptr(stream), C.byref(dF), C.byref(it))
    if rc != 0:
        raise QhpError(rc, "qhp_pibar")
    return dF.value, it.value


PIBAR_NOALLOC_MAX_N = 512 * 256 * 64      # QHP_PIBAR_NOALLOC_MAX_N of include/qhp.h


def qhp_pibar_noalloc(wA, wB, beta: float, out, max_iter: int = 1000, tol: float = 1e-13, stream=None):
    """qhp_pibar without any allocation, copy or synchronisation (include/qhp.h): enqueues the estimator on the
    stream; `out` is a caller-owned CUDA tensor of 2 doubles that receives (dF, iterations) once the stream
    has run.  Series longer than PIBAR_NOALLOC_MAX_N are rejected.  Calls overlapping on the GPU race on the
    library's static scratch array: keep them on one stream."""
    torch = _torch()
    _chk_dev(wA, torch.float64, None, "wA")
    _chk_dev(wB, torch.float64, None, "wB")
    _chk_dev(out, torch.float64, 2, "out")
    rc = lib().qhp_pibar_noalloc(_ptr(wA), int(wA.numel()), _ptr(wB), int(wB.numel()), float(beta), int(max_iter),
                                 float(tol), _stream_ptr(stream), _ptr(out))
    if rc != 0:
        raise QhpError(rc, (lib().qhp_last_error(None) or b"qhp_pibar_noalloc").decode())
