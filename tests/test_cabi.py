"""CPU-side checks of the boundary: libqhp.so loads and exports every symbol include/qhp.h
declares; argument errors are reported by code (these paths return before any CUDA call)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from workloads import water as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2212_03137_b200 import build
    build.build()
    from paper_2212_03137_b200 import binding
    return binding.lib()


def test_exports_every_declared_symbol(lib):
    from paper_2212_03137_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "qhp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(qhp_[a-z0-9_]+)\s*\(", hdr)))
    assert declared, "no declarations parsed"
    assert sorted(binding.SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def _create(lib, top, P, Pc, dt, T, kind=0, gamma0=1.0, n_seg=0):
    from paper_2212_03137_b200.binding import _Thermostat, _Topology
    keep = []
    t = _Topology()
    t.n_atoms, t.n_types, t.n_bonds, t.n_angles = top["n_atoms"], top["n_types"], top["n_bonds"], top["n_angles"]
    for k in ("type", "mol", "bond_idx", "angle_idx"):
        a = np.ascontiguousarray(top[k], dtype=np.int32); keep.append(a)
        setattr(t, k, a.ctypes.data_as(C.c_void_p))
    for k in ("mass", "charge", "lj_eps", "lj_sigma", "bond_k", "bond_r0", "angle_k", "angle_th0"):
        a = np.ascontiguousarray(top[k], dtype=np.float64); keep.append(a)
        setattr(t, k, a.ctypes.data_as(C.c_void_p))
    for d in range(3):
        t.box[d] = float(top["box"][d])
    t.r_cut, t.dsf_alpha, t.skin = top["r_cut"], top["dsf_alpha"], top["skin"]
    th = _Thermostat(kind, gamma0, 1, n_seg, 0.5, 0.01, 0)
    h = C.c_void_p()
    rc = lib.qhp_create(C.byref(t), P, Pc, dt, T, C.byref(th), None, C.byref(h))
    return rc, h, (lib.qhp_last_error(None) or b"").decode()


def test_create_argument_errors(lib):
    top = W.water_box(27)
    top["box"] = np.array([20.0, 20.0, 20.0])
    EINVAL = -1
    assert _create(lib, top, 7, 7, 2.5e-4, 300.0)[0] == EINVAL               # unsupported P
    assert _create(lib, top, 8, 9, 2.5e-4, 300.0)[0] == EINVAL               # P_contract > P
    assert _create(lib, top, 8, 0, 2.5e-4, 300.0)[0] == EINVAL
    assert _create(lib, top, 8, 8, -1.0, 300.0)[0] == EINVAL
    assert _create(lib, top, 2, 1, 5e-4, 300.0, kind=2, gamma0=20.0, n_seg=64)[0] == EINVAL   # adQTB needs P = 1
    assert _create(lib, top, 1, 1, 5e-4, 300.0, kind=2, gamma0=20.0, n_seg=48)[0] == EINVAL   # n_seg not 2^k
    # documented limits of include/qhp.h: n_seg a power of two in [8, 2048]; qhp_fft_c2c n a power of two in [8, 8192]
    assert _create(lib, top, 1, 1, 5e-4, 300.0, kind=2, gamma0=20.0, n_seg=4)[0] == EINVAL
    assert _create(lib, top, 1, 1, 5e-4, 300.0, kind=2, gamma0=20.0, n_seg=4096)[0] == EINVAL
    one = C.c_double(0.0)
    for n in (4, 12, 16384):
        assert lib.qhp_fft_c2c(C.byref(one), n, 1, -1, None) == EINVAL
    small = dict(top); small["box"] = np.array([17.0, 20.0, 20.0])
    rc, _, msg = _create(lib, small, 8, 8, 2.5e-4, 300.0)
    assert rc == EINVAL and "box" in msg
    bad = dict(top); bad["mol"] = top["mol"][::-1].copy()
    assert _create(lib, bad, 8, 8, 2.5e-4, 300.0)[0] == EINVAL               # molecules not contiguous
    assert lib.qhp_step(None, 1) == EINVAL
    assert lib.qhp_destroy(None) == 0


def test_python_binding_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2212_03137_b200 as qhp
    top = W.water_box(27)
    top["box"] = np.array([20.0, 20.0, 20.0])
    with pytest.raises(RuntimeError):
        qhp.System(top, 1, 1, 5e-4, 300.0)
