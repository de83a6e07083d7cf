"""Full-size parity at BASELINE.json's 216,000-atom configurations, in the launch configuration
bench.py times (configs[4] = C4: P = 32, P' = 4, PILE; configs[3] = C3: adQTB, n_seg = 1024).

The oracle's cell-list force routine (validated against its own O(N^2) routine in
tests/test_oracle_forces.py) makes whole-box forces affordable, so forces and the first steps are
compared on EVERY atom; neighbour rows and coloured-noise rows, which the oracle computes one by
one, are compared on a seeded sample.  Tolerances are BASELINE.json north_star's."""
import numpy as np
import pytest

from gpu_common import make_pair, oracle_adapt_from_segment, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

FTOL = 1e-10     # relative to max|F|
XTOL = 1e-8      # Angstrom


def _sample_atoms(n_atoms, k, seed):
    rng = np.random.Generator(np.random.Philox(key=[W.MASTER_SEED, seed]))
    s = rng.choice(n_atoms, size=k, replace=False)
    return np.concatenate([s, [0, 1, 2, n_atoms - 1]])          # plus the ends of the box


def _rows_from_gpu(sysg):
    count, nbr = sysg.pair_list()
    count = count.cpu().numpy().astype(np.int64)
    start = np.concatenate([[0], np.cumsum(count)])
    return count, start, nbr


def _check_lists(sysg, otop, cent, sample):
    import oracle as O
    nc, cell_of, order, cell_start = sysg.neighbor_lists()
    onc, ocell_of, oorder, ocell_start = O.cells(otop, cent)
    assert np.array_equal(nc.cpu().numpy(), onc)
    assert np.array_equal(cell_of.cpu().numpy(), ocell_of)
    assert np.array_equal(order.cpu().numpy(), oorder)
    assert np.array_equal(cell_start.cpu().numpy(), ocell_start)
    count, start, nbr = _rows_from_gpu(sysg)
    for i in sample:
        row = np.sort(nbr[start[i]:start[i + 1]].cpu().numpy())
        assert np.array_equal(row, np.sort(O.neighbours_of(otop, cent, int(i)))), f"neighbour row of atom {i}"
    # properties that hold at any size: symmetric full list, no self or intramolecular entries
    assert int(count.sum()) % 2 == 0
    i_of = np.repeat(np.arange(count.size), count)
    j_of = nbr.cpu().numpy()
    assert not np.any(i_of // 3 == j_of // 3)
    assert (i_of < j_of).sum() * 2 == i_of.size


def test_c4_full_size_lists_forces_steps():
    import oracle as O
    cfg = W.CONFIGS["C4"]
    top = W.water_box(cfg["n_mol"])
    P, Pc = cfg["P"], cfg["P_contract"]
    sysg, ref, x0, p0 = make_pair(top, P, Pc, cfg["dt_fs"], "pile", gamma0=cfg["gamma0"])
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1                       # the kernel bench.py times
    otop = O.Topology(top)
    cent = O.beads_to_nm(x0)[0]
    _check_lists(sysg, otop, cent, _sample_atoms(top["n_atoms"], 24, 11))
    ref.set_state(x0, p0, 0)
    G = sysg.forces().cpu().numpy()
    Gref = ref.forces()
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    sysg.step(10)                                               # half of north_star's 20 steps at full size
    ref.step(10)                                                # (~25 s per oracle step); 20 steps: smaller boxes
    x1, p1, st = sysg.get_state()
    xr, pr = ref.get_state()
    assert st == 10
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    assert np.abs(p1.cpu().numpy() - pr).max() < 1e-9 * np.abs(pr).max()
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-9 * np.abs(oref).max()
    sysg.check()


def test_c3_full_size_lists_forces_noise_steps():
    import ctypes as C
    import oracle as O
    cfg = W.CONFIGS["C3"]
    top = W.water_box(cfg["n_mol"])
    n_seg, dt = cfg["n_seg"], cfg["dt_fs"] * 1e-3
    sysg, ref, x0, p0 = make_pair(top, 1, 1, cfg["dt_fs"], "adqtb", gamma0=cfg["gamma0"], n_seg=n_seg,
                                  a_gamma=cfg["a_gamma"])
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1
    otop = O.Topology(top)
    sample = _sample_atoms(top["n_atoms"], 12, 12)
    _check_lists(sysg, otop, x0[0], sample)
    ref.set_state(x0, p0, 0)                                    # whole-box forces (oracle cell routine)
    G = sysg.forces().cpu().numpy().reshape(-1)
    assert np.abs(G - ref.F).max() < FTOL * np.abs(ref.F).max()
    sysg.step(1)
    # coloured force of the first segment: sampled rows against the oracle's FFT route (itself pinned
    # to the direct convolution sum in tests/test_oracle_adqtb.py); the oracle needs ~1 ms per atom
    Fc_dev, _ = sysg.adqtb_segment(want_v=False)
    sample = np.sort(sample)
    rows = (3 * sample[:, None] + np.arange(3)[None, :]).reshape(-1)
    import torch
    Fc_s = Fc_dev[torch.as_tensor(rows, device=Fc_dev.device)].cpu().numpy()
    Fref = O.qtb_colored_fft(otop, n_seg, W.MASTER_SEED, 0, ref.kernels(), atoms=sample)
    assert np.abs(Fc_s - Fref).max() < 1e-11 * np.sqrt((Fref ** 2).mean())
    del Fc_dev
    # first step: the position of an atom after one B A O A B step depends on the noise of that atom
    # only, so the oracle stepper is run on the whole box with its coloured force filled in for the
    # sampled atoms (zero elsewhere) and the sampled atoms are compared
    Fc1 = np.zeros((3 * top["n_atoms"], 1))
    Fc1[rows, 0] = Fref[:, 0]
    v1 = np.zeros_like(Fc1)
    O.lib().qo_adqtb_steps(otop.ref, C.c_double(dt), C.c_double(cfg["gamma0"]), C.c_int(1), C.c_int(0),
                           C.c_int(1), ref.x.ctypes.data_as(C.c_void_p), ref.p.ctypes.data_as(C.c_void_p),
                           ref.F.ctypes.data_as(C.c_void_p), Fc1.ctypes.data_as(C.c_void_p),
                           v1.ctypes.data_as(C.c_void_p), C.c_int(ref.uc))
    x1, _, st = sysg.get_state()
    assert st == 1
    assert np.abs(x1.cpu().numpy().reshape(-1)[rows] - ref.x[rows]).max() < XTOL
    sysg.step(3)
    sysg.check()


def test_c3_box_every_dof_segment_end_at_bench_size():
    """216,000 atoms, adQTB with n_seg = 64 (segment arrays 332 MB instead of 5.3 GB): two whole segments, so
    that the spectra launch over all 648,000 DOF, the fixed-order reduction of its per-CTA partials and the
    adaptation run at the size bench.py times; gamma_z to 1e-9 of the oracle's update of the product's own
    segment arrays (every DOF enters the per-type means)."""
    import oracle as O
    cfg = W.CONFIGS["C3"]
    top = W.water_box(cfg["n_mol"])
    n_seg, dt, g0 = 64, cfg["dt_fs"] * 1e-3, cfg["gamma0"]
    sysg, _, x0, p0 = make_pair(top, 1, 1, cfg["dt_fs"], "adqtb", gamma0=g0, n_seg=n_seg, a_gamma=cfg["a_gamma"])
    otop = O.Topology(top)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    g_prev = np.full((otop.n_types, n_seg + 1), g0)
    for seg in range(2):
        sysg.step(n_seg)
        Fc, v = sysg.adqtb_segment()
        g = sysg.adqtb_gamma().cpu().numpy()
        g_ref, _ = oracle_adapt_from_segment(otop, n_seg, dt, g0, cfg["a_gamma"], 0.01, v.cpu().numpy(),
                                             Fc.cpu().numpy(), g_prev)
        del Fc, v
        assert np.abs(g - g_ref).max() < 1e-9 * np.abs(g_ref).max(), seg
        assert np.abs(g - g_prev).max() > 1e-3
        g_prev = g
    sysg.check()
