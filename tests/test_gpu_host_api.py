"""The host entry points of the C ABI (the ones bench.py's end-to-end measurement goes through) and
the per-phase profiling / counter calls, against the device entry points and the oracle."""
import numpy as np
import pytest

from gpu_common import make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu


def test_host_state_round_trip_and_steps_match_device_path():
    import torch
    top = W.water_box(216)
    sysg, ref, x0, p0 = make_pair(top, 4, 2, 0.25, "pile")
    xh, ph = torch.as_tensor(x0).pin_memory(), torch.as_tensor(p0).pin_memory()
    sysg.set_state_host(xh, ph, 0)
    ref.set_state(x0, p0, 0)
    sysg.step(10)
    ref.step(10)
    xo, po = torch.empty_like(xh).pin_memory(), torch.empty_like(ph).pin_memory()
    assert sysg.get_state_host(xo, po) == 10
    xr, pr = ref.get_state()
    assert np.abs(xo.numpy() - xr).max() < 1e-8
    assert np.abs(po.numpy() - pr).max() < 1e-6 * np.abs(pr).max()
    # the same state through the device entry points
    x1, p1, st = sysg.get_state()
    assert st == 10 and np.array_equal(x1.cpu().numpy(), xo.numpy()) and np.array_equal(p1.cpu().numpy(), po.numpy())
    obs_h = np.asarray(sysg.observables_host())
    obs_d = sysg.observables().cpu().numpy()
    assert np.array_equal(obs_h, obs_d)
    assert np.abs(obs_h - ref.observables()).max() < 1e-7 * np.abs(ref.observables()).max()


def test_profile_and_counters_account_for_every_step():
    top = W.water_box(216)
    sysg, _, x0, p0 = make_pair(top, 2, 2, 0.25, "pile")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    c0 = sysg.counters()
    sysg.profile(True)
    sysg.step(7)
    prof = sysg.profile_read()
    sysg.profile(False)
    c1 = sysg.counters()
    assert prof["integrate"]["n"] == 7 and prof["pair"]["n"] == 7 and prof["rebuild"]["n"] == 7
    assert prof["integrate"]["ms"] > 0 and prof["pair"]["ms"] > 0
    assert prof["qtb_generate"]["n"] == 0 and prof["qtb_adapt"]["n"] == 0
    assert c1["launches"] - c0["launches"] == 7 * 3          # integrator + the fused rebuild chain (one cooperative launch) + pair forces
    assert c1["overflow"] == 0 and c1["pair_beads_in_cutoff"] > 0 and c1["list_entries"] >= c1["pair_beads_in_cutoff"] // 2
    sysg.check()


def test_graph_replay_equals_step_by_step():
    """Small (launch-bound) systems replay qhp_step from a CUDA graph of 32 steps (include/qhp.h): same kernels, same
    arguments, Philox step index from device memory -> the trajectory is bit-identical to one advanced a step at a
    time, list rebuilds and a get_state in the middle included; the launch counter counts the replayed kernels."""
    import torch
    top = W.water_box(216)
    a, _, x0, p0 = make_pair(top, 8, 8, 0.25, "pile")
    b, _, _, _ = make_pair(top, 8, 8, 0.25, "pile")
    for s in (a, b):
        s.set_state(to_dev(x0), to_dev(p0), 0)
    la = a.counters()["launches"]
    a.step(150)                          # odd remainder, > 2 graphs
    assert a.counters()["launches"] - la == 150 * 3
    xa, pa, sa = a.get_state()           # flushes the pending kick: the next call starts outside the steady state
    a.step(101)
    for _ in range(150):
        b.step(1)
    xb, pb, sb = b.get_state()
    assert sa == sb == 150 and torch.equal(xa, xb) and torch.equal(pa, pb)
    for _ in range(101):
        b.step(1)
    xa, pa, sa = a.get_state()
    xb, pb, sb = b.get_state()
    assert sa == sb == 251 and torch.equal(xa, xb) and torch.equal(pa, pb)
    assert a.counters()["rebuilds"] == b.counters()["rebuilds"] > 1
    a.check()
    # the graph path is the faster one on this launch-bound box (0.079 -> 0.073 ms per step on a B200): not asserted as a
    # time, but it must have been taken -- a profiled run uses plain launches and gives the same trajectory again
    c, _, _, _ = make_pair(top, 8, 8, 0.25, "pile")
    c.set_state(to_dev(x0), to_dev(p0), 0)
    c.profile(True)
    c.step(150)
    c.profile(False)
    xc, pc, _ = c.get_state()
    c.step(101)
    xc, pc, sc = c.get_state()
    assert sc == 251 and torch.equal(xa, xc) and torch.equal(pa, pc)
