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
