"""Pruned per-bead rows of the staged pair kernel (include/qhp.h qhp_set_pair_prune; R8).
The rows are an acceleration structure: the pair set V_s is summed over must still be every pair inside r_c.
A pair dropped near r_c is invisible in the forces (the shifted force vanishes there), so the sharp pin is the
integer: the number of pairs the pruned rows deliver inside r_c equals the count on the centroid table (itself
pinned to a KD-tree count in test_gpu_rpmd.py) at every step of a run with prunes and list rebuilds in it."""
import numpy as np
import pytest

from gpu_common import make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("P,Pc,dt_fs,thermo", [(4, 2, 0.5, "pile"), (1, 1, 1.0, "pile")])
def test_pruned_rows_hold_every_pair_inside_the_cutoff(P, Pc, dt_fs, thermo):
    top = W.water_box(5832)
    sysg, _, x0, p0 = make_pair(top, P, Pc, dt_fs, thermo, sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    st = sysg.pair_prune_stats()
    assert st["active"] == 1 and st["prunes"] == Pc                 # one prune per bead at set_state
    assert st["pair_beads_in_cutoff"] == sysg.counters()["pair_beads_in_cutoff"]
    full = sysg.counters()["list_entries"] * Pc
    assert st["pair_beads_in_cutoff"] <= st["entries"] < 0.8 * full  # the rows are denser than the centroid table
    r0 = sysg.counters()["rebuilds"]
    seen = [st["prunes"]]
    for _ in range(24):
        sysg.step(2)
        st = sysg.pair_prune_stats()
        assert st["pair_beads_in_cutoff"] == sysg.counters()["pair_beads_in_cutoff"]
        seen.append(st["prunes"])
    sysg.check()
    steps = 48
    assert sysg.counters()["rebuilds"] > r0                         # a list rebuild fell inside (rows renewed after it)
    assert Pc * 3 <= seen[-1] < Pc * steps // 2                      # several prunes, but not one per step
    assert any(a == b for a, b in zip(seen, seen[1:]))              # steps without a prune exist


def test_forces_and_trajectory_equal_the_unpruned_path():
    """Same seeded system with and without pruned rows: forces agree to rounding (summation order), and so do the
    positions after 40 steps with prunes and a rebuild in them; both against the oracle in test_gpu_rpmd.py."""
    import paper_2212_03137_b200 as qhp
    top = W.water_box(5832)
    a, _, x0, p0 = make_pair(top, 4, 2, 0.5, "pile", sigma_bead=0.05)
    b, _, _, _ = make_pair(top, 4, 2, 0.5, "pile", sigma_bead=0.05)
    b.set_pair_prune(0.0)
    for s in (a, b):
        s.set_state(to_dev(x0), to_dev(p0), 0)
    assert a.pair_prune_stats()["active"] == 1 and b.pair_prune_stats()["active"] == 0
    Fa, Fb = a.forces().cpu().numpy(), b.forces().cpu().numpy()
    assert np.abs(Fa - Fb).max() < 1e-12 * np.abs(Fb).max()
    a.step(40)
    b.step(40)
    xa, pa, _ = a.get_state()
    xb, pb, _ = b.get_state()
    assert (xa - xb).abs().max().item() < 1e-9
    assert (pa - pb).abs().max().item() < 1e-9 * pb.abs().max().item()
    assert a.pair_prune_stats()["prunes"] > 2
    with pytest.raises(qhp.QhpError):
        a.set_pair_prune(0.3)                                       # only before set_state


def test_prune_skin_at_or_above_the_list_skin_falls_back():
    top = W.water_box(5832)
    s, _, x0, p0 = make_pair(top, 1, 1, 0.5, "pile")
    s.set_pair_prune(top["skin"])
    s.set_state(to_dev(x0), to_dev(p0), 0)
    assert s.pair_prune_stats()["active"] == 0 and s.counters()["staged"] == 1
    s.step(3)
    s.check()


def test_pair_phase_is_timed_launch_by_launch():
    """qhp_profile_read_pair: one interval per step for each of k_prune_check, k_prune, k_pair_dense inside the pair
    phase of qhp_profile_read; the three together do not exceed the phase."""
    top = W.water_box(5832)
    s, _, x0, p0 = make_pair(top, 4, 2, 0.25, "pile")
    s.set_state(to_dev(x0), to_dev(p0), 0)
    s.step(3)
    s.profile(True)
    s.step(6)
    ph, pp = s.profile_read(), s.profile_read_pair()
    s.profile(False)
    assert ph["pair"]["n"] == 6
    assert all(pp[k]["n"] == 6 and pp[k]["ms"] > 0 for k in ("k_prune_check", "k_prune", "k_pair_dense"))
    assert sum(v["ms"] for v in pp.values()) <= ph["pair"]["ms"] * 1.001
    assert pp["k_pair_dense"]["ms"] > pp["k_prune_check"]["ms"]
    u = make_pair(top, 4, 2, 0.25, "pile")[0]
    u.set_pair_prune(0.0)
    u.set_state(to_dev(x0), to_dev(p0), 0)
    u.profile(True)
    u.step(2)
    assert all(v["n"] == 0 for v in u.profile_read_pair().values()) and u.profile_read()["pair"]["n"] == 2
