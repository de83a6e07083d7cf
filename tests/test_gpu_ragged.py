"""Ragged-molecule parity case: waters mixed with one-atom ions and two-atom molecules, four atom types
(workloads.water.ionic_water_box).  Tiles of the fused integrator, bonded ranges, intramolecular
exclusions and the per-type tables (pair parameters, adQTB gamma_z) must not assume O,H,H triples."""
import numpy as np
import pytest

from gpu_common import T_K, make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

FTOL, XTOL = 1e-10, 1e-8


@pytest.mark.parametrize("n_sites,P,Pc,staged", [(216, 4, 2, 0), (1728, 2, 1, 0), (5832, 4, 2, 1)])
def test_lists_forces_and_steps(n_sites, P, Pc, staged):
    import oracle as O
    top = W.ionic_water_box(n_sites)
    assert set(np.bincount(top["mol"])) == {1, 2, 3}
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    assert sysg.counters()["staged"] == staged
    otop = O.Topology(top)
    nc, cell_of, order, cell_start = sysg.neighbor_lists()
    onc, ocell_of, oorder, ocell_start = O.cells(otop, O.beads_to_nm(x0)[0])
    assert np.array_equal(nc.cpu().numpy(), onc) and np.array_equal(cell_of.cpu().numpy(), ocell_of)
    assert np.array_equal(order.cpu().numpy(), oorder) and np.array_equal(cell_start.cpu().numpy(), ocell_start)
    count, nbr = sysg.pair_list()
    count = count.cpu().numpy().astype(np.int64)
    i = np.repeat(np.arange(count.size), count)
    j = nbr.cpu().numpy().astype(np.int64)
    half = np.stack([i[i < j], j[i < j]], 1)
    half = half[np.lexsort((half[:, 1], half[:, 0]))]
    assert np.array_equal(half, O.pairs_brute(otop, O.beads_to_nm(x0)[0]))      # the O(N^2) definition
    G = sysg.forces().cpu().numpy()
    Gref = O.bead_forces(otop, P, Pc, x0)
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-10 * np.abs(oref).max()
    n = 20 if n_sites < 2000 else 6
    sysg.step(n); ref.step(n)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()


def test_adqtb_four_types_thread_per_molecule_integrator():
    """P = 1: the thread-per-molecule integrator with molecules of 1, 2 and 3 atoms; gamma_z for 4 types."""
    top = W.ionic_water_box(216)
    n_seg = 32
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    for seg in range(2):
        sysg.step(n_seg); ref.step(n_seg)
        g = sysg.adqtb_gamma().cpu().numpy()
        assert g.shape[0] == 4
        assert np.abs(g - ref.gamma).max() < 1e-9 * ref.gamma.max()
    sysg.step(5); ref.step(5)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()
