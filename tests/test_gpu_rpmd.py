"""GPU-vs-oracle parity of the RPMD path (BASELINE.json north_star tolerances):
neighbour objects bit-exact; forces within 1e-10 * max|F|; positions within 1e-8 A after 20 steps."""
import numpy as np
import pytest

from gpu_common import T_K, make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

FTOL = 1e-10     # relative to max|F|   (north_star)
XTOL = 1e-8      # Angstrom after 20 steps (north_star)


def _lists_check(sysg, top, x0):
    import oracle as O
    otop = O.Topology(top)
    cent = x0.mean(axis=0)
    nc, cell_of, order, cell_start = sysg.neighbor_lists()
    onc, ocell_of, oorder, ocell_start = O.cells(otop, O.beads_to_nm(x0)[0])
    assert np.array_equal(nc.cpu().numpy(), onc)
    assert np.array_equal(cell_of.cpu().numpy(), ocell_of)
    assert np.array_equal(order.cpu().numpy(), oorder)
    assert np.array_equal(cell_start.cpu().numpy(), ocell_start)
    return otop, O.beads_to_nm(x0)[0]


def _pairs_from_gpu(sysg):
    count, nbr = sysg.pair_list()
    count = count.cpu().numpy().astype(np.int64)
    nbr = nbr.cpu().numpy().astype(np.int64)
    i = np.repeat(np.arange(count.size), count)
    return count, i, nbr


@pytest.mark.parametrize("n_mol,P,Pc", [(216, 8, 8), (216, 8, 4), (343, 3, 2)])
def test_small_box_lists_forces_observables(n_mol, P, Pc):
    import oracle as O
    top = W.water_box(n_mol)
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    otop, cent = _lists_check(sysg, top, x0)
    # pair set == brute force definition, bit-exact
    count, i, j = _pairs_from_gpu(sysg)
    half = np.stack([i[i < j], j[i < j]], 1)
    half = half[np.lexsort((half[:, 1], half[:, 0]))]
    assert np.array_equal(half, O.pairs_brute(otop, cent))
    assert (i < j).sum() * 2 == i.size                      # full list is symmetric
    # contraction
    xc = sysg.contracted().cpu().numpy()
    assert np.abs(xc - O.contract(ref.Q, Pc)).max() < 1e-13
    # forces
    G = sysg.forces().cpu().numpy()
    Gref = O.bead_forces(otop, P, Pc, x0)
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    # observables
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-10 * np.abs(oref).max()
    # state round trip through the normal modes
    x1, p1, step = sysg.get_state()
    assert step == 0
    assert np.abs(x1.cpu().numpy() - x0).max() < 1e-13 and np.abs(p1.cpu().numpy() - p0).max() < 1e-11


@pytest.mark.parametrize("thermo,P,Pc", [("pile", 8, 8), ("none", 8, 8), ("pile", 8, 4), ("pile", 1, 1)])
def test_c0_20_steps_positions(thermo, P, Pc):
    """configs[0]: 216 waters, P = 8, dt = 0.25 fs, PILE gamma0 = 1/ps (plus contracted / classical variants)."""
    top = W.water_box(216)
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.25, thermo, gamma0=1.0)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(7)
    sysg.step(13)                       # two calls: the deferred half kick must carry over
    ref.step(20)
    x1, p1, step = sysg.get_state()
    xr, pr = ref.get_state()
    assert step == 20
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    assert np.abs(p1.cpu().numpy() - pr).max() < 1e-6 * np.abs(pr).max()
    G = sysg.forces().cpu().numpy()
    Gr = ref.forces()
    assert np.abs(G - Gr).max() < 1e-7 * np.abs(Gr).max()    # forces at positions that agree to 1e-8 A
    sysg.check()


def test_resume_is_bit_identical():
    top = W.water_box(216)
    sysg, _, x0, p0 = make_pair(top, 8, 4, 0.25, "pile")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    sysg.step(10)
    xa, pa, st = sysg.get_state()
    sysg.step(10)
    xb, pb, _ = sysg.get_state()
    sys2, _, _, _ = make_pair(top, 8, 4, 0.25, "pile")
    sys2.set_state(xa.clone(), pa.clone(), st)
    sys2.step(10)
    xc, pc, st2 = sys2.get_state()
    assert st2 == 20
    # get_state/set_state pass through the bead representation: equal up to the round trip
    assert (xb - xc).abs().max().item() < 1e-12
    assert (pb - pc).abs().max().item() < 1e-9


def test_c2_lists_forces_steps():
    """configs[2]: 4096 waters (12,288 atoms), P = 32, P' = 4: cell path (4x4x4 cells), several tiles,
    ragged last tile."""
    import oracle as O
    top = W.water_box(4096)
    sysg, ref, x0, p0 = make_pair(top, 32, 4, 0.25, "pile")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1      # 5184-atom neighbourhoods: the staged kernel without its fp32 copy
    ref.set_state(x0, p0, 0)
    otop, cent = _lists_check(sysg, top, x0)
    count, i, j = _pairs_from_gpu(sysg)
    half = np.stack([i[i < j], j[i < j]], 1)
    half = half[np.lexsort((half[:, 1], half[:, 0]))]
    assert np.array_equal(half, O.pairs_brute(otop, cent))
    G = sysg.forces().cpu().numpy()
    Gref = O.bead_forces(otop, 32, 4, x0)
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    sysg.step(20)
    ref.step(20)
    x1, _, _ = sysg.get_state()
    xr, _ = ref.get_state()
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-8 * np.abs(oref).max()
    sysg.check()


@pytest.mark.parametrize("P,Pc,skin,min_rebuilds", [(1, 1, 0.1, 5), (4, 2, 0.7, 1)])
def test_rebuild_during_run_keeps_parity(P, Pc, skin, min_rebuilds):
    """A small skin forces list rebuilds inside qhp_step; forces must not depend on the list."""
    top = W.water_box(216)
    top["skin"] = skin
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.5, "pile", gamma0=5.0, sigma_bead=0.002)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(20)
    ref.step(20)
    x1, _, _ = sysg.get_state()
    xr, _ = ref.get_state()
    sysg.check()
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    c = sysg.counters()
    assert c["rebuilds"] >= 1 + min_rebuilds and c["overflow"] == 0


def test_skin_smaller_than_bead_spread_is_reported():
    """A centroid list cannot cover beads farther than skin/2 from their centroid: ESTATE at check."""
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    top["skin"] = 0.05
    sysg, _, x0, p0 = make_pair(top, 4, 2, 0.5, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    with pytest.raises(qhp.QhpError):
        sysg.check()


def test_skin_guard_uses_the_norm_of_the_bead_offset():
    """One bead pair displaced by (d, d, d) with d < skin/2 < sqrt(3) d: every component is inside the bound,
    the distance is not -- the guard must fire (it compared components)."""
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    top["skin"] = 1.0
    sysg, _, x0, p0 = make_pair(top, 2, 2, 0.5, "pile", sigma_bead=0.0)
    x0 = x0.copy()
    x0[0, 0, :] += 0.4
    x0[1, 0, :] -= 0.4
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    with pytest.raises(qhp.QhpError):
        sysg.check()
    # the same displacement along one axis only stays inside skin/2: accepted
    sysg2, _, x0, p0 = make_pair(top, 2, 2, 0.5, "pile", sigma_bead=0.0)
    x0 = x0.copy()
    x0[0, 0, 0] += 0.4
    x0[1, 0, 0] -= 0.4
    sysg2.set_state(to_dev(x0), to_dev(p0), 0)
    sysg2.check()


def test_harmonic_oscillators_single_atom_molecules():
    """Tethered, non-interacting atoms (each its own molecule, no bonds): the harmonic system of the
    closed-form pins; exercises tether forces and ragged tiles."""
    top = W.oscillator_box(1000, 1.008, 769.3)
    sysg, ref, x0, p0 = make_pair(top, 6, 6, 0.25, "pile", gamma0=2.0, sigma_bead=0.02)
    sysg.set_state(to_dev(x0), to_dev(p0), 5)
    ref.set_state(x0, p0, 5)
    sysg.step(20)
    ref.step(20)
    x1, _, st = sysg.get_state()
    xr, _ = ref.get_state()
    assert st == 25
    assert np.abs(x1.cpu().numpy() - xr).max() < 1e-10
    obs = sysg.observables().cpu().numpy()
    assert np.abs(obs - ref.observables()).max() < 1e-9 * np.abs(ref.observables()).max()


def test_step_sees_the_error_flags_without_a_check():
    """qhp_step polls the device error flags asynchronously (include/qhp.h): a run with a list that cannot cover its
    beads stops at a later qhp_step call instead of going on until someone calls qhp_check."""
    import torch
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    top["skin"] = 0.05
    sysg, _, x0, p0 = make_pair(top, 4, 2, 0.5, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    sysg.step(2)                                   # the flag copy is enqueued behind these steps
    torch.cuda.synchronize()
    with pytest.raises(qhp.QhpError, match="skin too small"):
        sysg.step(2)
    good = W.water_box(216)
    sysg2, _, x0, p0 = make_pair(good, 4, 2, 0.5, "pile")
    sysg2.set_state(to_dev(x0), to_dev(p0), 0)
    for _ in range(3):
        sysg2.step(300)                            # crosses the 256-step poll inside a call
        torch.cuda.synchronize()
    sysg2.check()


def test_staged_pretest_rejects_no_pair_inside_the_cutoff():
    """The staged kernel drops list entries by a packed-half distance pre-test before the fp64 test.  A pair it
    wrongly dropped near r_c would be invisible in the forces (the shifted force vanishes at r_c), so the
    pre-test is pinned by the integer it must not change: the number of in-cutoff (ordered) pair-beads equals
    a KD-tree count on the oracle's contracted beads (Eq. 20), intramolecular pairs excluded."""
    import oracle as O
    from scipy.spatial import cKDTree
    top = W.water_box(5832)
    sysg, _, x0, p0 = make_pair(top, 4, 2, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    c = sysg.counters()
    assert c["staged"] == 1 and c["overflow"] == 0
    xc = O.contract(O.beads_to_nm(x0), 2)
    L = top["box"]
    want = 0
    for b in range(2):
        pr = cKDTree(np.mod(xc[b], L), boxsize=L).query_pairs(top["r_cut"], output_type="ndarray")
        d = xc[b][pr[:, 0]] - xc[b][pr[:, 1]]
        d -= L * np.rint(d / L)
        r2 = (d * d).sum(1)
        assert np.abs(r2 - top["r_cut"] ** 2).min() > 1e-9          # no decision rests on the last bits
        want += 2 * int((top["mol"][pr[:, 0]] != top["mol"][pr[:, 1]]).sum())
    assert c["pair_beads_in_cutoff"] == want


def test_staged_pair_kernel_mid_size():
    """5832 waters (17,496 atoms, 5 x 5 x 5 cells): the smallest water box the shared-memory staged pair
    kernel serves (>= 4 cells per dimension and the 27-cell neighbourhood fits); lists, forces,
    energy variant (observables) and 20 steps against the oracle."""
    import oracle as O
    top = W.water_box(5832)
    sysg, ref, x0, p0 = make_pair(top, 4, 2, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    c = sysg.counters()
    assert c["staged"] == 1 and c["overflow"] == 0
    ref.set_state(x0, p0, 0)
    otop, cent = _lists_check(sysg, top, x0)
    count, i, j = _pairs_from_gpu(sysg)
    for a in (0, 1, 7777, top["n_atoms"] - 1):
        assert np.array_equal(np.sort(j[i == a]), np.sort(O.neighbours_of(otop, cent, a)))
    assert (i < j).sum() * 2 == i.size
    G = sysg.forces().cpu().numpy()
    Gref = ref.forces()
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-10 * np.abs(oref).max()
    sysg.step(20)
    ref.step(20)
    x1, _, _ = sysg.get_state()
    xr, _ = ref.get_state()
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    sysg.check()


def test_orthorhombic_box_staged_kernel():
    """Non-cubic box (6 x 5 x 4 cells, different cell edges per dimension): cell indexing, the staged
    neighbourhood and the per-cell image shifts must not rely on a cubic box."""
    import oracle as O
    top = W.water_box(5832)
    scale = np.array([1.2, 1.0, 1.0 / 1.2])
    pos = top["positions"].reshape(-1, 3, 3)
    centre = pos[:, :1, :]
    top["positions"] = np.ascontiguousarray((centre * scale + (pos - centre)).reshape(-1, 3))
    top["box"] = top["box"] * scale
    sysg, ref, x0, p0 = make_pair(top, 2, 2, 0.25, "pile", sigma_bead=0.03)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1
    ref.set_state(x0, p0, 0)
    otop, cent = _lists_check(sysg, top, x0)
    assert tuple(sysg.neighbor_lists()[0].cpu().numpy()) == (6, 5, 4)
    count, i, j = _pairs_from_gpu(sysg)
    for a in (0, 5, 9000, top["n_atoms"] - 1):
        assert np.array_equal(np.sort(j[i == a]), np.sort(O.neighbours_of(otop, cent, a)))
    G = sysg.forces().cpu().numpy()
    Gref = ref.forces()
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    sysg.step(10)
    ref.step(10)
    x1, _, _ = sysg.get_state()
    assert np.abs(x1.cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()


@pytest.mark.parametrize("P,Pc", [(2, 1), (2, 2), (3, 3), (5, 3), (6, 3), (6, 6), (12, 5), (16, 16), (24, 12), (32, 1), (32, 32)])
def test_every_supported_bead_count(P, Pc):
    """All P the integrator is instantiated for, with odd / even / full / centroid-only contraction:
    forces at the start and positions after 10 steps (216 waters, one cell)."""
    import oracle as O
    top = W.water_box(216)
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.25, "pile", sigma_bead=0.03)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    G = sysg.forces().cpu().numpy()
    Gref = O.bead_forces(O.Topology(top), P, Pc, x0)
    assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
    sysg.step(10); ref.step(10)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()


def test_unsupported_arguments_are_rejected():
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    for P, Pc in [(7, 7), (8, 9), (8, 0), (0, 0)]:
        with pytest.raises(qhp.QhpError):
            qhp.System(top, P, Pc, 0.25e-3, T_K, "pile", gamma0=1.0, seed=1)
    with pytest.raises(qhp.QhpError):
        qhp.System(top, 8, 8, -1.0, T_K, "pile", gamma0=1.0, seed=1)
    sysg = qhp.System(top, 4, 2, 0.25e-3, T_K, "pile", gamma0=1.0, seed=1)
    with pytest.raises(qhp.QhpError):
        sysg.step(1)                                   # no state yet
    x0, p0 = W.initial_state(top, 4, T_K)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    sysg.step(0)                                       # zero steps is a no-op
    assert sysg.get_state()[2] == 0
