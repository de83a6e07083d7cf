"""Pins for O4: neighbour objects on centroids."""
import numpy as np

import oracle as O
from workloads import water as W


def _numpy_cells(top, c):
    rl = top["r_cut"] + top["skin"]
    nc = np.maximum(1, np.floor(top["box"] / rl)).astype(np.int64)
    q = []
    for d in range(3):
        s = c[:, d] * (1.0 / top["box"][d])
        s = s - np.floor(s)
        q.append(np.minimum((s * float(nc[d])).astype(np.int64), nc[d] - 1))
    return nc, (q[0] * nc[1] + q[1]) * nc[2] + q[2]


def test_cell_objects():
    top = W.water_box(4096)
    t = O.Topology(top)
    rng = np.random.default_rng(6)
    c = top["positions"] + 0.3 * rng.standard_normal(top["positions"].shape)
    c[5] -= top["box"]                      # atoms outside the primary cell are legal
    nc, cell_of, order, cell_start = O.cells(t, c)
    nc_ref, cell_ref = _numpy_cells(top, c)
    assert np.array_equal(nc, nc_ref) and tuple(nc) == (4, 4, 4)
    assert np.array_equal(cell_of, cell_ref)
    assert np.array_equal(np.sort(order), np.arange(t.n_atoms))          # permutation
    assert np.array_equal(order, np.argsort(cell_ref, kind="stable"))    # stable: ties by index
    assert cell_start[0] == 0 and cell_start[-1] == t.n_atoms and np.all(np.diff(cell_start) >= 0)
    assert np.all(np.diff(cell_of[order]) >= 0)
    assert np.array_equal(cell_start, np.searchsorted(cell_ref[order], np.arange(nc.prod() + 1)))


def test_degenerate_small_box_single_cell():
    top = W.water_box(216)                  # L = 18.64 < 2 r_list: one cell (G9)
    t = O.Topology(top)
    nc, cell_of, order, cell_start = O.cells(t, top["positions"])
    assert tuple(nc) == (1, 1, 1) and np.all(cell_of == 0)
    assert np.array_equal(order, np.arange(648)) and list(cell_start) == [0, 648]


def test_pair_set_against_numpy_distances():
    top = W.water_box(216)
    t = O.Topology(top)
    rng = np.random.default_rng(7)
    c = top["positions"] + 0.2 * rng.standard_normal(top["positions"].shape)
    pairs = O.pairs_brute(t, c)
    assert np.all(pairs[:, 0] < pairs[:, 1])
    key = pairs[:, 0].astype(np.int64) * t.n_atoms + pairs[:, 1]
    assert np.all(np.diff(key) > 0)                                       # sorted, unique
    d = c[:, None, :] - c[None, :, :]
    d -= top["box"] * np.rint(d / top["box"])
    r = np.sqrt((d ** 2).sum(-1))
    iu, ju = np.triu_indices(t.n_atoms, 1)
    other = top["mol"][iu] != top["mol"][ju]
    rl = top["r_cut"] + top["skin"]
    inside = set(map(tuple, np.stack([iu, ju], 1)[other & (r[iu, ju] < rl - 1e-9)]))
    maybe = set(map(tuple, np.stack([iu, ju], 1)[other & (r[iu, ju] < rl + 1e-9)]))
    got = set(map(tuple, pairs))
    assert inside <= got <= maybe
    # the per-atom view used to sample large boxes is the same set
    for i in (0, 17, 647):
        nb = O.neighbours_of(t, c, i)
        ref = sorted([b for (a, b) in got if a == i] + [a for (a, b) in got if b == i])
        assert list(nb) == ref
