"""Pins for O3/O7: potential and forces (BASELINE.json configs[0] force field)."""
import math

import numpy as np
import pytest

import oracle as O
from helpers import mini_top
from workloads import water as W

COUL = 332.063713


@pytest.fixture(scope="module")
def box216():
    top = W.water_box(216)
    return top, O.Topology(top)


def test_total_force_is_zero_sum(box216):
    top, t = box216
    rng = np.random.default_rng(3)
    x = top["positions"] + 0.05 * rng.standard_normal(top["positions"].shape)
    _, Ff = O.force_fast(t, x)
    _, Fs = O.force_slow(t, x)
    assert np.abs(Ff.sum(0)).max() < 1e-10
    assert np.abs(Fs.sum(0)).max() < 1e-10


def test_finite_difference_single_replica(box216):
    top, t = box216
    rng = np.random.default_rng(4)
    x = top["positions"] + 0.05 * rng.standard_normal(top["positions"].shape)
    _, F = O.force_total(t, x, cells=False)
    h = 1e-4
    for (a, c) in [(0, 0), (1, 2), (2, 1), (100, 0), (301, 1), (647, 2)]:
        xp, xm = x.copy(), x.copy()
        xp[a, c] += h
        xm[a, c] -= h
        up, _ = O.force_total(t, xp, cells=False)
        um, _ = O.force_total(t, xm, cells=False)
        fd = -(up - um) / (2 * h)
        assert abs(fd - F[a, c]) < 1e-6 * max(1.0, abs(F[a, c])), (a, c, fd, F[a, c])


def test_finite_difference_contracted_ring_polymer(box216):
    # G_i = -d(P U_nu)/dx_i with U_nu of Eq. 20 (P = 4, P' = 2)
    top, t = box216
    P, Pc = 4, 2
    x, _ = W.initial_state(top, P, 300.0, sigma_bead=0.05)
    G = O.bead_forces(t, P, Pc, x, cells=False)

    def U(xb):
        _, e = O.nm_forces(t, P, Pc, O.beads_to_nm(xb), cells=False)
        return e[0] + e[1]
    h = 1e-4
    for (i, a, c) in [(0, 0, 0), (1, 4, 2), (3, 200, 1), (2, 647, 0)]:
        xp, xm = x.copy(), x.copy()
        xp[i, a, c] += h
        xm[i, a, c] -= h
        fd = -P * (U(xp) - U(xm)) / (2 * h)
        assert abs(fd - G[i, a, c]) < 2e-6 * max(1.0, abs(G[i, a, c])), (i, a, c, fd, G[i, a, c])


def test_bead_forces_two_routes_agree(box216):
    # O7 matrix form == NM->bead of the projected forces of O5
    top, t = box216
    P, Pc = 8, 4
    x, _ = W.initial_state(top, P, 300.0, sigma_bead=0.05)
    G = O.bead_forces(t, P, Pc, x, cells=False)
    f, _ = O.nm_forces(t, P, Pc, O.beads_to_nm(x), cells=False)
    G2 = O.nm_to_beads(f)
    assert np.abs(G - G2).max() < 1e-11 * np.abs(G).max()


def test_contraction_identity_forces(box216):
    # P' = P: forces equal the uncontracted per-bead forces -grad V(x_i)
    top, t = box216
    P = 4
    x, _ = W.initial_state(top, P, 300.0, sigma_bead=0.05)
    G = O.bead_forces(t, P, P, x, cells=False)
    for i in range(P):
        _, F = O.force_total(t, x[i], cells=False)
        assert np.abs(G[i] - F).max() < 1e-11 * np.abs(F).max()


def test_cells_equal_brute_force():
    top = W.water_box(729)
    t = O.Topology(top)
    assert int(top["box"][0] // 9.0) == 3
    rng = np.random.default_rng(5)
    x = top["positions"] + 0.05 * rng.standard_normal(top["positions"].shape)
    x[10] += np.array([2 * top["box"][0], -top["box"][1], 0.0])   # unwrapped coordinates are legal
    ub, Fb = O.force_slow(t, x, cells=False)
    uc, Fc = O.force_slow(t, x, cells=True)
    assert abs(ub - uc) < 1e-10 * abs(ub)
    assert np.abs(Fb - Fc).max() < 1e-11 * np.abs(Fb).max()


def test_dsf_continuous_at_cutoff_and_closed_form():
    al, rc = 0.2, 9.0
    for r in [2.0, 5.0, 8.999999]:
        top = mini_top([[0, 0, 0], [r, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0])
        t = O.Topology(top)
        u, F = O.force_slow(t, top["positions"])
        fs = math.erfc(al * rc) / rc ** 2 + 2 * al / math.sqrt(math.pi) * math.exp(-(al * rc) ** 2) / rc
        u_ref = -COUL * (math.erfc(al * r) / r - math.erfc(al * rc) / rc + fs * (r - rc))
        f_ref = -COUL * (math.erfc(al * r) / r ** 2
                         + 2 * al / math.sqrt(math.pi) * math.exp(-(al * r) ** 2) / r - fs)
        assert abs(u - u_ref) < 1e-12 * max(1, abs(u_ref))
        assert abs(F[0, 0] - f_ref * (-1.0)) < 1e-12 * max(1, abs(f_ref))   # F_0 = fmag * (x_0-x_1)/r, (x_0-x_1)/r = -1
        assert np.allclose(F[0], -F[1])
    assert abs(u) < 1e-9 and abs(F[0, 0]) < 1e-6                      # -> 0 continuously at r_c
    # opposite charges attract: atom 0 at the origin is pulled towards +x
    top = mini_top([[0, 0, 0], [3.0, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0])
    _, F = O.force_slow(O.Topology(top), top["positions"])
    assert F[0, 0] > 0 and F[1, 0] < 0
    # beyond the cutoff: nothing
    top = mini_top([[0, 0, 0], [9.0, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0])
    u, F = O.force_slow(O.Topology(top), top["positions"])
    assert u == 0 and np.all(F == 0)


def test_lj_minimum_and_mixing():
    eps, sig = 0.1554, 3.1655
    rmin = 2 ** (1 / 6) * sig
    top = mini_top([[0, 0, 0], [0, rmin, 0]], [0, 0], [0.0], [eps], [sig])
    u, F = O.force_slow(O.Topology(top), top["positions"])
    shift = 4 * eps * ((sig / 9.0) ** 12 - (sig / 9.0) ** 6)
    assert abs(u - (-eps - shift)) < 1e-13
    assert np.abs(F).max() < 1e-12
    # inside the minimum the pair repels
    top = mini_top([[0, 0, 0], [0, 3.0, 0]], [0, 0], [0.0], [eps], [sig])
    _, F = O.force_slow(O.Topology(top), top["positions"])
    assert F[0, 1] < 0 and F[1, 1] > 0
    # a type with eps = 0 has no LJ with anything (O-H, H-H of the water model)
    top = mini_top([[0, 0, 0], [0, 3.0, 0]], [0, 1], [0.0, 0.0], [eps, 0.0], [sig, 0.0])
    u, F = O.force_slow(O.Topology(top), top["positions"])
    assert u == 0 and np.all(F == 0)


def test_minimum_image_and_exclusions():
    L = 40.0
    top = mini_top([[1.0, 0, 0], [L - 2.0, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0], box=L)
    u1, F1 = O.force_slow(O.Topology(top), top["positions"])
    top2 = mini_top([[1.0, 0, 0], [-2.0, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0], box=L)
    u2, F2 = O.force_slow(O.Topology(top2), top2["positions"])
    assert abs(u1 - u2) < 1e-13 and np.abs(F1 - F2).max() < 1e-12
    top3 = mini_top([[1.0, 0, 0], [-2.0, 0, 0]], [0, 1], [1.0, -1.0], [0, 0], [0, 0], box=L, mols=[0, 0])
    u3, F3 = O.force_slow(O.Topology(top3), top3["positions"])
    assert u3 == 0 and np.all(F3 == 0)          # intramolecular pairs excluded


def test_bond_angle_equilibrium_and_values():
    top = W.water_box(216)
    t = O.Topology(top)
    u, F = O.force_fast(t, top["positions"])     # generated at r0, theta0
    assert abs(u) < 1e-20 and np.abs(F).max() < 1e-9
    # stretch one O-H bond by 0.1 A along the bond: U = 1/2 k 0.01 + small angle term = 0
    x = top["positions"].copy()
    d = x[1] - x[0]
    x[1] += 0.1 * d / np.linalg.norm(d)
    u, F = O.force_fast(t, x)
    assert abs(u - 0.5 * 1059.162 * 0.01) < 1e-10
    assert abs(np.dot(F[1], d / np.linalg.norm(d)) + 1059.162 * 0.1) < 1e-9
    # open the angle by 0.05 rad keeping bond lengths
    x = top["positions"].copy()
    a, b = x[1] - x[0], x[2] - x[0]
    n = np.cross(a, b)
    n /= np.linalg.norm(n)
    th = 0.05
    b2 = b * np.cos(th) + np.cross(n, b) * np.sin(th)
    x[2] = x[0] + b2
    u, _ = O.force_fast(t, x)
    assert abs(u - 0.5 * 75.90 * th ** 2) < 1e-10


def test_ragged_molecules_four_types_finite_difference_and_cells():
    """workloads.water.ionic_water_box: molecules of 1, 2 and 3 atoms, four types (ions with LJ + charge):
    forces are minus the gradient of the energy, sum to zero, and the cell walk equals the double loop."""
    top = W.ionic_water_box(729)
    t = O.Topology(top)
    sizes = np.bincount(top["mol"])
    assert set(sizes) == {1, 2, 3}
    rng = np.random.default_rng(6)
    x = top["positions"] + 0.05 * rng.standard_normal(top["positions"].shape)
    ub, Fb = O.force_slow(t, x, cells=False)
    uc, Fc = O.force_slow(t, x, cells=True)
    assert abs(ub - uc) < 1e-10 * abs(ub) and np.abs(Fb - Fc).max() < 1e-11 * np.abs(Fb).max()
    _, F = O.force_total(t, x, cells=False)
    assert np.abs(F.sum(0)).max() < 1e-9
    first = np.concatenate([[0], np.cumsum(sizes)[:-1]])
    picks = [first[sizes == 1][0], first[sizes == 1][1], first[sizes == 2][0], first[sizes == 2][0] + 1, first[sizes == 3][5] + 2]
    h = 1e-4
    for a, c in zip(picks, (0, 1, 2, 0, 1)):
        xp, xm = x.copy(), x.copy()
        xp[a, c] += h
        xm[a, c] -= h
        up, _ = O.force_total(t, xp, cells=False)
        um, _ = O.force_total(t, xm, cells=False)
        fd = -(up - um) / (2 * h)
        assert abs(fd - F[a, c]) < 1e-6 * max(1.0, abs(F[a, c])), (a, c, fd, F[a, c])
