"""Pins of the oracle's BCOCB stepper (reading G25).
The half-step C is pinned as THE principal square root of the Cayley transform of the free ring-polymer
generator, computed here from its definition with a linear solve and scipy's sqrtm (neither uses the
oracle's closed form), then through invariants, its order against the exact rotation, and limits."""
import numpy as np
import scipy.linalg as sla

import oracle as O
from workloads import water as W

T_K = W.T_KELVIN
M_H = 1.008


def _free(n=2, mass=M_H):
    return O.Topology(W.oscillator_box(n, mass, 0.0))


def _mode_map(sim_factory, P, n_steps=1):
    """2x2 map (q, p) -> (q', p') of every mode, read off two basis states of atom 0 / x."""
    cols = []
    for q0, p0 in ((1.0, 0.0), (0.0, 1.0)):
        sim = sim_factory()
        x = np.zeros((P, 2, 3))
        sim.set_state(x, x.copy())
        sim.Q[:, 0, 0] = q0
        sim.Pm[:, 0, 0] = p0
        sim.f[:] = 0.0
        sim.step(n_steps)
        cols.append(np.stack([sim.Q[:, 0, 0], sim.Pm[:, 0, 0]], axis=0))     # [2][P]
    return np.stack(cols, axis=-1).transpose(1, 0, 2)                        # [P][2][2]


def _cayley(w, dt, m=M_H):
    A = np.array([[0.0, 1.0 / m], [-m * w * w, 0.0]])
    I = np.eye(2)
    return np.linalg.solve(I - 0.5 * dt * A, I + 0.5 * dt * A)


def test_one_free_step_is_the_cayley_transform():
    P = 8
    w = O.nm_freq(P, T_K)
    for dt in (0.25e-3, 2e-3, 50e-3):                    # w_max dt = 0.16, 1.3, 31
        M = _mode_map(lambda: O.Rpmd(_free(), P, P, dt, T_K, "none", 0.0, 1, cells=False, a_block="cayley"), P)
        for n in range(P):
            ref = _cayley(w[n], dt)
            assert np.abs(M[n] - ref).max() < 1e-13 * np.abs(ref).max(), (n, dt)
            assert abs(np.linalg.det(M[n]) - 1.0) < 1e-13


def test_half_step_is_the_principal_square_root():
    """With the O block between the halves the deterministic part of a step is C diag(1, c1) C, which
    separates C from the other square roots of cay(dt A); the noise cancels in the difference of two
    trajectories with the same seed."""
    P, dt, g0 = 4, 1e-3, 3.0
    w = O.nm_freq(P, T_K)
    top = _free()
    def run(q0, p0):
        sim = O.Rpmd(top, P, P, dt, T_K, "pile", g0, 99, cells=False, a_block="cayley")
        x = np.zeros((P, 2, 3))
        sim.set_state(x, x.copy(), 5)
        sim.Q[:, 0, 0] = q0; sim.Pm[:, 0, 0] = p0
        sim.f[:] = 0.0
        sim.step(1)
        return np.stack([sim.Q[:, 0, 0], sim.Pm[:, 0, 0]])
    base = run(0.0, 0.0)
    cols = [run(1.0, 0.0) - base, run(0.0, 1.0) - base]
    for n in range(P):
        M = np.array([[cols[0][0, n], cols[1][0, n]], [cols[0][1, n], cols[1][1, n]]])
        S = np.real(sla.sqrtm(_cayley(w[n], dt)))
        g = g0 if n == 0 else max(g0, w[n])
        ref = S @ np.diag([1.0, np.exp(-g * dt)]) @ S
        assert np.abs(M - ref).max() < 1e-12 * np.abs(ref).max(), n


def test_mode_energies_conserved_and_bounded_for_any_timestep():
    P = 8
    w = O.nm_freq(P, T_K)
    rng = np.random.default_rng(3)
    for dt in (0.5e-3, 20e-3, 1.0):                      # up to w_max dt ~ 600: still a rotation
        sim = O.Rpmd(_free(4), P, P, dt, T_K, "none", 0.0, 1, cells=False, a_block="cayley")
        sim.set_state(rng.standard_normal((P, 4, 3)) * 0.1, rng.standard_normal((P, 4, 3)) * 3.0)
        E0 = sim.Pm[1:] ** 2 / (2 * M_H) + 0.5 * M_H * (w[1:] ** 2)[:, None, None] * sim.Q[1:] ** 2
        sim.step(1000)
        E1 = sim.Pm[1:] ** 2 / (2 * M_H) + 0.5 * M_H * (w[1:] ** 2)[:, None, None] * sim.Q[1:] ** 2
        assert np.abs(E1 - E0).max() < 1e-11 * np.abs(E0).max()


def test_rotation_angle_and_third_order_agreement_with_the_exact_block():
    P = 4
    w = O.nm_freq(P, T_K)
    errs = []
    for dt in (0.4e-3, 0.2e-3):
        C = _mode_map(lambda: O.Rpmd(_free(), P, P, dt, T_K, "none", 0.0, 1, cells=False, a_block="cayley"), P)
        E = _mode_map(lambda: O.Rpmd(_free(), P, P, dt, T_K, "none", 0.0, 1, cells=False), P)
        for n in range(1, P):
            assert abs(C[n][0, 0] - np.cos(2 * np.arctan(0.5 * w[n] * dt))) < 1e-14
            assert abs(E[n][0, 0] - np.cos(w[n] * dt)) < 1e-14
        assert np.array_equal(C[0], E[0])                # centroid: the same translation
        errs.append(np.abs(C[P // 2][0, 1] - E[P // 2][0, 1]))
    assert 7.5 < errs[0] / errs[1] < 8.5                 # local error (w dt)^3 / 12


def test_P1_is_unchanged_and_water_is_reversible_and_second_order():
    top = W.water_box(27)
    top["box"] = np.array([20.0] * 3)
    ot = O.Topology(top)
    x0, p0 = W.initial_state(top, 1, T_K)
    a = O.Rpmd(ot, 1, 1, 0.5e-3, T_K, "pile", 1.0, 5)
    b = O.Rpmd(ot, 1, 1, 0.5e-3, T_K, "pile", 1.0, 5, a_block="cayley")
    a.set_state(x0, p0); b.set_state(x0, p0)
    a.step(5); b.step(5)
    assert np.array_equal(a.Q, b.Q) and np.array_equal(a.Pm, b.Pm)

    x0, p0 = W.initial_state(top, 4, T_K, sigma_bead=0.03)
    r = O.Rpmd(ot, 4, 2, 0.25e-3, T_K, "none", 1.0, 0, a_block="cayley")
    r.set_state(x0, p0)
    Q0 = r.Q.copy()
    r.step(12); r.Pm *= -1.0; r.step(12)
    assert np.abs(r.Q - Q0).max() < 1e-11

    errs = []
    for dt, n in ((0.4e-3, 8), (0.2e-3, 16)):
        e = O.Rpmd(ot, 4, 2, dt, T_K, "none", 1.0, 0)
        c = O.Rpmd(ot, 4, 2, dt, T_K, "none", 1.0, 0, a_block="cayley")
        e.set_state(x0, p0); c.set_state(x0, p0)
        e.step(n); c.step(n)
        errs.append(np.abs(e.Q - c.Q).max())
    assert errs[0] > 1e-9 and 3.5 < errs[0] / errs[1] < 4.5


def test_respa_with_n_alt_1_is_bcocb():
    top = W.water_box(27)
    top["box"] = np.array([20.0] * 3)
    ot = O.Topology(top)
    x0, p0 = W.initial_state(top, 4, T_K, sigma_bead=0.03)
    a = O.Rpmd(ot, 4, 2, 0.25e-3, T_K, "pile", 1.0, 7, a_block="cayley")
    b = O.RpmdRespa(ot, 4, 2, 0.25e-3, T_K, "pile", 1.0, 7, n_alt=1, a_block="cayley")
    e = O.RpmdRespa(ot, 4, 2, 0.25e-3, T_K, "pile", 1.0, 7, n_alt=1)
    for s in (a, b, e):
        s.set_state(x0, p0, 3); s.step(12)
    assert np.abs(a.Q - b.Q).max() < 1e-13 and np.abs(a.Pm - b.Pm).max() < 1e-11 * np.abs(a.Pm).max()
    assert np.abs(a.Q - e.Q).max() > 1e-9                  # and it is not the exact-A stepper
