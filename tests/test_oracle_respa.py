"""Pins of the oracle's BAOAB-RESPA stepper (Eq. 19).
None of them re-uses the stepper's own arithmetic: they are limits that reduce to the single-step
integrator, symmetries of the splitting, its order, and a conserved quantity."""
import numpy as np
import pytest

import oracle as O
from workloads import water as W

T_K = W.T_KELVIN


def _state(n_mol=27, P=4, box=20.0, sigma=0.03):
    top = W.water_box(n_mol)
    top["box"] = np.array([box] * 3)
    x0, p0 = W.initial_state(top, P, T_K, sigma_bead=sigma)
    return top, O.Topology(top), x0, p0


def test_n_alt_1_is_plain_baoab():
    top, otop, x0, p0 = _state()
    a = O.Rpmd(otop, 4, 2, 0.25e-3, T_K, "pile", 1.0, 7)
    b = O.RpmdRespa(otop, 4, 2, 0.25e-3, T_K, "pile", 1.0, 7, n_alt=1)
    a.set_state(x0, p0, 3); b.set_state(x0, p0, 3)
    a.step(12); b.step(12)
    assert np.abs(a.Q - b.Q).max() < 1e-13 and np.abs(a.Pm - b.Pm).max() < 1e-11 * np.abs(a.Pm).max()


def test_without_slow_potential_respa_is_plain_baoab():
    """V_s = 0 (no charges, no LJ): the Bs blocks do nothing, so n_alt inner steps == n_alt plain steps."""
    top, _, x0, p0 = _state()
    top["charge"] = np.zeros(2); top["lj_eps"] = np.zeros(2)
    otop = O.Topology(top)
    a = O.Rpmd(otop, 4, 4, 0.25e-3, T_K, "pile", 2.0, 11)
    b = O.RpmdRespa(otop, 4, 4, 0.25e-3, T_K, "pile", 2.0, 11, n_alt=4)
    a.set_state(x0, p0, 0); b.set_state(x0, p0, 0)
    a.step(8); b.step(8)
    assert np.abs(a.Q - b.Q).max() < 1e-13


def test_time_reversal_without_thermostat():
    top, otop, x0, p0 = _state()
    r = O.RpmdRespa(otop, 4, 2, 0.25e-3, T_K, "none", 1.0, 0, n_alt=3)
    r.set_state(x0, p0, 0)
    Q0 = r.Q.copy()
    r.step(12)
    r.Pm *= -1.0
    r.step(12)
    assert np.abs(r.Q - Q0).max() < 1e-11


def test_second_order_convergence_to_single_step_trajectory():
    """|RESPA(n_alt) - BAOAB| after a fixed time scales as dt^2 (symmetric Trotter splitting)."""
    top, otop, x0, p0 = _state()
    errs = []
    for dt, n in ((0.4e-3, 8), (0.2e-3, 16)):
        a = O.Rpmd(otop, 4, 2, dt, T_K, "none", 1.0, 0)
        b = O.RpmdRespa(otop, 4, 2, dt, T_K, "none", 1.0, 0, n_alt=4)
        a.set_state(x0, p0, 0); b.set_state(x0, p0, 0)
        a.step(n); b.step(n)
        errs.append(np.abs(a.Q - b.Q).max())
    assert errs[0] > 0 and 3.0 < errs[0] / errs[1] < 5.5


def test_ring_polymer_hamiltonian_is_conserved():
    """No thermostat: H = sum Pm^2/2m + sum m w_n^2 Q_n^2/2 + U (Eq. 1-4 with the scaled modes; U of
    Eq. 20) drifts only by the O(dt^2) splitting error, and a wrong slow kick would break it."""
    top, otop, x0, p0 = _state()
    P, Pc = 4, 2
    m = np.repeat(otop.mass[otop.type], 3)[None, :]
    om = O.nm_freq(P, T_K)[:, None]

    def H(r):
        obs = O.observables(otop, P, Pc, T_K, r.Q, r.Pm, r.uc)
        spring = 0.5 * (m * om ** 2 * r.Q.reshape(P, -1) ** 2).sum() / O.ACC
        return obs[2] + spring + obs[1]

    drift = []
    for dt, n in ((0.2e-3, 40), (0.1e-3, 80)):
        r = O.RpmdRespa(otop, P, Pc, dt, T_K, "none", 1.0, 0, n_alt=4)
        r.set_state(x0, p0, 0)
        h0 = H(r)
        hs = []
        for _ in range(n // 4):
            r.step(4)
            hs.append(H(r))
        drift.append(np.abs(np.array(hs) - h0).max())
    scale = abs(h0)
    assert drift[0] < 1e-3 * scale
    assert 2.5 < drift[0] / drift[1] < 6.0
