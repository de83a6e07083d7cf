"""Pins of the oracle's RATIO adaptation (Eq. 24-26)."""
import numpy as np

import oracle as O
from workloads import water as W

ACC = O.ACC


def _top(n_types=2):
    top = W.water_box(8)
    return top, O.Topology(top)


def test_window_recursion_has_its_geometric_closed_form():
    """Eq. 26 with constant input C1 after an initial average C0: <C>^(k) = C1 + (C0 - C1) w^k; and a
    constant input is a fixed point for any tau."""
    top, t = _top()
    n_seg, dt, g0 = 8, 0.5e-3, 20.0
    nf = n_seg + 1
    rng = np.random.default_rng(1)
    C0v, C0f = rng.uniform(1, 2, (2, nf)), rng.uniform(1, 2, (2, nf))
    C1v, C1f = rng.uniform(1, 2, (2, nf)), rng.uniform(1, 2, (2, nf))
    tau = np.array([0.01, 0.003])
    g = np.full((2, nf), g0)
    g, av, af = O.qtb_adapt_ratio(t, n_seg, g0, 0.01, dt, tau, True, C0v, C0f, np.zeros((2, nf)), np.zeros((2, nf)), g)
    assert np.array_equal(av, C0v) and np.array_equal(af, C0f)           # reading G24: first segment initialises
    for k in range(1, 6):
        g, av, af = O.qtb_adapt_ratio(t, n_seg, g0, 0.01, dt, tau, False, C1v, C1f, av, af, g)
        w = np.exp(-n_seg * dt / tau)[:, None]
        assert np.allclose(av, C1v + (C0v - C1v) * w ** k, rtol=1e-13)
        assert np.allclose(af, C1f + (C0f - C1f) * w ** k, rtol=1e-13)
    g2, av2, af2 = O.qtb_adapt_ratio(t, n_seg, g0, 0.01, dt, tau, False, av, af, av, af, g)
    assert np.allclose(av2, av, rtol=1e-15) and np.allclose(af2, af, rtol=1e-15)


def test_eq24_zero_fdt_deviation_is_the_fixed_point():
    """Eq. 24: Delta_FDT = 0 under the SIMPLE definition (qo_qtb_adapt leaves gamma unchanged) <=> gamma is
    what RATIO returns.  Spectra are built so that m gamma* C_vv = Re C_vF for a chosen gamma*."""
    top, t = _top()
    n_seg, dt, g0 = 16, 0.5e-3, 20.0
    nf = n_seg + 1
    rng = np.random.default_rng(2)
    gstar = rng.uniform(5.0, 60.0, (2, nf))
    Cvv = rng.uniform(0.5, 3.0, (2, nf))
    CvF = (t.mass[:, None] / ACC) * gstar * Cvv
    g_simple = O.qtb_adapt(t, n_seg, g0, 0.5, 0.01, Cvv, CvF, gstar)
    assert np.abs(g_simple - gstar).max() < 1e-10 * g0                  # Delta = 0: SIMPLE does not move
    start = np.full((2, nf), g0)
    g_ratio, _, _ = O.qtb_adapt_ratio(t, n_seg, g0, 0.01, dt, np.array([0.1, 0.1]), True, Cvv, CvF,
                                      np.zeros((2, nf)), np.zeros((2, nf)), start)
    assert np.allclose(g_ratio, gstar, rtol=1e-13)


def test_lower_bound_untouched_types_and_empty_bins():
    top, t = _top()
    n_seg, dt, g0 = 8, 0.5e-3, 20.0
    nf = n_seg + 1
    Cvv = np.ones((2, nf)); CvF = np.full((2, nf), -1.0)               # negative ratio -> clamped
    Cvv[0, 3] = 0.0                                                     # empty bin keeps its gamma
    g = np.full((2, nf), 7.0)
    out, _, _ = O.qtb_adapt_ratio(t, n_seg, g0, 0.01, dt, np.array([0.05, -1.0]), True, Cvv, CvF,
                                  np.zeros((2, nf)), np.zeros((2, nf)), g)
    assert np.all(out[1] == 7.0)                                        # tau <= 0: not a RATIO type
    assert out[0, 3] == 7.0
    assert np.all(np.delete(out[0], 3) == 0.01 * g0)


def test_free_particle_ratio_is_frequency_independent():
    """G14: for O-only dynamics Re C_vF / (m C_vv) = (1 - a)/b * 418.4 = gamma0 (1 - (gamma0 dt)^2/24 + ...),
    independent of frequency; RATIO with a long window recovers it from the oracle's own segments."""
    n_atoms, n_seg, dt, T_K, g0 = 120, 128, 0.0005, 300.0, 400.0
    top = W.oscillator_box(n_atoms, 1.008, 0.0)
    t = O.Topology(top)
    sim = O.Adqtb(t, dt, T_K, g0, 3, n_seg, a_gamma=0.0, cells=False, ratio_tau=[1.0e3])
    x, p = W.initial_state(top, 1, T_K)
    sim.set_state(x, p)
    sim.step(n_seg)                       # the first segment starts from the initial state: leave it out
    sim.ratio_started = False
    gam0 = sim.gamma.copy()
    sim.gamma[:] = g0                     # keep the noise at gamma0 (no feedback): we test the estimator
    for _ in range(8):
        sim.step(n_seg)
        est = sim.gamma.copy()
        sim.gamma[:] = g0
    a = np.exp(-g0 * dt); b = np.sqrt((1 - a * a) * dt / (2 * g0))
    expect = (1 - a) / b                  # in 1/ps: b carries the 1/sqrt(gamma0) that makes it a rate
    sl = slice(5, n_seg // 2)             # the mid-kick velocity has vanishing gain towards Nyquist (G14): noisy there
    assert abs(est[0, sl].mean() / expect - 1) < 0.05
    assert est[0, sl].std() / expect < 0.1
