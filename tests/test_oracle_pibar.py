"""Pins of the oracle's PI-BAR estimator (Eq. 27-28): an exact
special case, Bennett's implicit equation solved by an independent root finder, the A <-> B antisymmetry,
and closed-form free-energy differences of classical and finite-P ring-polymer harmonic oscillators
sampled exactly (no MD involved)."""
import numpy as np
from scipy.optimize import brentq

import oracle as O

KB = 1.987204258640832e-3
HBAR = 1.5178728306651436e-2
ACC = 418.4
BETA = 1.0 / (KB * 300.0)


def test_constant_shift_is_exact_in_one_iteration():
    rng = np.random.default_rng(0)
    for c in (-3.0, 0.0, 0.7):
        dF, it = O.pibar(np.full(50, c), np.full(80, -c), BETA)
        assert abs(dF - c) < 1e-13 and it <= 2
    # ... also when added on top of a fluctuating difference: dF(U_B + c) = dF(U_B) + c
    wA, wB = rng.normal(1.0, 0.5, 300), rng.normal(-0.4, 0.6, 200)
    d0, _ = O.pibar(wA, wB, BETA)
    d1, _ = O.pibar(wA + 0.9, wB - 0.9, BETA)
    assert abs(d1 - d0 - 0.9) < 1e-11


def test_fixed_point_solves_bennetts_implicit_equation():
    rng = np.random.default_rng(1)
    wA, wB = rng.normal(0.8, 0.7, 4000), rng.normal(-0.3, 0.5, 2500)
    f = lambda x: 1.0 / (1.0 + np.exp(BETA * x))
    g = lambda Cc: f(wA - Cc).sum() - f(wB + Cc).sum()      # n_A <f>_A = n_B <f>_B at the solution
    Cs = brentq(g, -10.0, 10.0, xtol=1e-14, rtol=1e-14)
    ref = Cs - np.log(wB.size / wA.size) / BETA
    dF, it = O.pibar(wA, wB, BETA)
    assert abs(dF - ref) < 1e-10 and 1 < it < 1000
    # antisymmetry under A <-> B
    dR, _ = O.pibar(wB, wA, BETA)
    assert abs(dR + dF) < 1e-10


def test_classical_harmonic_oscillators():
    """V = k x^2 / 2: Z ~ k^-1/2 per dimension, dF_AB = (1/beta) ln(Z_A/Z_B) = (1/2 beta) ln(k_B/k_A)."""
    rng = np.random.default_rng(2)
    kA, kB, n = 30.0, 55.0, 200_000
    xA = rng.normal(0.0, 1.0 / np.sqrt(BETA * kA), n)
    xB = rng.normal(0.0, 1.0 / np.sqrt(BETA * kB), n)
    wA = 0.5 * (kB - kA) * xA ** 2
    wB = 0.5 * (kA - kB) * xB ** 2
    dF, _ = O.pibar(wA, wB, BETA)
    ref = 0.5 / BETA * np.log(kB / kA)
    assert abs(dF - ref) < 5 * 0.6 / np.sqrt(n) / BETA      # a few standard errors of a BAR estimate (kT units)
    assert dF > 0                                            # the stiffer state B has the smaller Z


def test_ring_polymer_harmonic_oscillators_finite_P():
    """Path-integral version: U_nu = (1/P) sum_i m w^2 x_i^2 / 2 = (m w^2 / 2) sum_n Q_n^2 in scaled normal
    modes, each mode Gaussian with variance 1 / (beta m (w^2 + w_n^2)), so
    Z_nu ~ prod_n (w^2 + w_n^2)^-1/2 and dF = (1/2 beta) sum_n ln[(w_B^2 + w_n^2) / (w_A^2 + w_n^2)]."""
    rng = np.random.default_rng(3)
    P, m, n = 8, 1.008 / ACC, 200_000                       # mass in kcal/mol ps^2 / A^2
    wn = O.nm_freq(P, 300.0)
    wA, wB = 500.0, 700.0                                    # rad/ps: beta hbar w ~ 12.7 and 17.8, strongly quantum
    QA = rng.standard_normal((n, P)) / np.sqrt(BETA * m * (wA ** 2 + wn ** 2))
    QB = rng.standard_normal((n, P)) / np.sqrt(BETA * m * (wB ** 2 + wn ** 2))
    dU_A = 0.5 * m * (wB ** 2 - wA ** 2) * (QA ** 2).sum(axis=1)       # U_B - U_A on samples of A
    dU_B = 0.5 * m * (wA ** 2 - wB ** 2) * (QB ** 2).sum(axis=1)
    dF, _ = O.pibar(dU_A, dU_B, BETA)
    ref = 0.5 / BETA * np.log((wB ** 2 + wn ** 2) / (wA ** 2 + wn ** 2)).sum()
    assert abs(dF - ref) < 5 * 1.0 / np.sqrt(n) / BETA
    # the classical formula would be off by much more than the error bar: the pin sees the beads
    assert abs(ref - 1.0 / BETA * np.log(wB / wA)) > 50 / np.sqrt(n) / BETA
