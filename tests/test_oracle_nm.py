"""Pins for O1/O2: normal-mode matrix, frequencies, contraction (Eq. 2, 4, 10-11, 20)."""
import numpy as np
import pytest

import oracle as O
from workloads import water as W
from helpers import read_golden

KB, HBAR, ACC = 1.987204258640832e-3, 1.5178728306651436e-2, 418.4


def cyclic(P):
    A = np.zeros((P, P))
    for i in range(P):
        A[i, i] += 2
        A[i, (i + 1) % P] -= 1
        A[i, (i - 1) % P] -= 1
    return A


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5, 8, 16, 32, 64])
def test_T_orthogonal_and_diagonalises_eq2(P):
    T = O.nm_matrix(P)
    assert np.abs(T.T @ T - np.eye(P)).max() < 1e-14
    if P == 1:
        return
    D = T.T @ cyclic(P) @ T
    k = np.array([0] + [(n + 1) // 2 for n in range(1, P)])
    if P % 2 == 0:
        k[P - 1] = P // 2
    lam = 4 * np.sin(np.pi * k / P) ** 2
    assert np.abs(D - np.diag(lam)).max() < 1e-14 * 4 * 4
    assert np.all(np.diff(lam) > -1e-15)            # ascending
    # frequencies are the square roots of the eigenvalues of Eq. 2 (prefactor P/(beta hbar))
    w = O.nm_freq(P, 300.0)
    assert np.allclose(w, P * KB * 300.0 / HBAR * np.sqrt(lam), rtol=1e-14, atol=1e-12)


def test_P2_special_case():
    # for P = 2 the two -1 of Eq. 2 coincide: [[2,-2],[-2,2]]
    assert np.array_equal(cyclic(2), np.array([[2., -2.], [-2., 2.]]))
    T = O.nm_matrix(2)
    assert np.allclose(T, np.array([[1, 1], [1, -1]]) / np.sqrt(2), atol=1e-16)


def test_centroid_and_eq4():
    rng = np.random.default_rng(0)
    P = 8
    x = rng.standard_normal((P, 5, 3))
    Q = O.beads_to_nm(x)
    assert np.allclose(Q[0], x.mean(0), atol=1e-15)            # Q_0 = centroid
    T = O.nm_matrix(P)
    x4 = Q[0][None] + np.sqrt(P) * np.einsum("in,n...->i...", T[:, 1:], Q[1:])   # Eq. 4 literally
    assert np.allclose(x4, x, atol=1e-14)
    assert np.allclose(O.nm_to_beads(Q), x, rtol=1e-13, atol=1e-14)


def test_force_projection_eq10_11_and_parseval():
    rng = np.random.default_rng(1)
    P = 16
    F = rng.standard_normal((P, 7, 3))
    f = O.beads_to_nm(F)
    T = O.nm_matrix(P)
    assert np.allclose(f[0], F.sum(0) / P, atol=1e-14)                      # Eq. 10
    assert np.allclose(f[3], np.einsum("i,i...->...", T[:, 3], F) / np.sqrt(P), atol=1e-14)   # Eq. 11
    assert abs((F ** 2).sum() - P * (f ** 2).sum()) < 1e-13 * (F ** 2).sum()


@pytest.mark.parametrize("P,Pc", [(8, 8), (32, 32), (8, 1), (32, 4), (32, 5), (16, 2), (6, 3)])
def test_contraction_matrix(P, Pc):
    Cm = O.contraction_matrix(P, Pc)
    assert np.abs(Cm.sum(1) - 1).max() < 1e-14                  # rows sum to 1
    if Pc == P:
        assert np.abs(Cm - np.eye(P)).max() < 1e-14             # full polymer recovered (l.180)
    if Pc == 1:
        assert np.abs(Cm - 1.0 / P).max() < 1e-15               # centroid (l.180)
    # matrix form of O2 written out here independently
    T, Tc = O.nm_matrix(P), O.nm_matrix(Pc)
    ref = np.sqrt(Pc / P) * Tc @ T[:, :Pc].T
    assert np.abs(Cm - ref).max() < 1e-14


def test_contracted_beads_of_smooth_ring_polymer():
    # a ring polymer that only contains modes k <= 1 is reproduced exactly on P' >= 3 beads:
    # x(tau) = c + a cos(2 pi tau) + b sin(2 pi tau) sampled at tau = j/P'
    P, Pc = 32, 4
    c, a, b = 0.3, 0.2, -0.1
    x = np.array([c + a * np.cos(2 * np.pi * i / P) + b * np.sin(2 * np.pi * i / P) for i in range(P)])
    xc = O.contract(O.beads_to_nm(x.reshape(P, 1)), Pc)[:, 0]
    ref = np.array([c + a * np.cos(2 * np.pi * j / Pc) + b * np.sin(2 * np.pi * j / Pc) for j in range(Pc)])
    assert np.allclose(xc, ref, atol=1e-14)


def test_expand_force_is_chain_rule_of_contraction():
    rng = np.random.default_rng(2)
    P, Pc = 16, 4
    Fc = rng.standard_normal((Pc, 3, 3))
    fs = O.expand_force(Fc, P)
    assert np.all(fs[Pc:] == 0)
    # bead-space: G^s_i = (P/Pc) sum_j C[j][i] Fc_j ; f^s_n = (1/sqrt P) sum_i T[i][n] G^s_i
    Cm = O.contraction_matrix(P, Pc)
    G = P / Pc * np.einsum("ji,j...->i...", Cm, Fc)
    assert np.allclose(O.beads_to_nm(G), fs, atol=1e-13)


def test_harmonic_closed_form_values():
    m, w, T_K = 1.008, 565.10, 300.0
    for P_s, q2_s in read_golden("harmonic_q2.txt"):
        P, q2 = int(P_s), float(q2_s)
        if P == 0:
            val = HBAR * ACC / (2 * m * w) / np.tanh(HBAR * w / (2 * KB * T_K))
        else:
            wk = O.nm_freq(P, T_K)
            val = KB * T_K * ACC / m * np.sum(1.0 / (w ** 2 + wk ** 2))
        assert abs(val - q2) < 2e-5 * q2, (P, val, q2)


def test_trigonometric_contraction_variant_equals_fourier_resampling():
    """Variant 1 of reading G3: the contracted beads are the band-limited (Fourier) interpolant of the P
    bead positions evaluated at P' equidistant points -- scipy.signal.resample computes exactly that,
    independently; the literal Eq. 20 differs from it on the Nyquist mode of an even P' only."""
    import scipy.signal as ss
    rng = np.random.default_rng(11)
    try:
        for P, Pc in [(32, 4), (8, 4), (16, 2), (12, 6), (32, 5), (8, 3), (8, 8), (6, 1)]:
            x = rng.standard_normal((P, 7))
            Q = O.beads_to_nm(x)
            ref = ss.resample(x, Pc, axis=0)
            O.set_contraction_variant(1)
            xv = O.contract(Q, Pc)
            Cv = O.contraction_matrix(P, Pc)
            O.set_contraction_variant(0)
            xl = O.contract(Q, Pc)
            assert np.abs(xv - ref).max() < 1e-13, (P, Pc)
            if Pc % 2 == 0 and Pc < P:
                assert np.abs(xl - ref).max() > 1e-3                  # the literal reading is something else ...
                d = xl - xv                                           # ... by a pure (-1)^j pattern
                assert np.abs(d + np.roll(d, 1, axis=0)).max() < 1e-13
            else:
                assert np.array_equal(xl, xv)
            assert np.abs(Cv.sum(axis=1) - 1).max() < 1e-14           # rows still sum to one (centroid preserved)
            # chain rule: expand_force is the transpose of the contraction
            Fc = rng.standard_normal((Pc, 7))
            O.set_contraction_variant(1)
            fs = O.expand_force(Fc, P)
            O.set_contraction_variant(0)
            G = O.nm_to_beads(fs)
            assert np.abs(G - (P / Pc) * np.einsum("ji,jd->id", Cv, Fc)).max() < 1e-12
        # both force routes of the oracle (normal modes / explicit contraction matrix) follow the switch
        top = W.water_box(27)
        top["box"] = np.array([20.0] * 3)
        t = O.Topology(top)
        x, _ = W.initial_state(top, 8, 300.0, sigma_bead=0.05)
        O.set_contraction_variant(1)
        f, _ = O.nm_forces(t, 8, 4, O.beads_to_nm(x), cells=False)
        Gm = O.bead_forces(t, 8, 4, x, cells=False)
        O.set_contraction_variant(0)
        Gl = O.bead_forces(t, 8, 4, x, cells=False)
        assert np.abs(O.nm_to_beads(f) - Gm).max() < 1e-11 * np.abs(Gm).max()
        assert np.abs(Gl - Gm).max() > 1e-6 * np.abs(Gm).max()
    finally:
        O.set_contraction_variant(0)
