"""Statistical checks of the CUDA path against closed forms (BASELINE.json north_star pins, here sampled
on the GPU where long runs are cheap): the finite-P harmonic <q^2> and centroid-virial kinetic energy of
PILE-thermostatted RPMD, and the quantum kinetic energy of a harmonic oscillator under the
QTB.  They complement the step-by-step parity tests: a sampling error that parity over 20
steps cannot see (a wrong thermostat variance, a biased noise spectrum) fails here."""
import numpy as np
import pytest

from gpu_common import to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

KB, HBAR, ACC = 1.987204258640832e-3, 1.5178728306651436e-2, 418.4
T_K, M_H, W0 = 300.0, 1.008, 565.10                      # rad/ps: a 3000 cm^-1 O-H stretch


@pytest.mark.parametrize("P,a_block", [(8, "exact"), (32, "exact"), (8, "cayley")])
def test_rpmd_pile_harmonic_closed_forms(P, a_block):
    import oracle as O
    import paper_2212_03137_b200 as qhp
    n = 1024
    top = W.oscillator_box(n, M_H, M_H * W0 ** 2 / ACC)
    sysg = qhp.System(top, P, P, 0.25e-3, T_K, "pile", gamma0=100.0, seed=2024)
    sysg.set_a_block(a_block)
    x, p = W.initial_state(top, P, T_K, sigma_bead=0.05)
    sysg.set_state(to_dev(x), to_dev(p), 0)
    sysg.step(4000)                                       # 1 ps: many relaxation times of every mode
    q2, kcv, cnt = 0.0, 0.0, 0
    for _ in range(150):
        sysg.step(40)
        xb, _, _ = sysg.get_state()
        q2 += float((xb ** 2).mean())
        kcv += float(sysg.observables()[0]) / (3 * n)
        cnt += 1
    q2, kcv = q2 / cnt, kcv / cnt
    wk = O.nm_freq(P, T_K)                                # the only use of the oracle here: the free-RP frequencies
    q2_ref = KB * T_K * ACC / M_H * np.sum(1.0 / (W0 ** 2 + wk ** 2))
    kcv_ref = 0.5 * KB * T_K * np.sum(W0 ** 2 / (W0 ** 2 + wk ** 2))
    assert abs(q2 / q2_ref - 1) < 0.01, (q2, q2_ref)
    assert abs(kcv / kcv_ref - 1) < 0.01, (kcv, kcv_ref)
    assert q2_ref > 3 * KB * T_K * ACC / (M_H * W0 ** 2)  # far from the classical value
    sysg.check()


def test_qtb_harmonic_kinetic_energy_is_quantum():
    """K per DOF = (1/2) int dw/2pi 2 g0 w^2 Theta(w) / ((w0^2 - w^2)^2 + g0^2 w^2) over |w| < pi/dt, which
    tends to (hbar w0 / 4) coth(beta hbar w0 / 2) for small g0; no adaptation (a_gamma = 0)."""
    import paper_2212_03137_b200 as qhp
    n, g0, dt, n_seg = 1024, 20.0, 0.5e-3, 1024
    top = W.oscillator_box(n, M_H, M_H * W0 ** 2 / ACC)
    sysg = qhp.System(top, 1, 1, dt, T_K, "adqtb", gamma0=g0, seed=2025, n_seg=n_seg, a_gamma=0.0)
    x, p = W.initial_state(top, 1, T_K)
    sysg.set_state(to_dev(x), to_dev(p), 0)
    sysg.step(2 * n_seg)
    ks = []
    for _ in range(60):
        sysg.step(128)
        _, pb, _ = sysg.get_state()
        ks.append(float((pb ** 2).mean()) / (2 * M_H) / ACC)
    K = np.mean(ks)
    w = np.linspace(1e-6, np.pi / dt, 400001)
    th = 0.5 * HBAR * w / np.tanh(0.5 * HBAR * w / (KB * T_K))
    f = 2 * g0 * w ** 2 * th / ((W0 ** 2 - w ** 2) ** 2 + g0 ** 2 * w ** 2)
    K_ref = 0.5 * 2 * np.trapezoid(f, w) / (2 * np.pi)
    K_q = 0.25 * HBAR * W0 / np.tanh(0.5 * HBAR * W0 / (KB * T_K))
    assert abs(K_ref / K_q - 1.0424) < 0.01
    assert abs(K / K_ref - 1) < 0.02, (K, K_ref, K_q)
    assert K > 5 * 0.5 * KB * T_K
    sysg.check()
