"""Pins for O5/O8: BAOAB in normal modes with TRPMD/PILE (Eq. 16-17)."""
import numpy as np

import oracle as O
from workloads import water as W

KB, HBAR, ACC = 1.987204258640832e-3, 1.5178728306651436e-2, 418.4


def _free_box(n, mass=1.008):
    return W.oscillator_box(n, mass, 0.0)


def test_A_block_conserves_mode_energies_periodic_and_reversible():
    top = _free_box(4)
    t = O.Topology(top)
    P, T_K = 8, 300.0
    w = O.nm_freq(P, T_K)
    dt = 2 * np.pi / w[1] / 1000.0                 # 1000 steps = one period of modes 1,2
    rng = np.random.default_rng(8)
    x = rng.standard_normal((P, 4, 3)) * 0.1
    p = rng.standard_normal((P, 4, 3)) * 3.0
    sim = O.Rpmd(t, P, P, dt, T_K, "none", 0.0, 1, cells=False)
    sim.set_state(x, p)
    assert np.all(sim.f == 0)
    m = 1.008
    E0 = sim.Pm ** 2 / (2 * m) + 0.5 * m * (w ** 2)[:, None, None] * sim.Q ** 2
    Q0, P0 = sim.Q.copy(), sim.Pm.copy()
    sim.step(1000)
    E1 = sim.Pm ** 2 / (2 * m) + 0.5 * m * (w ** 2)[:, None, None] * sim.Q ** 2
    assert np.abs(E1 - E0).max() < 1e-12 * np.abs(E0).max()      # rounding random walk of 2000 rotations
    assert np.abs(sim.Q[1:3] - Q0[1:3]).max() < 1e-11 and np.abs(sim.Pm[1:3] - P0[1:3]).max() < 1e-9
    assert np.allclose(sim.Q[0], Q0[0] + 1000 * dt * P0[0] / m, rtol=1e-12)    # centroid translation
    sim.step(9000)
    E2 = sim.Pm ** 2 / (2 * m) + 0.5 * m * (w ** 2)[:, None, None] * sim.Q ** 2
    assert np.abs(E2 - E0).max() < 1e-11 * np.abs(E0).max()
    # time reversal
    sim.Pm *= -1
    sim.step(10000)
    assert np.abs(sim.Q - Q0).max() < 1e-10 and np.abs(sim.Pm + P0).max() < 1e-8


def test_O_block_coefficients_and_variance():
    # O only: f = 0, omega irrelevant -> run with dt so large that c1 ~ 0: Pm becomes a fresh
    # Maxwell draw of variance m kB T ACC (Eq. 7 / Eq. 16)
    top = _free_box(2000, mass=15.999)
    t = O.Topology(top)
    P, T_K = 2, 300.0
    sim = O.Rpmd(t, P, P, 1.0, T_K, "pile", 50.0, 12345, cells=True)
    x = np.zeros((P, 2000, 3))
    sim.set_state(x, x.copy())
    sim.f[:] = 0
    lib = O.lib()
    sim.step(1)
    var = (sim.Pm ** 2).mean(axis=(1, 2))
    target = 15.999 * KB * T_K * ACC
    assert np.all(np.abs(var / target - 1) < 5 * np.sqrt(2 / 6000))
    for g, dt in [(1.0, 0.00025), (2513.0, 0.00025)]:
        c1 = np.exp(-g * dt)
        c2 = np.sqrt(1 - c1 * c1)
        assert abs(c1 * c1 + c2 * c2 - 1) < 1e-15


def test_P1_is_classical_baoab_langevin():
    m, k = 1.008, 769.3
    top = W.oscillator_box(5, m, k)
    t = O.Topology(top)
    T_K, dt, g, seed = 300.0, 0.0005, 5.0, 99
    rng = np.random.default_rng(9)
    x = rng.standard_normal((1, 5, 3)) * 0.05
    p = rng.standard_normal((1, 5, 3)) * 2.0
    sim = O.Rpmd(t, 1, 1, dt, T_K, "pile", g, seed, cells=False)
    sim.set_state(x, p, step0=7)
    sim.step(50)
    xo, po = sim.get_state()
    # textbook BAOAB (Leimkuhler-Matthews) written out with numpy
    q, pp = x[0].copy(), p[0].copy()
    c1 = np.exp(-g * dt)
    c2 = np.sqrt(1 - c1 ** 2)
    for s in range(7, 57):
        pp += 0.5 * dt * ACC * (-k * q)
        q += 0.5 * dt * pp / m
        z = np.array([O.normals3(seed, a, 0, 3, s) for a in range(5)])
        pp = c1 * pp + np.sqrt(m * KB * T_K * ACC) * c2 * z
        q += 0.5 * dt * pp / m
        pp += 0.5 * dt * ACC * (-k * q)
    assert np.abs(xo[0] - q).max() < 1e-13 and np.abs(po[0] - pp).max() < 1e-11


def test_harmonic_q2_and_centroid_virial_closed_forms():
    # finite-P closed forms: <q^2> = (1/(beta m)) sum_k 1/(w^2 + w_k^2),
    # <K_CV> per DOF = (kB T/2) sum_k w^2/(w^2 + w_k^2)
    m, w0, T_K, P = 1.008, 565.10, 300.0, 8
    k = m * w0 ** 2 / ACC
    n = 64
    top = W.oscillator_box(n, m, k)
    t = O.Topology(top)
    sim = O.Rpmd(t, P, P, 0.00025, T_K, "pile", 100.0, 2024, cells=False)
    x, p = W.initial_state(top, P, T_K, sigma_bead=0.05)
    sim.set_state(x, p)
    sim.step(2000)
    q2, kcv, cnt = 0.0, 0.0, 0
    for _ in range(600):
        sim.step(30)
        xb = O.nm_to_beads(sim.Q)
        q2 += (xb ** 2).mean()
        kcv += (1.5 * n * KB * T_K - 0.5 * (sim.Q[1:] * sim.f[1:]).sum()) / (3 * n)
        cnt += 1
    q2 /= cnt
    kcv /= cnt
    wk = O.nm_freq(P, T_K)
    q2_ref = KB * T_K * ACC / m * np.sum(1 / (w0 ** 2 + wk ** 2))
    kcv_ref = 0.5 * KB * T_K * np.sum(w0 ** 2 / (w0 ** 2 + wk ** 2))
    assert abs(q2 / q2_ref - 1) < 0.03, (q2, q2_ref)
    assert abs(kcv / kcv_ref - 1) < 0.03, (kcv, kcv_ref)
    # and it is far from the classical value, so the test has teeth
    assert q2_ref > 4 * KB * T_K * ACC / (m * w0 ** 2)
    obs = sim.observables()
    assert abs(obs[0] - (1.5 * n * KB * T_K - 0.5 * (sim.Q[1:] * sim.f[1:]).sum())) < 1e-10


def test_observables_definitions():
    top = W.water_box(216)
    t = O.Topology(top)
    P, Pc, T_K = 4, 2, 300.0
    x, p = W.initial_state(top, P, T_K, sigma_bead=0.05)
    Q, Pm = O.beads_to_nm(x), O.beads_to_nm(p)
    out = O.observables(t, P, Pc, T_K, Q, Pm, cells=False)
    # bead-space centroid-virial estimator: (3N/2 beta) + (1/2P) sum_i (x_i - x_c).grad V(x_i)
    G = O.bead_forces(t, P, Pc, x, cells=False)          # = -grad of P*U_nu
    xc = x.mean(0)
    kcv = 1.5 * 648 * KB * T_K - 0.5 / P * ((x - xc[None]) * G).sum()
    assert abs(out[0] - kcv) < 1e-9 * abs(kcv)
    uf = np.mean([O.force_fast(t, x[i])[0] for i in range(P)])
    xt = O.contract(Q, Pc)
    us = np.mean([O.force_slow(t, xt[j])[0] for j in range(Pc)])
    assert abs(out[1] - (uf + us)) < 1e-10 * abs(uf + us)
    m = top["mass"][top["type"]]
    knm = (Pm ** 2 / (2 * m[None, :, None])).sum() / ACC
    assert abs(out[2] - knm) < 1e-12 * knm
    assert abs(out[3] - 2 * knm / (3 * 648 * P * KB)) < 1e-9
