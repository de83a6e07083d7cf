"""Pins for O9-O11: QTB kernel, segmented coloured noise, spectra, adaptation
(Eq. 12-14, 21-23; l.199-209, 248)."""
import numpy as np
import pytest

import oracle as O
from helpers import read_golden
from workloads import water as W

KB, HBAR, ACC = 1.987204258640832e-3, 1.5178728306651436e-2, 418.4


def test_theta_limits_and_bose_form():
    T_K = 300.0
    kT = KB * T_K
    assert O.lib().qo_theta(0.0, T_K) == kT
    assert abs(O.lib().qo_theta(1e-3, T_K) / kT - 1) < 1e-9                 # classical limit
    w = 5000.0
    assert abs(O.lib().qo_theta(w, T_K) / (0.5 * HBAR * w) - 1) < 1e-12     # zero-point limit
    for w in (10.0, 100.0, 565.1, 2000.0):                                   # north_star form
        bose = HBAR * w * (0.5 + 1.0 / np.expm1(HBAR * w / kT))
        assert abs(O.lib().qo_theta(w, T_K) - bose) < 1e-13 * bose


def test_kernel_is_real_even_and_transforms_back_to_H():
    n_seg, dt, T_K = 64, 0.0005, 300.0
    g = 20.0 * (1 + 0.3 * np.cos(np.arange(n_seg + 1) * 0.1))
    H = O.qtb_filter(n_seg, dt, T_K, 1.008, g)
    w = 2 * np.pi * np.arange(n_seg + 1) / (2 * n_seg * dt)
    assert abs(w[-1] - np.pi / dt) < 1e-9                                    # cutoff pi/dt
    th = O.theta(w, T_K)
    assert np.allclose(H, np.sqrt(2 * (1.008 / ACC) * g * th / dt), rtol=1e-14)
    h = O.qtb_kernel(H)
    k = np.arange(-n_seg, n_seg)
    assert np.abs(h[1:] - h[1:][::-1]).max() < 1e-13 * np.abs(h).max()       # h[k] = h[-k]
    # N_k-point DFT of h (direct) gives back H: G10 deterministic check
    j = np.arange(n_seg + 1)
    Hback = (h[None, :] * np.exp(-2j * np.pi * j[:, None] * k[None, :] / (2 * n_seg))).sum(1)
    assert np.abs(Hback.imag).max() < 1e-11 * H.max()
    assert np.abs(Hback.real - H).max() < 1e-12 * H.max()
    # classical flat spectrum: h is a delta
    Hc = O.qtb_filter(n_seg, dt, T_K, 1.008, np.full(n_seg + 1, 20.0), classical=True)
    hc = O.qtb_kernel(Hc)
    assert abs(hc[n_seg] - Hc[0]) < 1e-12 * Hc[0]
    assert np.abs(np.delete(hc, n_seg)).max() < 1e-12 * Hc[0]


def _top(n):
    return W.oscillator_box(n, 1.008, 769.3)


def test_fft_variant_equals_direct_sum():
    top = _top(3)
    t = O.Topology(top)
    n_seg = 32
    g = 20.0 * (1 + 0.5 * np.sin(np.arange(n_seg + 1) * 0.2) ** 2)
    h = O.qtb_kernel(O.qtb_filter(n_seg, 0.0005, 300.0, 1.008, g))[None]
    for seg in (0, 3):
        Fd = O.qtb_colored_direct(t, n_seg, 5, seg, h)
        Ff = O.qtb_colored_fft(t, n_seg, 5, seg, h)
        assert np.abs(Fd - Ff).max() < 1e-12 * np.abs(Fd).max()
    # definition written out once more in numpy for one value: F_c[n] = sum_k h[k] r[n-k+n_seg]
    r = O.qtb_white(5, 1, 0, 3 * n_seg)
    n = 7
    val = sum(h[0][k + n_seg] * r[2, n - k + n_seg] for k in range(-n_seg, n_seg))
    Fd0 = O.qtb_colored_direct(t, n_seg, 5, 0, h)
    assert abs(val - Fd0[3 * 1 + 2, n]) < 1e-12 * abs(val)


def test_segments_concatenate_to_one_long_convolution():
    # "memory consistent between segments"
    top = _top(2)
    t = O.Topology(top)
    n_seg, nsegs = 16, 5
    g = 20.0 * (1 + 0.5 * np.cos(np.arange(n_seg + 1) * 0.3))
    h = O.qtb_kernel(O.qtb_filter(n_seg, 0.0005, 300.0, 1.008, g))
    F = np.concatenate([O.qtb_colored_direct(t, n_seg, 11, s, h[None]) for s in range(nsegs)], axis=1)
    for a in range(2):
        r = O.qtb_white(11, a, 0, (nsegs + 2) * n_seg)
        for c in range(3):
            full = np.convolve(r[c], h, mode="full")      # full[m] = sum_k' h[k'] r[m-k'], k' = k+n_seg
            ref = full[2 * n_seg: 2 * n_seg + nsegs * n_seg]
            assert np.abs(F[3 * a + c] - ref).max() < 1e-12 * np.abs(ref).max()


def test_noise_power_spectrum_matches_eq13():
    # averaged periodogram -> 2 m gamma Theta(omega)  (Eq. 13), away from the lowest bins
    n_atoms, n_seg, dt, T_K, g0 = 150, 256, 0.0005, 300.0, 20.0
    top = _top(n_atoms)
    t = O.Topology(top)
    g = np.full(n_seg + 1, g0)
    h = O.qtb_kernel(O.qtb_filter(n_seg, dt, T_K, 1.008, g))[None]
    Fc = O.qtb_colored_fft(t, n_seg, 77, 2, h)
    per = dt / n_seg * np.abs(np.fft.rfft(Fc, n=2 * n_seg, axis=1)) ** 2
    psd = per.mean(0)
    w = 2 * np.pi * np.arange(n_seg + 1) / (2 * n_seg * dt)
    ref = 2 * (1.008 / ACC) * g0 * O.theta(w, T_K)
    for lo, hi in [(30, 60), (100, 140), (200, 250)]:
        ratio = psd[lo:hi].mean() / ref[lo:hi].mean()
        assert abs(ratio - 1) < 0.04, (lo, hi, ratio)
    # quantum: high frequencies carry far more power than the classical 2 m gamma kB T
    assert psd[200:250].mean() > 5 * 2 * (1.008 / ACC) * g0 * KB * T_K


def test_classical_limit_is_white_noise_baoab():
    m, k = 1.008, 769.3
    top = W.oscillator_box(4, m, k)
    t = O.Topology(top)
    dt, T_K, g0, seed, n_seg = 0.0005, 300.0, 20.0, 31, 16
    rng = np.random.default_rng(10)
    x = rng.standard_normal((1, 4, 3)) * 0.05
    p = rng.standard_normal((1, 4, 3)) * 2.0
    sim = O.Adqtb(t, dt, T_K, g0, seed, n_seg, a_gamma=0.0, classical=True, direct=True, cells=False)
    sim.set_state(x, p)
    sim.step(40)
    xo, po = sim.get_state()
    q, pp = x[0].copy(), p[0].copy()
    a = np.exp(-g0 * dt)
    for n in range(40):
        pp += 0.5 * dt * ACC * (-k * q)
        q += 0.5 * dt * pp / m
        z = np.array([O.normals3(seed, at, 0, 4, n + n_seg) for at in range(4)])   # G17
        pp = a * pp + np.sqrt(m * KB * T_K * ACC * (1 - a * a)) * z
        q += 0.5 * dt * pp / m
        pp += 0.5 * dt * ACC * (-k * q)
    assert np.abs(xo[0] - q).max() < 1e-12 and np.abs(po[0] - pp).max() < 1e-10


def test_spectra_fft_equals_direct_and_parseval():
    top = W.water_box(216)
    top["n_atoms"] = 648
    t = O.Topology(top)
    n_seg, dt = 32, 0.0005
    rng = np.random.default_rng(12)
    v = rng.standard_normal((1944, n_seg))
    F = rng.standard_normal((1944, n_seg))
    Cd = O.qtb_spectra_direct(t, n_seg, dt, v, F)
    Cf = O.qtb_spectra_fft(t, n_seg, dt, v, F)
    for a, b in zip(Cd, Cf):
        assert np.abs(a - b).max() < 1e-12 * np.abs(a).max()
    # Parseval on the zero-padded DFT: sum_j' |V_j'|^2 = N_k sum_n v_n^2 (full N_k grid)
    wgt = np.ones(n_seg + 1)
    wgt[1:-1] = 2
    tdof = np.repeat(top["type"], 3)
    for z in range(2):
        lhs = (Cd[0][z] * wgt).sum() * n_seg / dt
        rhs = 2 * n_seg * (v[tdof == z] ** 2).sum(1).mean()
        assert abs(lhs - rhs) < 1e-12 * rhs


def test_adaptation_toy_case():
    rows = read_golden("adapt_toy.txt")
    data = {}
    for r in rows:
        data[(r[0], int(r[1]))] = np.array([float(v) for v in r[2:]])
    top = W.oscillator_box(2, 1.0, 0.0)
    top["n_types"] = 2
    top["type"] = np.array([0, 1], np.int32)
    for k in ("mass", "charge", "lj_eps", "lj_sigma"):
        top[k] = np.array([0.0, 0.0])
    top["mass"] = np.array([418.4, 836.8])
    top["tether_k"] = None
    t = O.Topology(top)
    gin = np.stack([data[("gamma_in", z)] for z in range(2)])
    Cvv = np.stack([data[("Cvv", z)] for z in range(2)])
    CvF = np.stack([data[("CvF", z)] for z in range(2)])
    gout = O.qtb_adapt(t, 8, 10.0, 0.5, 0.01, Cvv, CvF, gin)
    ref = np.stack([data[("gamma_out", z)] for z in range(2)])
    assert np.abs(gout - ref).max() < 1e-13


def test_fdt_fixed_point_for_O_only_dynamics():
    # G14: free particles (no force): Re C_vF / (m C_vv) = (1-a)/b * ... frequency independent;
    # with gamma(omega) = gamma0 the mean FDT deviation is ~0 relative to either term (l.124).
    # gamma0 * T_segment = 400/ps * 0.064 ps = 25.6: the free-particle velocity spectrum is a
    # Lorentzian of half-width gamma0 whose rectangular-window leakage is ~1/(gamma0 T_segment)
    # of the signal in every bin (4 % here; it would be 78 % at gamma0 = 20/ps and n_seg = 128).
    n_atoms, n_seg, dt, T_K, g0 = 120, 128, 0.0005, 300.0, 400.0
    top = W.oscillator_box(n_atoms, 1.008, 0.0)
    t = O.Topology(top)
    sim = O.Adqtb(t, dt, T_K, g0, 3, n_seg, a_gamma=0.0, cells=False)
    x, p = W.initial_state(top, 1, T_K)
    sim.set_state(x, p)
    sim.step(6 * n_seg)
    Cvv = np.mean([h[0] for h in sim.history[1:]], axis=0)[0]
    CvF = np.mean([h[1] for h in sim.history[1:]], axis=0)[0]
    lhs = (1.008 / ACC) * g0 * Cvv
    sl = slice(5, n_seg - 5)
    rel = np.abs(lhs[sl] - CvF[sl]).mean() / np.abs(CvF[sl]).mean()
    assert rel < 0.12, rel
    ratio = CvF[sl].sum() / lhs[sl].sum()
    assert abs(ratio - 1) < 0.05, ratio


def test_harmonic_kinetic_energy_is_quantum():
    # K per DOF = 1/2 int dw/2pi 2 g0 w^2 Theta(w) / ((w0^2-w^2)^2 + g0^2 w^2) over |w| < pi/dt
    # (SURVEY.md pins; tends to (hbar w0/4) coth(beta hbar w0/2) as g0 -> 0)
    m, w0, T_K, g0, dt, n_seg = 1.008, 565.10, 300.0, 20.0, 0.0005, 256
    k = m * w0 ** 2 / ACC
    n = 64
    top = W.oscillator_box(n, m, k)
    t = O.Topology(top)
    sim = O.Adqtb(t, dt, T_K, g0, 2025, n_seg, a_gamma=0.0, cells=False)
    x, p = W.initial_state(top, 1, T_K)
    sim.set_state(x, p)
    sim.step(2 * n_seg)
    ks = []
    for _ in range(40):
        sim.step(n_seg // 2)
        ks.append((sim.p ** 2).mean() / (2 * m) / ACC)
    K = np.mean(ks)
    w = np.linspace(1e-6, np.pi / dt, 400001)
    th = 0.5 * HBAR * w / np.tanh(0.5 * HBAR * w / (KB * T_K))
    f = 2 * g0 * w ** 2 * th / ((w0 ** 2 - w ** 2) ** 2 + g0 ** 2 * w ** 2)
    K_ref = 0.5 * 2 * np.trapezoid(f, w) / (2 * np.pi)
    K_q = 0.25 * HBAR * w0 / np.tanh(0.5 * HBAR * w0 / (KB * T_K))
    assert abs(K_ref / K_q - 1.0424) < 0.01            # value quoted in SURVEY.md §8(c)
    assert abs(K / K_ref - 1) < 0.05, (K, K_ref, K_q)
    assert K > 5 * 0.5 * KB * T_K                       # nowhere near classical equipartition


# ---------------------------------------------------------------- kernel-correction hook (reading G11)
def test_kappa_identity_and_amplitude_convention():
    """kappa(omega_j) multiplies the AMPLITUDE filter H (PSD gets kappa^2): kappa = 1 is bit-identical,
    and kappa = sqrt(kB T / Theta) turns the quantum kernel of a flat gamma into the classical delta."""
    n_seg, dt, T_K, m = 64, 0.0005, 300.0, 15.999
    g = np.full(n_seg + 1, 20.0)
    H0 = O.qtb_filter(n_seg, dt, T_K, m, g)
    assert np.array_equal(O.qtb_filter(n_seg, dt, T_K, m, g, kappa=np.ones(n_seg + 1)), H0)
    w = 2 * np.pi * np.arange(n_seg + 1) / (2 * n_seg * dt)
    kap = np.sqrt(KB * T_K / O.theta(w, T_K))
    assert kap[0] == 1.0 and kap[-1] < 0.3                                    # a real, non-trivial factor
    h = O.qtb_kernel(O.qtb_filter(n_seg, dt, T_K, m, g, kappa=kap))
    Hc = np.sqrt(2 * (m / ACC) * 20.0 * KB * T_K / dt)
    assert abs(h[n_seg] - Hc) < 1e-12 * Hc
    assert np.abs(np.delete(h, n_seg)).max() < 1e-12 * Hc
    # DFT of the corrected kernel = kappa x DFT of the uncorrected one (G10 check carried over)
    kap2 = 1.0 + 0.4 * np.sin(np.arange(n_seg + 1) * 0.3)
    h2 = O.qtb_kernel(O.qtb_filter(n_seg, dt, T_K, m, g, kappa=kap2))
    h0 = O.qtb_kernel(H0)
    ext = lambda a: np.concatenate([a, a[-2:0:-1]])                          # even extension to N_k
    D = lambda h: np.fft.fft(np.roll(h, -n_seg)).real                        # h[k], k = 0..N_k-1 ordering
    assert np.abs(D(h2) - ext(kap2) * D(h0)).max() < 1e-12 * np.abs(D(h0)).max()


def test_kappa_classicalising_factor_gives_white_noise_baoab():
    """With kappa = sqrt(kB T / Theta) and adaptation off, the adQTB trajectory is the white-noise BAOAB
    one (the pin of test_classical_limit_is_white_noise_baoab reached through the hook, Theta kept)."""
    top = W.oscillator_box(4, 1.008, 769.3)
    t = O.Topology(top)
    dt, T_K, g0, seed, n_seg = 0.0005, 300.0, 20.0, 31, 16
    rng = np.random.default_rng(10)
    x = rng.standard_normal((1, 4, 3)) * 0.05
    p = rng.standard_normal((1, 4, 3)) * 2.0
    ref = O.Adqtb(t, dt, T_K, g0, seed, n_seg, a_gamma=0.0, classical=True, direct=True, cells=False)
    sim = O.Adqtb(t, dt, T_K, g0, seed, n_seg, a_gamma=0.0, classical=False, direct=True, cells=False)
    w = 2 * np.pi * np.arange(n_seg + 1) / (2 * n_seg * dt)
    sim.kappa = np.sqrt(KB * T_K / O.theta(w, T_K))
    for s in (ref, sim):
        s.set_state(x, p)
        s.step(40)
    assert np.abs(sim.get_state()[0] - ref.get_state()[0]).max() < 1e-12
    assert np.abs(sim.get_state()[1] - ref.get_state()[1]).max() < 1e-10
    # and without the factor the quantum trajectory differs (the hook is not a no-op)
    q = O.Adqtb(t, dt, T_K, g0, seed, n_seg, a_gamma=0.0, classical=False, direct=True, cells=False)
    q.set_state(x, p)
    q.step(40)
    assert np.abs(q.get_state()[0] - ref.get_state()[0]).max() > 1e-6


def test_kappa_constant_scales_the_coloured_force():
    top = W.oscillator_box(3, 1.008, 769.3)
    t = O.Topology(top)
    n_seg, dt, T_K = 32, 0.0005, 300.0
    g = 20.0 * (1 + 0.5 * np.sin(np.arange(n_seg + 1) * 0.2) ** 2)
    h1 = O.qtb_kernel(O.qtb_filter(n_seg, dt, T_K, 1.008, g))[None]
    h3 = O.qtb_kernel(O.qtb_filter(n_seg, dt, T_K, 1.008, g, kappa=np.full(n_seg + 1, 3.0)))[None]
    F1 = O.qtb_colored_direct(t, n_seg, 5, 2, h1)
    F3 = O.qtb_colored_direct(t, n_seg, 5, 2, h3)
    assert np.abs(F3 - 3.0 * F1).max() < 1e-13 * np.abs(F1).max()
