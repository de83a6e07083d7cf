"""GPU-vs-oracle parity of the adQTB path: coloured-noise segments, BAOAB with the coloured force,
segment spectra and the gamma_z(omega) adaptation (Eq. 12-14, 21-23; l.199-209, 248)."""
import numpy as np
import pytest

from gpu_common import make_pair, oracle_adapt_from_segment, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu


def test_small_segments_full_parity():
    """216 waters, n_seg = 64, three segments with adaptation: F_c, v_seg, gamma, positions."""
    top = W.water_box(216)
    n_seg = 64
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    for seg in range(3):
        sysg.step(n_seg)
        ref.step(n_seg)
        Fc, v = sysg.adqtb_segment()
        Fc, v = Fc.cpu().numpy(), v.cpu().numpy()
        assert np.abs(Fc - ref.Fc).max() < 1e-11 * np.sqrt((ref.Fc ** 2).mean())
        assert np.abs(v - ref.vseg).max() < 1e-9 * np.sqrt((ref.vseg ** 2).mean())
        g = sysg.adqtb_gamma().cpu().numpy()
        assert np.abs(g - ref.gamma).max() < 1e-9 * ref.gamma.max()
    x1, p1, st = sysg.get_state()
    xr, pr = ref.get_state()
    assert st == 3 * n_seg
    assert np.abs(x1.cpu().numpy() - xr).max() < 1e-8
    sysg.check()


def test_direct_sum_noise_definition():
    """F_c against the oracle's direct convolution sum (the definition, no FFT on the oracle side)."""
    import oracle as O
    top = W.water_box(27)
    top["box"] = np.array([20.0, 20.0, 20.0])
    n_seg = 32
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    sysg.step(1)
    Fc, _ = sysg.adqtb_segment(want_v=False)
    otop = O.Topology(top)
    Fref = O.qtb_colored_direct(otop, n_seg, W.MASTER_SEED, 0, ref.kernels())
    assert np.abs(Fc.cpu().numpy() - Fref).max() < 1e-11 * np.sqrt((Fref ** 2).mean())


def test_classical_limit_is_white_noise_baoab():
    """Theta == kB T: the coloured force is h[0] r(n + n_seg): the step is white-noise BAOAB (reading G16)."""
    top = W.water_box(216)
    n_seg = 16
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.0, classical=True)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(20)
    ref.step(20)
    x1, _, _ = sysg.get_state()
    xr, _ = ref.get_state()
    assert np.abs(x1.cpu().numpy() - xr).max() < 1e-8


def test_c1_first_segment_and_boundary():
    """configs[1]: 216 waters, dt = 0.5 fs, gamma0 = 20/ps, n_seg = 1024 (4096-point FFT), A = 0.5:
    one full segment, the adaptation at its end, and 20 steps into the second segment."""
    top = W.water_box(216)
    n_seg = 1024
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(20)
    ref.step(20)
    x1, _, _ = sysg.get_state()
    assert np.abs(x1.cpu().numpy() - ref.get_state()[0]).max() < 1e-8     # north_star: 20 steps
    Fc, _ = sysg.adqtb_segment(want_v=False)
    assert np.abs(Fc.cpu().numpy() - ref.Fc).max() < 1e-11 * np.sqrt((ref.Fc ** 2).mean())
    sysg.step(n_seg - 20)
    ref.step(n_seg - 20)
    # trajectories diverge chaotically over 1024 steps (Lyapunov growth of rounding differences): the
    # velocities are compared with a tolerance that reflects it, and gamma_z is compared at 1e-9 against the
    # oracle's spectra + adaptation applied to the product's OWN segment arrays
    g = sysg.adqtb_gamma().cpu().numpy()
    Fc, v = sysg.adqtb_segment()
    Fc, v = Fc.cpu().numpy(), v.cpu().numpy()
    dv = np.abs(v - ref.vseg).max() / np.sqrt((ref.vseg ** 2).mean())
    assert dv < 1e-4
    import oracle as O
    g_ref, _ = oracle_adapt_from_segment(O.Topology(top), n_seg, 0.5e-3, 20.0, 0.5, 0.01, v, Fc,
                                         np.full_like(g, 20.0))
    assert np.abs(g - g_ref).max() < 1e-9 * g_ref.max()
    assert np.abs(g - 20.0).max() > 0.1                     # the adaptation did move gamma
    sysg.check()


@pytest.mark.parametrize("tau", [None, [0.05, -1.0]])
def test_c1_segment_size_gamma_at_1e9(tau):
    """configs[1]'s n_seg = 1024 (128-thread spectra groups, 9 bins per thread, 2048-point in-kernel FFT): gamma_z
    after each of two adapting segments to 1e-9 of the oracle's update of the product's own v_seg, F_c; SIMPLE
    (Eq. 23) and, for the types with tau > 0, RATIO (Eq. 24-26)."""
    import oracle as O
    top = W.water_box(216)
    n_seg, dt, g0 = 1024, 0.5e-3, 20.0
    sysg, _, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=g0, n_seg=n_seg, a_gamma=0.5)
    otop = O.Topology(top)
    ratio = None
    if tau is not None:
        sysg.adqtb_ratio(tau)
        z = np.zeros((otop.n_types, n_seg + 1))
        ratio = dict(tau=tau, avv=z, avf=z.copy(), started=False)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    g_prev = np.full((otop.n_types, n_seg + 1), g0)
    for seg in range(2):
        sysg.step(n_seg)
        Fc, v = sysg.adqtb_segment()
        g = sysg.adqtb_gamma().cpu().numpy()
        g_ref, ratio = oracle_adapt_from_segment(otop, n_seg, dt, g0, 0.5, 0.01, v.cpu().numpy(), Fc.cpu().numpy(),
                                                 g_prev, ratio)
        assert np.abs(g - g_ref).max() < 1e-9 * np.abs(g_ref).max(), seg
        g_prev = g
    sysg.check()


@pytest.mark.parametrize("tau", [[0.05, -1.0], [0.02, 0.1]])
def test_ratio_adaptation_matches_oracle(tau):
    """RATIO adaptation (Eq. 24-26) for the types with tau > 0, SIMPLE (Eq. 23) for the others:
    gamma_z(omega) after each of four segments, and the trajectory they drive."""
    top = W.water_box(216)
    n_seg = 64
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    ref.ratio_tau = np.asarray(tau, float)
    sysg.adqtb_ratio(tau)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    for seg in range(4):
        sysg.step(n_seg)
        ref.step(n_seg)
        g = sysg.adqtb_gamma().cpu().numpy()
        assert np.abs(g - ref.gamma).max() < 1e-8 * np.abs(ref.gamma).max(), seg
    x1, _, _ = sysg.get_state()
    assert np.abs(x1.cpu().numpy() - ref.get_state()[0]).max() < 1e-7
    sysg.adqtb_ratio(None)                      # back to SIMPLE for every type
    sysg.step(n_seg)
    ref.ratio_tau = None
    ref.step(n_seg)
    assert np.abs(sysg.adqtb_gamma().cpu().numpy() - ref.gamma).max() < 1e-7 * np.abs(ref.gamma).max()
    sysg.check()


def test_kappa_hook_matches_oracle():
    """Kernel-correction factor kappa(omega_j) on the noise filter (reading G11): F_c, gamma and
    positions over three adapting segments with a non-trivial kappa; NULL restores the identity; bad input."""
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    n_seg = 64
    kap = 1.0 + 0.4 * np.sin(np.arange(n_seg + 1) * 0.3) - 0.3 * np.arange(n_seg + 1) / n_seg
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    sysg.adqtb_kappa(kap)
    ref.kappa = kap
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    for seg in range(3):
        sysg.step(n_seg)
        ref.step(n_seg)
        Fc, _ = sysg.adqtb_segment(want_v=False)
        assert np.abs(Fc.cpu().numpy() - ref.Fc).max() < 1e-11 * np.sqrt((ref.Fc ** 2).mean()), seg
        g = sysg.adqtb_gamma().cpu().numpy()
        assert np.abs(g - ref.gamma).max() < 1e-9 * ref.gamma.max(), seg
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < 1e-8
    sysg.adqtb_kappa(None)                       # identity again from the next segment on
    ref.kappa = None
    sysg.step(n_seg)
    ref.step(n_seg)
    Fc, _ = sysg.adqtb_segment(want_v=False)
    assert np.abs(Fc.cpu().numpy() - ref.Fc).max() < 1e-11 * np.sqrt((ref.Fc ** 2).mean())
    bad = kap.copy()
    bad[3] = np.nan
    with pytest.raises(qhp.QhpError):
        sysg.adqtb_kappa(bad)
    sysg.check()


def test_kappa_classicalising_factor_is_white_noise_baoab():
    """kappa = sqrt(kB T / Theta(omega)) with Theta kept quantum: the GPU trajectory equals the oracle's CLASSICAL
    (Theta == kB T) one — the factor enters as an amplitude on H, at the right frequencies."""
    import oracle as O
    top = W.water_box(216)
    n_seg = 16
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.0)
    ref.classical = True
    w = 2 * np.pi * np.arange(n_seg + 1) / (2 * n_seg * 0.5e-3)
    sysg.adqtb_kappa(np.sqrt(1.987204258640832e-3 * 300.0 / O.theta(w, 300.0)))
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(20)
    ref.step(20)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < 1e-8


def test_n_seg_2048_segment_parity():
    """The documented upper limit n_seg = 2048 (8192-point noise transform, 4096-point spectra, one DOF per
    spectra round): F_c of the first segment against the oracle, gamma_z after it from the product's arrays."""
    import oracle as O
    top = W.water_box(27)
    top["box"] = np.array([20.0, 20.0, 20.0])
    n_seg, g0 = 2048, 20.0
    sysg, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=g0, n_seg=n_seg, a_gamma=0.5)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(n_seg)
    ref.step(1)                                          # generates the oracle's first segment
    Fc, v = sysg.adqtb_segment()
    Fc, v = Fc.cpu().numpy(), v.cpu().numpy()
    assert np.abs(Fc - ref.Fc).max() < 1e-11 * np.sqrt((ref.Fc ** 2).mean())
    otop = O.Topology(top)
    g_ref, _ = oracle_adapt_from_segment(otop, n_seg, 0.5e-3, g0, 0.5, 0.01, v, Fc, np.full((otop.n_types, n_seg + 1), g0))
    g = sysg.adqtb_gamma().cpu().numpy()
    assert np.abs(g - g_ref).max() < 1e-9 * np.abs(g_ref).max()
    sysg.check()


def test_restart_with_adapted_gamma_continues_the_run():
    """create -> adqtb_set_gamma -> set_state at a segment boundary in a NEW handle continues an adapted run: the third
    segment equals that of the uninterrupted run (and of the oracle, which ran uninterrupted) -- gamma_z is the only
    adQTB state that has to travel with (x, p, step) for the SIMPLE scheme (Eq. 23); Philox is stateless."""
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    n_seg = 64
    a, ref, x0, p0 = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    a.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    a.step(2 * n_seg)
    ref.step(3 * n_seg)
    x2, p2, st = a.get_state()
    g2 = a.adqtb_gamma().clone()
    assert st == 2 * n_seg and (g2 - 20.0).abs().max().item() > 1e-3      # the run has adapted
    with pytest.raises(qhp.QhpError):
        a.step(1) or a.adqtb_set_gamma(g2)                                # inside a segment: refused
    b, _, _, _ = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    b.adqtb_set_gamma(g2)
    b.set_state(x2, p2, 2 * n_seg)
    b.step(n_seg)
    xb, pb, stb = b.get_state()
    xr, pr = ref.get_state()
    assert stb == 3 * n_seg
    assert np.abs(xb.cpu().numpy() - xr).max() < 1e-8
    assert np.abs(b.adqtb_gamma().cpu().numpy() - ref.gamma).max() < 1e-9 * ref.gamma.max()
    # without the setter the restarted handle would colour its noise with gamma_0
    c, _, _, _ = make_pair(top, 1, 1, 0.5, "adqtb", gamma0=20.0, n_seg=n_seg, a_gamma=0.5)
    c.set_state(x2, p2, 2 * n_seg)
    c.step(n_seg)
    assert np.abs(c.get_state()[0].cpu().numpy() - xr).max() > 1e-6
    b.check()
