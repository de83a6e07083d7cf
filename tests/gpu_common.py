"""Shared fixtures of the GPU parity tests: build the same seeded system on both sides."""
import numpy as np

from workloads import water as W

T_K = W.T_KELVIN


def to_dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def make_pair(top, P, Pc, dt_fs, thermostat, gamma0=1.0, seed=W.MASTER_SEED, state_seed=W.MASTER_SEED,
              sigma_bead=0.01, **kw):
    """Returns (gpu System, oracle driver, x0, p0)."""
    import oracle as O
    import paper_2212_03137_b200 as qhp
    x0, p0 = W.initial_state(top, P, T_K, seed=state_seed, sigma_bead=sigma_bead)
    sysg = qhp.System(top, P, Pc, dt_fs * 1e-3, T_K, thermostat, gamma0=gamma0, seed=seed, **kw)
    otop = O.Topology(top)
    if thermostat == "adqtb":
        ref = O.Adqtb(otop, dt_fs * 1e-3, T_K, gamma0, seed, kw["n_seg"], kw.get("a_gamma", 0.0),
                      kw.get("gamma_min_frac", 0.01), classical=kw.get("classical", False))
    else:
        ref = O.Rpmd(otop, P, Pc, dt_fs * 1e-3, T_K, thermostat, gamma0, seed)
    return sysg, ref, x0, p0


def oracle_adapt_from_segment(otop, n_seg, dt_ps, gamma0, a_gamma, gmin_frac, vseg, Fc, gamma_before,
                              ratio=None):
    """End-of-segment update of gamma_z(omega) by the oracle's own routines (spectra Eq. 21-22 through its
    DFT, per-type means, SIMPLE Eq. 23 / RATIO Eq. 24-26, lower bound l.248) applied to GIVEN segment arrays
    vseg, Fc [3N][n_seg] -- the product's own arrays in the tests that call it, which takes the chaotic
    divergence of two 1024-step trajectories out of the comparison.  ratio = dict(tau, avv, avf, started) or
    None; returns (gamma_after, ratio)."""
    import oracle as O
    Cvv, CvF = O.qtb_spectra_fft(otop, n_seg, dt_ps, vseg, Fc)
    g = O.qtb_adapt(otop, n_seg, gamma0, a_gamma, gmin_frac, Cvv, CvF, gamma_before)
    if ratio is not None:
        tau = np.asarray(ratio["tau"], float)
        g_r, avv, avf = O.qtb_adapt_ratio(otop, n_seg, gamma0, gmin_frac, dt_ps, tau, not ratio["started"],
                                          Cvv, CvF, ratio["avv"], ratio["avf"], gamma_before)
        for z in range(otop.n_types):
            if tau[z] > 0:
                g[z] = g_r[z]
        ratio = dict(tau=tau, avv=avv, avf=avf, started=True)
    return g, ratio
