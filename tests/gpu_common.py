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
