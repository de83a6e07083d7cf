"""Small topology builders for the oracle pins (no method arithmetic)."""
import numpy as np


def mini_top(pos, types, charge, eps, sigma, mass=None, box=40.0, mols=None):
    n = len(pos)
    nt = len(charge)
    return dict(
        n_atoms=n, n_types=nt, n_bonds=0, n_angles=0,
        type=np.asarray(types, np.int32),
        mol=np.arange(n, dtype=np.int32) if mols is None else np.asarray(mols, np.int32),
        mass=np.ones(nt) if mass is None else np.asarray(mass, float),
        charge=np.asarray(charge, float), lj_eps=np.asarray(eps, float),
        lj_sigma=np.asarray(sigma, float), tether_k=None,
        bond_idx=np.zeros((0, 2), np.int32), bond_k=np.zeros(0), bond_r0=np.zeros(0),
        angle_idx=np.zeros((0, 3), np.int32), angle_k=np.zeros(0), angle_th0=np.zeros(0),
        box=np.array([box] * 3), r_cut=9.0, dsf_alpha=0.2, skin=2.0,
        positions=np.asarray(pos, float),
    )


def read_golden(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    with open(path) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
