"""Seeded synthetic inputs: flexible 3-site water boxes and initial ring-polymer states.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2212_03137_b200/`).  It holds none of the method's arithmetic (no normal
modes, no forces, no thermostat): only geometry, parameters and random draws from
numpy's own Philox bit generator.

The boxes stand in for the paper's Tinker-HP "puddle" (96,000 atoms) and "pond"
(288,000 atoms) water inputs (Sec. III.D), which are not available;
shapes, density and force-field parameters are BASELINE.json `configs[0..4]`
(recipe: SURVEY.md §8(d), restated in DESIGN.md "Input recipe").

Units: Angstrom, ps, amu, kcal/mol, K, e.
"""
from __future__ import annotations

import numpy as np

MASTER_SEED = 221203137

# unit constants (SURVEY.md §8(c) "Units and constants", CODATA 2018)
KB = 1.987204258640832e-3      # kcal/mol/K
ACC = 418.4                    # 1 kcal/mol = 418.4 amu A^2/ps^2

# BASELINE.json configs[0]: force field of the flexible 3-site water
WATER_FF = dict(
    bond_k=1059.162, bond_r0=1.012,                # kcal/mol/A^2, A
    angle_k=75.90, angle_th0_deg=113.24,           # kcal/mol/rad^2, deg
    lj_eps_O=0.1554, lj_sigma_O=3.1655,            # kcal/mol, A
    q_O=-0.84, q_H=+0.42,
    m_O=15.999, m_H=1.008,
    dsf_alpha=0.2, r_cut=9.0, skin=2.0,
    vol_per_molecule=30.004625,                    # A^3 at 0.997 g/cm^3, M = 18.015
)


def lattice_dims(n_mol: int) -> tuple[int, int, int]:
    """Most cubic exact factorisation nx*ny*nz == n_mol with nx <= ny <= nz."""
    best = None
    for nx in range(1, int(round(n_mol ** (1 / 3))) + 2):
        if n_mol % nx:
            continue
        rest = n_mol // nx
        for ny in range(nx, int(rest ** 0.5) + 2):
            if rest % ny:
                continue
            nz = rest // ny
            if nz < ny:
                continue
            score = nz - nx
            if best is None or score < best[0]:
                best = (score, (nx, ny, nz))
    if best is None:
        raise ValueError(f"cannot factor {n_mol}")
    return best[1]


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random rotation matrices from normalised 4-vectors of normals."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def water_box(n_mol: int, seed: int = MASTER_SEED) -> dict:
    """Topology + centroid positions of `n_mol` waters on a lattice, random orientations.

    Returns a dict of numpy arrays / scalars; atom order O,H,H per molecule,
    type = {0,1,1}, mol = atom // 3.  Keys match the fields of `qhp_topology`
    (include/qhp.h) and of the oracle's topology.
    """
    ff = WATER_FF
    L = (n_mol * ff["vol_per_molecule"]) ** (1.0 / 3.0)
    nx, ny, nz = lattice_dims(n_mol)
    rng = np.random.Generator(np.random.Philox(key=[seed, 0]))
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    O = np.stack([(ii.ravel() + 0.5) * L / nx, (jj.ravel() + 0.5) * L / ny,
                  (kk.ravel() + 0.5) * L / nz], axis=1)
    th = np.deg2rad(ff["angle_th0_deg"])
    r0 = ff["bond_r0"]
    h_local = np.array([[r0 * np.sin(th / 2), 0.0, r0 * np.cos(th / 2)],
                        [-r0 * np.sin(th / 2), 0.0, r0 * np.cos(th / 2)]])
    R = _random_rotations(rng, n_mol)
    H = O[:, None, :] + np.einsum("mij,hj->mhi", R, h_local)
    pos = np.empty((n_mol, 3, 3))
    pos[:, 0] = O
    pos[:, 1:] = H
    pos = pos.reshape(3 * n_mol, 3)
    n_atoms = 3 * n_mol
    mol = (np.arange(n_atoms) // 3).astype(np.int32)
    typ = np.tile(np.array([0, 1, 1], dtype=np.int32), n_mol)
    o_idx = 3 * np.arange(n_mol, dtype=np.int32)
    bond_idx = np.stack([np.stack([o_idx, o_idx + 1], 1), np.stack([o_idx, o_idx + 2], 1)], 1)
    bond_idx = bond_idx.reshape(-1, 2).astype(np.int32)
    angle_idx = np.stack([o_idx + 1, o_idx, o_idx + 2], 1).astype(np.int32)   # (end, centre, end)
    return dict(
        n_atoms=n_atoms, n_types=2, n_bonds=2 * n_mol, n_angles=n_mol,
        type=typ, mol=mol,
        mass=np.array([ff["m_O"], ff["m_H"]]),
        charge=np.array([ff["q_O"], ff["q_H"]]),
        lj_eps=np.array([ff["lj_eps_O"], 0.0]),
        lj_sigma=np.array([ff["lj_sigma_O"], 0.0]),
        tether_k=None,
        bond_idx=bond_idx,
        bond_k=np.full(2 * n_mol, ff["bond_k"]), bond_r0=np.full(2 * n_mol, r0),
        angle_idx=angle_idx,
        angle_k=np.full(n_mol, ff["angle_k"]), angle_th0=np.full(n_mol, th),
        box=np.array([L, L, L]),
        r_cut=ff["r_cut"], dsf_alpha=ff["dsf_alpha"], skin=ff["skin"],
        positions=np.ascontiguousarray(pos),
    )


def ionic_water_box(n_sites: int, ion_every: int = 7, seed: int = MASTER_SEED) -> dict:
    """A water box in which every `ion_every`-th lattice site holds, in turn, a monatomic cation (one-atom
    molecule), a monatomic anion, or a charged diatomic (two atoms, one bond, no angle) instead of a water:
    molecules of 1, 2 and 3 atoms mixed in atom order, four atom types, net charge zero for n_sites a
    multiple of 3 * ion_every.  Not a workload of the paper: the ragged-molecule parity case (tiles, bonded
    ranges, exclusions and the per-type tables must not assume O,H,H triples)."""
    w = water_box(n_sites, seed)
    ff = WATER_FF
    pos_w = w["positions"].reshape(n_sites, 3, 3)
    typ, mol, pos, bonds, bk, br, angles, ak, at = [], [], [], [], [], [], [], [], []
    kind = 0
    for m in range(n_sites):
        a0 = len(typ)
        if m % ion_every == ion_every - 1:
            k = kind % 3
            kind += 1
            if k == 0:                                  # cation, type 2
                typ += [2]; pos += [pos_w[m, 0]]
            elif k == 1:                                # anion, type 3
                typ += [3]; pos += [pos_w[m, 0]]
            else:                                       # diatomic O-H (types 0, 1), one bond; carries -0.42
                typ += [0, 1]; pos += [pos_w[m, 0], pos_w[m, 1]]
                bonds += [[a0, a0 + 1]]; bk += [ff["bond_k"]]; br += [ff["bond_r0"]]
        else:
            typ += [0, 1, 1]; pos += list(pos_w[m])
            bonds += [[a0, a0 + 1], [a0, a0 + 2]]; bk += [ff["bond_k"]] * 2; br += [ff["bond_r0"]] * 2
            angles += [[a0 + 1, a0, a0 + 2]]; ak += [ff["angle_k"]]; at += [np.deg2rad(ff["angle_th0_deg"])]
        mol += [m] * (len(typ) - a0)
    out = dict(w)
    out.update(
        n_atoms=len(typ), n_types=4, n_bonds=len(bonds), n_angles=len(angles),
        type=np.array(typ, np.int32), mol=np.array(mol, np.int32),
        mass=np.array([ff["m_O"], ff["m_H"], 22.99, 35.45]),
        charge=np.array([ff["q_O"], ff["q_H"], 0.92, -0.50]),       # cation + anion + diatomic: 0.92 - 0.50 - 0.42 = 0
        lj_eps=np.array([ff["lj_eps_O"], 0.0, 0.0874, 0.0356]),
        lj_sigma=np.array([ff["lj_sigma_O"], 0.0, 2.439, 4.478]),
        bond_idx=np.array(bonds, np.int32).reshape(-1, 2), bond_k=np.array(bk), bond_r0=np.array(br),
        angle_idx=np.array(angles, np.int32).reshape(-1, 3), angle_k=np.array(ak), angle_th0=np.array(at),
        positions=np.ascontiguousarray(np.array(pos)),
    )
    return out


def oscillator_box(n_atoms: int, mass: float, k_tether: float, box: float = 1000.0,
                   seed: int = MASTER_SEED) -> dict:
    """`n_atoms` uncharged, non-interacting atoms tethered harmonically to the origin.

    V = 1/2 k |x|^2 per atom: the harmonic system for which the paper's methods
    have closed forms (SURVEY.md §8(c) pins).  Each atom is its own
    molecule; no LJ, no charge.  Start positions are small distinct seeded offsets (two atoms
    never coincide, so the zero-charge pair terms stay finite).
    """
    rng = np.random.Generator(np.random.Philox(key=[seed, 2]))
    return dict(
        n_atoms=n_atoms, n_types=1, n_bonds=0, n_angles=0,
        type=np.zeros(n_atoms, np.int32), mol=np.arange(n_atoms, dtype=np.int32),
        mass=np.array([mass]), charge=np.array([0.0]),
        lj_eps=np.array([0.0]), lj_sigma=np.array([0.0]),
        tether_k=np.array([k_tether]),
        bond_idx=np.zeros((0, 2), np.int32), bond_k=np.zeros(0), bond_r0=np.zeros(0),
        angle_idx=np.zeros((0, 3), np.int32), angle_k=np.zeros(0), angle_th0=np.zeros(0),
        box=np.array([box, box, box]), r_cut=9.0, dsf_alpha=0.2, skin=2.0,
        positions=0.05 * rng.standard_normal((n_atoms, 3)),
    )


def initial_state(top: dict, P: int, T_K: float, seed: int = MASTER_SEED,
                  sigma_bead: float = 0.01) -> tuple[np.ndarray, np.ndarray]:
    """Bead positions and bead momenta, both [P][n_atoms][3] fp64.

    Beads = centroid + sigma_bead * N(0,1) (BASELINE.json configs[0]); bead momenta
    are Maxwell draws with variance P*m*kB*T*ACC (amu A/ps)^2, which is the bead-space
    image of "every scaled normal-mode momentum ~ N(0, m kB T)" (Eq. 7,
    SURVEY.md G21) since the transfer matrix is orthogonal.  No COM-momentum removal.
    """
    rng = np.random.Generator(np.random.Philox(key=[seed, 1]))
    n = top["n_atoms"]
    x = top["positions"][None, :, :] + (sigma_bead * rng.standard_normal((P, n, 3)) if P > 1 else 0.0)
    m = top["mass"][top["type"]]
    sp = np.sqrt(P * m * KB * T_K * ACC)
    p = rng.standard_normal((P, n, 3)) * sp[None, :, None]
    return np.ascontiguousarray(x), np.ascontiguousarray(p)


# BASELINE.json configs[0..4]
CONFIGS = {
    "C0": dict(n_mol=216, P=8, P_contract=8, dt_fs=0.25, steps=200, thermostat="pile", gamma0=1.0),
    "C1": dict(n_mol=216, P=1, P_contract=1, dt_fs=0.5, steps=8 * 1024, thermostat="adqtb",
               gamma0=20.0, n_seg=1024, a_gamma=0.5),
    "C2": dict(n_mol=4096, P=32, P_contract=4, dt_fs=0.25, steps=500, thermostat="pile", gamma0=1.0),
    "C3": dict(n_mol=72000, P=1, P_contract=1, dt_fs=0.5, steps=4 * 1024, thermostat="adqtb",
               gamma0=20.0, n_seg=1024, a_gamma=0.5),
    "C4": dict(n_mol=72000, P=32, P_contract=4, dt_fs=0.25, steps=100, thermostat="pile", gamma0=1.0),
}
T_KELVIN = 300.0
