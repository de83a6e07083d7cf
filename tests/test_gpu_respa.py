"""GPU-vs-oracle parity of BAOAB-RESPA (Eq. 19): V_f in the
inner loop of n_alt steps, V_s (on the contracted beads) once per outer step."""
import numpy as np
import pytest

from gpu_common import T_K, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

XTOL = 1e-8      # Angstrom (north_star)


def _pair(top, P, Pc, dt_fs, thermo, n_alt, gamma0=1.0, sigma_bead=0.01):
    import oracle as O
    import paper_2212_03137_b200 as qhp
    x0, p0 = W.initial_state(top, P, T_K, sigma_bead=sigma_bead)
    sysg = qhp.System(top, P, Pc, dt_fs * 1e-3, T_K, thermo, gamma0=gamma0, seed=W.MASTER_SEED)
    sysg.set_respa(n_alt)
    ref = O.RpmdRespa(O.Topology(top), P, Pc, dt_fs * 1e-3, T_K, thermo, gamma0, W.MASTER_SEED, n_alt)
    return sysg, ref, x0, p0


@pytest.mark.parametrize("thermo,P,Pc,n_alt", [("pile", 8, 4, 4), ("none", 8, 8, 2), ("pile", 1, 1, 5)])
def test_small_box_20_inner_steps(thermo, P, Pc, n_alt):
    top = W.water_box(216)
    sysg, ref, x0, p0 = _pair(top, P, Pc, 0.25, thermo, n_alt)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(2 * n_alt)
    sysg.step(20 - 2 * n_alt)                 # two calls: the pending kicks of both parts must carry over
    ref.step(20)
    x1, p1, st = sysg.get_state()
    xr, pr = ref.get_state()
    assert st == 20
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    assert np.abs(p1.cpu().numpy() - pr).max() < 1e-6 * np.abs(pr).max()
    G = sysg.forces().cpu().numpy()
    Gr = O_forces(ref)
    assert np.abs(G - Gr).max() < 1e-7 * np.abs(Gr).max()
    obs = sysg.observables().cpu().numpy()
    oref = ref.observables()
    assert np.abs(obs - oref).max() < 1e-7 * np.abs(oref).max()
    sysg.check()


def O_forces(ref):
    import oracle as O
    return O.nm_to_beads(ref.f)


def test_staged_kernel_and_contraction_with_respa():
    """5832 waters (staged pair kernel), P = 4 contracted to 2, n_alt = 2."""
    top = W.water_box(5832)
    sysg, ref, x0, p0 = _pair(top, 4, 2, 0.25, "pile", 2, sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1
    ref.set_state(x0, p0, 0)
    sysg.step(8)
    ref.step(8)
    x1, _, _ = sysg.get_state()
    assert np.abs(x1.cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()


def test_step_count_must_be_a_multiple_of_n_alt():
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    sysg, _, x0, p0 = _pair(top, 2, 2, 0.25, "pile", 4)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    with pytest.raises(qhp.QhpError):
        sysg.step(3)
    sysg.step(4)
    with pytest.raises(qhp.QhpError):
        sysg.set_respa(3)                     # 4 is not a multiple of 3
    sysg.set_respa(1)
    sysg.step(1)
    sysg.check()


def test_n_alt_switch_mid_run_matches_oracle():
    """qhp_set_respa between steps: the pending closing kick of the last outer step must be applied with the
    n_alt it was taken under (4 -> 1 and 1 -> 4).  The oracle side chains three drivers through their state."""
    import oracle as O
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    P, Pc, dt = 8, 4, 0.25e-3
    x0, p0 = W.initial_state(top, P, T_K)
    sysg = qhp.System(top, P, Pc, dt, T_K, "pile", gamma0=1.0, seed=W.MASTER_SEED)
    sysg.set_respa(4)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    sysg.step(4)
    sysg.set_respa(1)
    sysg.step(4)
    sysg.set_respa(4)
    sysg.step(8)
    x1, p1, st = sysg.get_state()
    assert st == 16
    otop = O.Topology(top)
    x, p, step = x0, p0, 0
    for n_alt, n in ((4, 4), (1, 4), (4, 8)):
        ref = O.RpmdRespa(otop, P, Pc, dt, T_K, "pile", 1.0, W.MASTER_SEED, n_alt)
        ref.set_state(x, p, step)
        ref.step(n)
        x, p = ref.get_state()
        step += n
    assert np.abs(x1.cpu().numpy() - x).max() < XTOL
    assert np.abs(p1.cpu().numpy() - p).max() < 1e-6 * np.abs(p).max()
    sysg.check()
