"""GPU-vs-oracle parity of the BCOCB variant (G25): the A
half-steps of the fused integrator take the square-root-Cayley coefficients instead of cos / sin."""
import numpy as np
import pytest

from gpu_common import T_K, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

XTOL = 1e-8      # Angstrom (north_star)


def _pair(top, P, Pc, dt_fs, thermo, n_alt=1, gamma0=1.0, sigma_bead=0.01):
    import oracle as O
    import paper_2212_03137_b200 as qhp
    x0, p0 = W.initial_state(top, P, T_K, sigma_bead=sigma_bead)
    sysg = qhp.System(top, P, Pc, dt_fs * 1e-3, T_K, thermo, gamma0=gamma0, seed=W.MASTER_SEED)
    sysg.set_a_block("cayley")
    sysg.set_respa(n_alt)
    ot = O.Topology(top)
    if n_alt == 1:
        ref = O.Rpmd(ot, P, Pc, dt_fs * 1e-3, T_K, thermo, gamma0, W.MASTER_SEED, a_block="cayley")
    else:
        ref = O.RpmdRespa(ot, P, Pc, dt_fs * 1e-3, T_K, thermo, gamma0, W.MASTER_SEED, n_alt, a_block="cayley")
    return sysg, ref, x0, p0


@pytest.mark.parametrize("thermo,P,Pc,dt_fs,n_alt", [("pile", 8, 4, 0.25, 1), ("none", 16, 4, 0.5, 1),
                                                     ("pile", 32, 4, 0.25, 1), ("pile", 8, 2, 0.25, 4)])
def test_small_box_20_steps(thermo, P, Pc, dt_fs, n_alt):
    import oracle as O
    top = W.water_box(216)
    sysg, ref, x0, p0 = _pair(top, P, Pc, dt_fs, thermo, n_alt)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(8)
    sysg.step(12)
    ref.step(20)
    x1, p1, st = sysg.get_state()
    xr, pr = ref.get_state()
    assert st == 20
    assert np.abs(x1.cpu().numpy() - xr).max() < XTOL
    assert np.abs(p1.cpu().numpy() - pr).max() < 1e-6 * np.abs(pr).max()
    # and the switch really changed the trajectory: the exact-A oracle is somewhere else
    ex = O.Rpmd(O.Topology(top), P, Pc, dt_fs * 1e-3, T_K, thermo, 1.0, W.MASTER_SEED) if n_alt == 1 else None
    if ex is not None:
        ex.set_state(x0, p0, 0); ex.step(20)
        assert np.abs(ex.get_state()[0] - xr).max() > 100 * XTOL
    sysg.check()


def test_switching_back_to_the_exact_block():
    import oracle as O
    top = W.water_box(216)
    sysg, ref, x0, p0 = _pair(top, 8, 4, 0.25, "pile")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    ref.set_state(x0, p0, 0)
    sysg.step(5); ref.step(5)
    sysg.set_a_block("exact")
    ex = O.Rpmd(O.Topology(top), 8, 4, 0.25e-3, T_K, "pile", 1.0, W.MASTER_SEED)
    ex.set_state(*ref.get_state(), 5)
    sysg.step(5); ex.step(5)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ex.get_state()[0]).max() < XTOL
    with pytest.raises(Exception):
        sysg.set_a_block("verlet")
    sysg.check()


def test_staged_kernel_mid_size():
    top = W.water_box(5832)
    sysg, ref, x0, p0 = _pair(top, 4, 2, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    assert sysg.counters()["staged"] == 1
    ref.set_state(x0, p0, 0)
    sysg.step(6); ref.step(6)
    assert np.abs(sysg.get_state()[0].cpu().numpy() - ref.get_state()[0]).max() < XTOL
    sysg.check()
