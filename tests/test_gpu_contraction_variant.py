"""GPU-vs-oracle parity with the trigonometric-interpolation contraction (reading G3, variant;
PAPER.md:178-180 Eq. 20): contracted beads, forces and 20 steps for even P' < P; odd P' and P' = P are
untouched by the switch."""
import numpy as np
import pytest

from gpu_common import T_K, make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu

FTOL, XTOL = 1e-10, 1e-8


@pytest.mark.parametrize("P,Pc", [(8, 4), (32, 4), (16, 2), (6, 3), (8, 8)])
def test_trig_variant_matches_oracle(P, Pc):
    import oracle as O
    import scipy.signal as ss
    top = W.water_box(216)
    sysg, ref, x0, p0 = make_pair(top, P, Pc, 0.25, "pile", sigma_bead=0.05)
    sysg.set_contraction("trig")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    try:
        O.set_contraction_variant(1)
        ref.set_state(x0, p0, 0)
        xc = sysg.contracted().cpu().numpy()
        assert np.abs(xc - O.contract(ref.Q, Pc)).max() < 1e-13
        assert np.abs(xc - ss.resample(x0, Pc, axis=0)).max() < 1e-12        # and it is the Fourier interpolant
        G = sysg.forces().cpu().numpy()
        Gref = O.bead_forces(O.Topology(top), P, Pc, x0)
        assert np.abs(G - Gref).max() < FTOL * np.abs(Gref).max()
        sysg.step(20); ref.step(20)
        xr = ref.get_state()[0]
        assert np.abs(sysg.get_state()[0].cpu().numpy() - xr).max() < XTOL
        obs, oref = sysg.observables().cpu().numpy(), ref.observables()
        assert np.abs(obs - oref).max() < 1e-9 * np.abs(oref).max()
    finally:
        O.set_contraction_variant(0)
    lit = O.Rpmd(O.Topology(top), P, Pc, 0.25e-3, T_K, "pile", 1.0, W.MASTER_SEED)
    lit.set_state(x0, p0, 0); lit.step(20)
    differs = np.abs(lit.get_state()[0] - xr).max() > 100 * XTOL
    assert differs == (Pc % 2 == 0 and Pc < P)
    sysg.check()


def test_switch_is_rejected_after_set_state():
    import paper_2212_03137_b200 as qhp
    top = W.water_box(216)
    sysg, _, x0, p0 = make_pair(top, 8, 4, 0.25, "pile")
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    with pytest.raises(qhp.QhpError):
        sysg.set_contraction("trig")
