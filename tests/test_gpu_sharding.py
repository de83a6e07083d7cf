"""Bead-sharded evaluation of V_s (Sec. III.C; SURVEY.md §8(f) NEXT-5a) on ONE GPU:
(i) the bead slices a rank would launch, run one after the other, reproduce the unsliced slow forces bit for bit;
(ii) two systems configured as ranks 0 and 1 of 2 (qhp_set_comm with an exchange callback that rendezvouses on the
host and copies the peer's block device-to-device) follow the unsharded trajectory bit for bit.  No kernel waits on
another kernel; no multi-GPU run is claimed (unmeasured on hardware)."""
import ctypes as C
import threading

import numpy as np
import pytest

from gpu_common import T_K, make_pair, to_dev
from workloads import water as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_mol,P,Pc,slices", [(216, 8, 8, (2, 4, 8)), (5832, 4, 4, (2, 4)), (4096, 32, 4, (2, 4))])
def test_bead_slices_bit_identical(n_mol, P, Pc, slices):
    top = W.water_box(n_mol)
    sysg, _, x0, p0 = make_pair(top, P, Pc, 0.25, "pile", sigma_bead=0.05)
    sysg.set_state(to_dev(x0), to_dev(p0), 0)
    G = sysg.forces().cpu().numpy()
    assert np.isfinite(G).all()
    for g in slices:
        sysg.pair_slices(g)                       # F_s := NaN, then g slice launches
        assert np.array_equal(sysg.forces().cpu().numpy(), G), g
    sysg.check()


def test_two_ranks_emulated_follow_the_unsharded_trajectory():
    import torch
    import paper_2212_03137_b200 as qhp
    from paper_2212_03137_b200.binding import ALLGATHER_FN
    top = W.water_box(5832)
    P, Pc, dt, nsteps = 4, 4, 0.25e-3, 12
    x0, p0 = W.initial_state(top, P, T_K, sigma_bead=0.05)
    ref = qhp.System(top, P, Pc, dt, T_K, "pile", gamma0=1.0, seed=W.MASTER_SEED)
    ref.set_state(to_dev(x0), to_dev(p0), 0)
    ref.step(nsteps)
    xr, pr, _ = ref.get_state()

    world = 2
    bar = threading.Barrier(world)
    ptrs, streams, errors = {}, {}, []

    def make_cb(rank):
        def cb(ctx, ptr, nbytes, rk, wd, cuda_stream):
            try:
                ptrs[rk] = ptr
                streams[rk].synchronize()         # my slice is complete
                bar.wait(timeout=60)
                peer = 1 - rk
                n = nbytes // 8
                mine = qhp.binding._wrap_device_f64(ptr, n * wd)
                theirs = qhp.binding._wrap_device_f64(ptrs[peer], n * wd)
                with torch.cuda.stream(streams[rk]):
                    mine[peer * n:(peer + 1) * n].copy_(theirs[peer * n:(peer + 1) * n])
                streams[rk].synchronize()
                bar.wait(timeout=60)              # nobody overwrites a block before the peer has read it
                return 0
            except Exception as e:                # noqa: BLE001
                errors.append(repr(e))
                return 1
        return ALLGATHER_FN(cb)

    out = {}

    def run(rank):
        try:
            torch.cuda.set_device(0)
            streams[rank] = torch.cuda.Stream()
            with torch.cuda.stream(streams[rank]):
                s = qhp.System(top, P, Pc, dt, T_K, "pile", gamma0=1.0, seed=W.MASTER_SEED, stream=streams[rank])
                cbf = make_cb(rank)
                s._ok(s._L.qhp_set_comm(s._h, rank, world, cbf, None))
                s.set_state(to_dev(x0), to_dev(p0), 0)
                s.step(nsteps)
                x, p, st = s.get_state()
                streams[rank].synchronize()
                out[rank] = (x.cpu().numpy(), p.cpu().numpy(), st)
                s.check()
        except Exception as e:                    # noqa: BLE001
            errors.append(repr(e))
            bar.abort()

    th = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join(timeout=300)
    assert not errors, errors
    for r in range(world):
        assert out[r][2] == nsteps
        assert np.array_equal(out[r][0], xr.cpu().numpy())
        assert np.array_equal(out[r][1], pr.cpu().numpy())


def test_set_comm_argument_errors():
    import paper_2212_03137_b200 as qhp
    from paper_2212_03137_b200.binding import ALLGATHER_FN
    top = W.water_box(216)
    s = qhp.System(top, 8, 4, 0.25e-3, T_K, "pile", gamma0=1.0, seed=1)
    cb = ALLGATHER_FN(lambda *a: 0)
    assert s._L.qhp_set_comm(s._h, 0, 3, cb, None) != 0          # 3 does not divide P' = 4
    assert s._L.qhp_set_comm(s._h, 2, 2, cb, None) != 0          # rank out of range
    assert s._L.qhp_set_comm(s._h, 1, 2, cb, None) == 0
    assert s._L.qhp_set_comm(s._h, 0, 1, cb, None) == 0          # back to one process
