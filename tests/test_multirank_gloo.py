"""N > 1 path on CPU (world_size 2, gloo).  The hot path does not shard in this round ("replicas
only"): every rank runs an independent replica and the only cross-rank step is the
max-over-ranks timing of bench.py.  These tests run that logic, and the rank-0-only reference arm,
in two real processes."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
# each rank "measured" a different time; the job time is the slowest rank's
ms = bench.max_over_ranks(3.0 + 2.0 * rank, 2, device="cpu")
val = bench.job_throughput(2, 648, 8, 10, ms * 1e-3)
dist.barrier()
print(json.dumps(dict(rank=rank, ms=ms, value=val)))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_job_throughput_two_processes(tmp_path):
    port = 29500 + os.getpid() % 2000
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 5.0                                    # max(3, 5) on every rank
        assert o["value"] == pytest.approx(2 * 648 * 8 * 10 / 5.0e-3)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1) == 7.5
    assert bench.job_throughput(1, 100, 4, 5, 2.0) == 1000.0


def test_reference_arm_only_rank0_prints():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 alone runs the oracle and prints; the
    other rank exits 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C0",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C0",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0


SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch
import torch.distributed as dist
from paper_2212_03137_b200.binding import allgather_inplace
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank, world = dist.get_rank(), 2
# F_s is bead-major [P'][N][3]: with P' = 4 beads on 2 ranks, rank r owns beads 2r, 2r+1 = one contiguous block
Pc, N = 4, 5
full = torch.arange(Pc * N * 3, dtype=torch.float64) * 0.5 + 1.0
buf = torch.full((Pc * N * 3,), float("nan"), dtype=torch.float64)
n = buf.numel() // world
buf[rank * n:(rank + 1) * n] = full[rank * n:(rank + 1) * n]        # the slice this rank "computed"
allgather_inplace(buf, rank, world)
dist.barrier()
print(json.dumps(dict(rank=rank, equal=bool(torch.equal(buf, full)))))
dist.destroy_process_group()
"""


def test_bead_slice_allgather_two_processes(tmp_path):
    """The exchange step of the bead-sharded V_s (qhp_set_comm): every rank contributes the contiguous
    bead-major block of its contracted beads, afterwards every rank holds all of F_s.  Host buffers, gloo; on GPUs
    the same call runs over NCCL inside the callback of the library."""
    port = 31500 + os.getpid() % 2000
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        assert json.loads(out.strip().splitlines()[-1])["equal"]
