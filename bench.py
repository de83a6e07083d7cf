#!/usr/bin/env python
"""bench.py -- throughput of the Quantum-HP hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl ours|reference]

A "step" is one pass of the whole hot path (SURVEY.md §8(a) rows R1-R12 for RPMD, Q1-Q7 for adQTB)
over the synthetic water box of the chosen BASELINE.json config: one `qhp_step(1)`.
Default workload C4 = configs[4]: 72,000 waters (216,000 atoms), P = 32 beads, P' = 4 contracted
beads, dt = 0.25 fs, PILE -- the configuration BASELINE.json's metric (bead-atom-steps/s and ns/day at
216k atoms) is quoted on.  `--workload C3` times the 216k-atom adQTB configuration.

* value     = N_gpus * n_atoms * P * K / (max over ranks of the device time of K steps), state
              resident in HBM.
* e2e       = the same K steps through the host entry points of the C ABI: qhp_set_state_host
              (pinned host -> device), qhp_step(K), qhp_get_state_host + qhp_observables_host
              (device -> host), all inside the timed region.
* roofline  = the dominant kernel (pair forces, FP64-ALU bound): algorithmic flops per launch /
              its average device time, measured with CUDA events recorded by the library on its
              stream around every launch inside the timed region (qhp_profile).
* cpu_baseline = the oracle (oracle/, plain C, one thread) timed on this box's host on one step of
              the same workload.
N > 1 (torchrun): the path does not shard in this round ("replicas only"): every rank
runs an independent replica of the workload on its own GPU; barrier + max-over-ranks timing.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import water as W  # noqa: E402

# algorithmic work of the pair kernel per in-cutoff pair-bead: minimum
# image + distance 15 flop, DSF Coulomb (rsqrt, exp, erfc) + LJ + force accumulation 95 flop.
FLOP_PER_PAIR_BEAD = 110.0
# FP64 ALU peak derived from unit counts: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (max SM clock);
# bench.py also measures it live with qhp_dfma_probe and reports both.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum of one k_pair_staged<false> launch at C4, from the
# `ncu --set full` capture summarised in profiles/r1c_summary.md (per launch, like `achieved`)
NCU_TRAFFIC_BYTES = {("C4", "k_pair_staged"): 1.3637e9 + 2.39e7,      # profiles/r1d_summary.md (dram read + write per launch)
                     ("C3", "k_pair_staged"): 3.409e8 + 9.5e6}


def measure_dfma_peak() -> float:
    """Dependent-FMA probe on every SM (8 chains per thread): measured FP64 FMA throughput, TFLOP/s."""
    import torch
    import paper_2212_03137_b200 as qhp
    grid, block, iters = 148 * 8, 256, 1 << 16
    qhp.qhp_dfma_probe(grid, block, iters)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = float("inf")
    for _ in range(3):
        e0.record()
        qhp.qhp_dfma_probe(grid, block, iters)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return 2.0 * grid * block * iters / (best * 1e-3) / 1e12


def workload(name: str) -> dict:
    cfg = dict(W.CONFIGS[name])
    cfg["name"] = name
    return cfg


def peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return dict(hbm_gbs=float(d["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([c.strip() for c in ln.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))


def max_over_ranks(x: float, world: int, device: str = "cuda") -> float:
    """Replicas only: every rank times its own replica; the job's time is the slowest
    rank's.  One all-reduce(MAX) of a scalar on the job's process group (nccl on GPUs, gloo in the
    CPU tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world: int, n_atoms: int, P: int, steps: int, seconds: float) -> float:
    """bead-atom-steps/s of the whole job: all ranks' replicas over the slowest rank's time (weak scaling)."""
    return world * n_atoms * P * steps / seconds


def build_system(cfg: dict):
    import paper_2212_03137_b200 as qhp
    top = W.water_box(cfg["n_mol"])
    kw = {}
    if cfg["thermostat"] == "adqtb":
        kw = dict(n_seg=cfg["n_seg"], a_gamma=cfg["a_gamma"])
    sysg = qhp.System(top, cfg["P"], cfg["P_contract"], cfg["dt_fs"] * 1e-3, W.T_KELVIN, cfg["thermostat"],
                      gamma0=cfg["gamma0"], seed=W.MASTER_SEED, **kw)
    x0, p0 = W.initial_state(top, cfg["P"], W.T_KELVIN)
    return top, sysg, x0, p0


def oracle_steps(cfg: dict, top: dict, x0, p0, n: int):
    """Oracle driver advanced n steps; returns (driver, seconds per step) -- setup is not timed."""
    import oracle as O
    otop = O.Topology(top)
    if cfg["thermostat"] == "adqtb":
        ref = O.Adqtb(otop, cfg["dt_fs"] * 1e-3, W.T_KELVIN, cfg["gamma0"], W.MASTER_SEED, cfg["n_seg"], cfg["a_gamma"])
    else:
        ref = O.Rpmd(otop, cfg["P"], cfg["P_contract"], cfg["dt_fs"] * 1e-3, W.T_KELVIN, cfg["thermostat"],
                     cfg["gamma0"], W.MASTER_SEED)
    ref.set_state(x0, p0, 0)
    if cfg["thermostat"] == "adqtb":
        ref._new_segment()                       # noise generation is per segment, not per step
        ref._seg_of_Fc = 0
    t0 = time.perf_counter()
    ref.step(n)
    return ref, (time.perf_counter() - t0) / n


def run_reference(args):
    """--impl reference: the oracle as it stands, on this box's host cores (one thread)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload(args.workload)
    # bounded sample: the same force field / density / P / P', on a box small enough that
    # K + W oracle steps end within a few minutes (oracle cost ~ 1e-4 s per atom per step at P=32/P'=4)
    per_atom = 1.0e-4 * (cfg["P"] + 8 * cfg["P_contract"]) / 64.0
    n_mol = cfg["n_mol"]
    for cand in (72000, 4096, 1728, 512, 216):
        if cand <= cfg["n_mol"]:
            n_mol = cand
            if (args.steps + args.warmup + 1) * 3 * cand * per_atom <= 150.0:
                break
    scfg = dict(cfg, n_mol=n_mol)
    top = W.water_box(n_mol)
    x0, p0 = W.initial_state(top, cfg["P"], W.T_KELVIN)
    import oracle as O
    O.build()
    ref, _ = oracle_steps(scfg, top, x0, p0, max(args.warmup, 1))
    t0 = time.perf_counter()
    ref.step(args.steps)
    dt = time.perf_counter() - t0
    n_atoms = 3 * n_mol
    value = n_atoms * cfg["P"] * args.steps / dt
    sample = f"{n_mol} waters ({n_atoms} atoms) of the {cfg['name']} workload, P={cfg['P']}, P'={cfg['P_contract']}, {args.steps} steps"
    line = dict(impl="reference", metric="bead_atom_steps_per_s", value=value, unit="bead-atom-steps/s", n_gpus=0,
                steps=args.steps, warmup=args.warmup, ms_per_step=1e3 * dt / args.steps, higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=cfg["name"], sample=sample, thermostat=cfg["thermostat"]),
                cpu_baseline=dict(value=value, unit="bead-atom-steps/s", cores=1, kind="oracle", sample=sample),
                e2e=dict(value=value, unit="bead-atom-steps/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="C4", choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--a-block", choices=["exact", "cayley"], default="exact", help="cayley = BCOCB (PAPER.md:151); exact = the BASELINE.json configs")
    ap.add_argument("--n-alt", type=int, default=1, help="BAOAB-RESPA inner steps per V_s evaluation (PAPER.md Eq. 19); 1 = the BASELINE.json configs")
    ap.add_argument("--n-mol", type=int, default=0, help="profiling aid: the same workload on a box of this many waters (0 = the BASELINE.json size)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    from paper_2212_03137_b200 import build as qbuild
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if rank == 0:
        qbuild.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()

    cfg = workload(args.workload)
    if args.n_mol > 0:
        cfg["n_mol"] = args.n_mol
    top, sysg, x0, p0 = build_system(cfg)
    N, P, K = top["n_atoms"], cfg["P"], args.steps
    xd = torch.as_tensor(x0).cuda()
    pd = torch.as_tensor(p0).cuda()
    if args.a_block != "exact":
        sysg.set_a_block(args.a_block)
    if args.n_alt > 1:
        sysg.set_respa(args.n_alt)
        args.warmup = -(-args.warmup // args.n_alt) * args.n_alt
        args.steps = K = -(-args.steps // args.n_alt) * args.n_alt
    sysg.set_state(xd, pd, 0)
    sysg.step(args.warmup)
    sysg.check()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K steps, state resident in HBM ------------------------------------------
    c0 = sysg.counters()
    sysg.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        barrier()
        e0.record()
        sysg.step(K)
        e1.record()
        barrier()
    ms = e0.elapsed_time(e1)
    prof = sysg.profile_read()
    sysg.profile(False)
    c1 = sysg.counters()
    launches = c1["launches"] - c0["launches"]          # kernels the library launched inside the timed region
    ms = max_over_ranks(ms, world)
    value = job_throughput(world, N, P, K, ms * 1e-3)
    ns_day = K * cfg["dt_fs"] * 1e-6 / (ms * 1e-3) * 86400.0

    # ---- roofline of the dominant kernel (pair forces) ------------------------------------------
    pair_ms = prof["pair"]["ms"] / max(prof["pair"]["n"], 1)
    int_ms = prof["integrate"]["ms"] / max(prof["integrate"]["n"], 1)
    pair_beads = c1["pair_beads_in_cutoff"]             # ordered (full list): each pair from both sides
    flops_algo = 0.5 * pair_beads * FLOP_PER_PAIR_BEAD  # algorithmic: every unordered pair-bead once
    ach = flops_algo / (pair_ms * 1e-3) / 1e12 if pair_ms > 0 else 0.0
    pk = peaks()
    kname = "k_pair_staged" if c1.get("staged") else "k_pair"
    dfma_tf = measure_dfma_peak()
    roofline = dict(kernel=kname, bound="alu", achieved=ach, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s",
                    frac=ach / FP64_PEAK_TFLOPS, traffic=NCU_TRAFFIC_BYTES.get((cfg["name"], kname)),
                    peak_source="derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz",
                    peak_measured=dfma_tf, frac_of_measured=ach / dfma_tf if dfma_tf > 0 else None,
                    executed_tflops=2.0 * ach, ms_per_launch=pair_ms,
                    note="achieved counts each unordered in-cutoff pair-bead once (110 flop); the kernel "
                         "evaluates both directions (full list, no atomics), see executed_tflops; "
                         "peak_measured = live qhp_dfma_probe")
    # second kernel: fused integrator pass, HBM-bound: 4 x 8 B per (DOF, bead) + 2 x 24 B * P'/P ... per atom-bead
    int_bytes = 4.0 * 8 * 3 * N * P + (32.0 + 24.0) * N * cfg["P_contract"]
    int_gbs = int_bytes / (int_ms * 1e-3) / 1e9 if int_ms > 0 else 0.0
    kernels = dict(k_integrate=dict(bound="hbm", ms_per_launch=int_ms, achieved=int_gbs, peak=pk["hbm_gbs"], unit="GB/s",
                                    frac=int_gbs / pk["hbm_gbs"], peak_source=pk["source"]),
                   rebuild_chain=dict(ms_per_step=prof["rebuild"]["ms"] / max(prof["rebuild"]["n"], 1),
                                      rebuilds=c1["rebuilds"] - c0["rebuilds"]),
                   qtb_generate=dict(ms_per_segment=prof["qtb_generate"]["ms"] / max(prof["qtb_generate"]["n"], 1), n=prof["qtb_generate"]["n"]),
                   qtb_adapt=dict(ms_per_segment=prof["qtb_adapt"]["ms"] / max(prof["qtb_adapt"]["n"], 1), n=prof["qtb_adapt"]["n"]))

    # ---- e2e through the host entry points ----------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        xh = torch.as_tensor(x0).pin_memory()
        ph = torch.as_tensor(p0).pin_memory()
        xo, po = torch.empty_like(xh).pin_memory(), torch.empty_like(ph).pin_memory()
        sysg.set_state_host(xh, ph, 0)          # untimed pass: allocates the staging buffers
        sysg.step(3 * args.n_alt)
        sysg.get_state_host(xo, po)
        sysg.observables_host()                 # every call of the timed region has run once (lazy module loading, buffers)
        barrier()
        t0 = time.perf_counter()
        sysg.set_state_host(xh, ph, 0)
        t1 = time.perf_counter()
        sysg.step(K)
        sysg.get_state_host(xo, po)             # synchronises: the host buffers are valid on return
        t2 = time.perf_counter()
        obs = sysg.observables_host()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        parts = dict(set_state_host=1e3 * (t1 - t0), steps_and_get_state_host=1e3 * (t2 - t1), observables_host=1e3 * (t0 + t_e2e - t2))
        t_e2e = max_over_ranks(t_e2e, world)
        nbytes = xh.numel() * 8
        e2e = dict(value=job_throughput(world, N, P, K, t_e2e), unit="bead-atom-steps/s",
                   h2d_bytes_per_step=2 * nbytes / K, d2h_bytes_per_step=(2 * nbytes + 32) / K,
                   ms_total=1e3 * t_e2e, ms_parts=parts, what="set_state_host + qhp_step(K) + get_state_host + observables_host",
                   observables=[float(v) for v in obs])
    sysg.check()

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- oracle on the host cores (bounded sample: one step of the same workload) ----------------
    cpu = None
    if not args.no_cpu_baseline:
        import oracle as O
        O.build()
        n_cpu = 1 if N > 20000 else (5 if N > 2000 else 20)
        _, s_per_step = oracle_steps(cfg, top, x0, p0, n_cpu)
        cpu = dict(value=N * P / s_per_step, unit="bead-atom-steps/s", cores=1, kind="oracle",
                   sample=f"{n_cpu} step(s) of the full {cfg['name']} workload ({N} atoms, P={P}, P'={cfg['P_contract']}), "
                          f"{s_per_step:.2f} s/step, setup (initial forces) not timed",
                   host_cores_available=os.cpu_count())

    line = dict(metric="bead_atom_steps_per_s", value=value, unit="bead-atom-steps/s", n_gpus=world, steps=K,
                warmup=args.warmup, ms_per_step=ms / K, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic",
                config=dict(workload=cfg["name"], n_atoms=N, P=P, P_contract=cfg["P_contract"], dt_fs=cfg["dt_fs"],
                            thermostat=cfg["thermostat"], n_alt=args.n_alt, a_block=args.a_block, ns_per_day=ns_day, parallelism="replicas only" if world > 1 else "1 GPU",
                            l2="inputs larger than L2 (state + neighbour table >> 126 MB)" if N > 100000 else "inputs smaller than L2",
                            pair_beads_in_cutoff=pair_beads, list_entries=c1["list_entries"]),
                clocks=clk.summary(), e2e=e2e, gpu_launches=int(launches),
                roofline=roofline, kernels=kernels, cpu_baseline=cpu)
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
