#!/usr/bin/env python
"""bench.py -- throughput of the Quantum-HP hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl ours|reference]

A "step" is one pass of the whole hot path (SURVEY.md §8(a) rows R1-R12 for RPMD, Q1-Q7 for adQTB)
over the synthetic water box of the chosen BASELINE.json config: one `qhp_step(1)`.
Default workload C4 = configs[4]: 72,000 waters (216,000 atoms), P = 32 beads, P' = 4 contracted
beads, dt = 0.25 fs, PILE -- the configuration BASELINE.json's metric (bead-atom-steps/s and ns/day at
216k atoms) is quoted on.  The default run appends an adQTB leg (`adqtb`: C3 = configs[3], 216,000 atoms,
one whole 1024-step segment with noise generation and adaptation), so that one run measures both halves of
the metric; `--workload C3` times that configuration alone.

* value     = N_gpus * n_atoms * P * K / (max over ranks of the device time of K steps), state
              resident in HBM.
* e2e       = the same K steps through the host entry points of the C ABI: qhp_set_state_host
              (pinned host -> device), qhp_step(K), qhp_get_state_host + qhp_observables_host
              (device -> host), all inside the timed region.
* roofline  = the dominant kernel (pair forces, FP64-ALU bound): algorithmic flops per launch /
              its average device time, measured with CUDA events recorded by the library on its
              stream around every launch inside the timed region (qhp_profile).
* kernels   = the same for every hot kernel: {ms, algorithmic units, achieved, peak, frac}; the list-rebuild
              chain also carries its amortised cost from an untimed 500-step continuation.
* cpu_baseline = the oracle (oracle/, plain C, one thread) timed on this box's host on 5 steps of a
              bounded sample (4096 waters) of the same workload.
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
# dram__bytes_read.sum + dram__bytes_write.sum of one k_pair_dense<false> / k_pair_staged<false> launch (per launch, like `achieved`) and the
# `ncu --set full` capture it was read from; refreshed whenever the kernel changes (the value is a property of that
# capture, not of this run: `traffic_source` says which)
NCU_TRAFFIC = {("C4", "k_pair_dense"): (9.21201e8 + 2.3565e7, "profiles/r2b_summary.md (prof_r2b_c4, ncu --set full)"),
               ("C3", "k_pair_dense"): (2.30314e8 + 7.261e6, "profiles/r2b_summary.md (prof_r2b_c3, ncu --set full)"),
               ("C4", "k_pair_staged"): (1.363542e9 + 2.4354e7, "profiles/r2_summary.md (prof_r2_hot, ncu --set full)"),
               ("C3", "k_pair_staged"): (3.409152e8 + 7.760e6, "profiles/r2_summary.md (prof_r2_c3, ncu --set full)")}


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


PRUNE_SKIN = None       # --prune-skin: None = the library's default (include/qhp.h qhp_set_pair_prune)


def build_system(cfg: dict):
    import paper_2212_03137_b200 as qhp
    top = W.water_box(cfg["n_mol"])
    kw = {}
    if cfg["thermostat"] == "adqtb":
        kw = dict(n_seg=cfg["n_seg"], a_gamma=cfg["a_gamma"])
    sysg = qhp.System(top, cfg["P"], cfg["P_contract"], cfg["dt_fs"] * 1e-3, W.T_KELVIN, cfg["thermostat"],
                      gamma0=cfg["gamma0"], seed=W.MASTER_SEED, **kw)
    if PRUNE_SKIN is not None:
        sysg.set_pair_prune(PRUNE_SKIN)
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


def time_workload(sysg, cfg, top, x0, p0, K, args, world, local, dist_barrier):
    """Warm-up, then the timed region of K steps with the state resident in HBM; returns the measurements."""
    import torch
    N, P = top["n_atoms"], cfg["P"]
    xd, pd = torch.as_tensor(x0).cuda(), torch.as_tensor(p0).cuda()
    sysg.set_state(xd, pd, 0)
    sysg.step(args.warmup)
    sysg.check()
    c0 = sysg.counters()
    sysg.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        dist_barrier()
        e0.record()
        sysg.step(K)
        e1.record()
        dist_barrier()
    ms = e0.elapsed_time(e1)
    prof = sysg.profile_read()
    prof_pair = sysg.profile_read_pair()
    sysg.profile(False)
    c1 = sysg.counters()
    if c1["overflow"]:
        raise RuntimeError(f"error flags {c1['overflow']} after the timed steps (list overflow / skin / staged region): the timing is void")
    prune = sysg.pair_prune_stats()
    ms = max_over_ranks(ms, world)
    out = dict(ms=ms, prof=prof, prof_pair=prof_pair, prune=prune, c0=c0, c1=c1, clocks=clk.summary(), launches=int(c1["launches"] - c0["launches"]),
               value=job_throughput(world, N, P, K, ms * 1e-3), ns_day=K * cfg["dt_fs"] * 1e-6 / (ms * 1e-3) * 86400.0)
    return out


def e2e_workload(sysg, cfg, top, x0, p0, K, args, world, dist_barrier):
    """The same K steps through the host entry points of the C ABI, copies inside the timed region."""
    import torch
    N, P = top["n_atoms"], cfg["P"]
    xh, ph = torch.as_tensor(x0).pin_memory(), torch.as_tensor(p0).pin_memory()
    xo, po = torch.empty_like(xh).pin_memory(), torch.empty_like(ph).pin_memory()
    sysg.set_state_host(xh, ph, 0)          # untimed pass: allocates the staging buffers
    sysg.step(3 * args.n_alt)
    sysg.get_state_host(xo, po)
    sysg.observables_host()                 # every call of the timed region has run once (lazy module loading, buffers)
    dist_barrier()
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
    return dict(value=job_throughput(world, N, P, K, t_e2e), unit="bead-atom-steps/s",
                h2d_bytes_per_step=2 * nbytes / K, d2h_bytes_per_step=(2 * nbytes + 32) / K,
                ms_total=1e3 * t_e2e, ms_parts=parts, what="set_state_host + qhp_step(K) + get_state_host + observables_host",
                observables=[float(v) for v in obs])


def kernel_blocks(cfg, N, m, pk, dfma_tf, amortised=None):
    """Per-kernel roofline blocks {ms, units, achieved, peak, frac} from the library's per-phase CUDA events."""
    P, Pc, prof, c1, c0 = cfg["P"], cfg["P_contract"], m["prof"], m["c1"], m["c0"]
    per = lambda k: prof[k]["ms"] / max(prof[k]["n"], 1)
    phase_ms, int_ms = per("pair"), per("integrate")
    pair_beads = c1["pair_beads_in_cutoff"]             # ordered (full list): each pair from both sides
    flops = 0.5 * pair_beads * FLOP_PER_PAIR_BEAD       # algorithmic: every unordered pair-bead once
    pp, dense = m.get("prof_pair"), bool(m.get("prune", {}).get("active"))
    if dense:       # pruned-row path: the dominant kernel is k_pair_dense, timed launch by launch inside the pair phase
        kname = "k_pair_dense"
        pair_ms = pp[kname]["ms"] / max(pp[kname]["n"], 1)
    else:
        kname = "k_pair_staged" if c1.get("staged") else "k_pair"
        pair_ms = phase_ms
    ach = flops / (pair_ms * 1e-3) / 1e12 if pair_ms > 0 else 0.0
    tr = NCU_TRAFFIC.get((cfg["name"], kname))
    pair = dict(kernel=kname, bound="alu", ms_per_launch=pair_ms, units=0.5 * pair_beads, unit_name="unordered in-cutoff pair-beads",
                flop_per_unit=FLOP_PER_PAIR_BEAD, achieved=ach, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s", frac=ach / FP64_PEAK_TFLOPS,
                peak_source="derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz", peak_measured=dfma_tf,
                frac_of_measured=ach / dfma_tf if dfma_tf > 0 else None, executed_tflops=2.0 * ach,
                traffic=tr[0] if tr else None, traffic_source=tr[1] if tr else None)
    if dense:
        steps = max(pp[kname]["n"], 1)
        pair["pair_phase"] = dict(ms_per_step=phase_ms, frac_of_phase=flops / (phase_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                                  k_prune_check_ms_per_step=pp["k_prune_check"]["ms"] / steps,
                                  k_prune_ms_per_step=pp["k_prune"]["ms"] / steps,
                                  pruned_entries_per_pair_bead=m["prune"]["entries"] / max(pair_beads, 1),
                                  what="V_s per step = k_prune_check + k_prune (returns at once unless a bead's rows are due) + k_pair_dense")
    if P == 1:      # adQTB / classical step (Q1): 7 x 8 B per DOF + 56 B per atom (pos4 write, Fs read)
        int_bytes, iname = 7.0 * 8 * 3 * N + 56.0 * N, "k_integrate_mol1"
    else:           # fused RPMD pass: 4 x 8 B per (DOF, bead) + (32 + 24) B x P' per atom
        int_bytes, iname = 4.0 * 8 * 3 * N * P + (32.0 + 24.0) * N * Pc, "k_integrate"
    int_gbs = int_bytes / (int_ms * 1e-3) / 1e9 if int_ms > 0 else 0.0
    ks = {kname: pair,
          iname: dict(bound="hbm", ms_per_launch=int_ms, units=int_bytes, unit_name="algorithmic bytes", achieved=int_gbs,
                      peak=pk["hbm_gbs"], unit="GB/s", frac=int_gbs / pk["hbm_gbs"], peak_source=pk["source"]),
          "rebuild_chain": dict(ms_per_step=per("rebuild"), rebuilds=int(c1["rebuilds"] - c0["rebuilds"]),
                                what="cells + contraction + list kernels, enqueued every step (early exit unless a rebuild is due)")}
    if amortised:
        ks["rebuild_chain"]["amortised"] = amortised
    if cfg["thermostat"] == "adqtb" and prof["qtb_generate"]["n"] > 0:
        ns, dof = cfg["n_seg"], 3.0 * N
        gen_ms, ad_ms = per("qtb_generate"), per("qtb_adapt")
        # Q2-Q4 per DOF and segment: 3 n_seg Box-Muller normals (~100 flop) + forward and inverse 4 n_seg-point complex
        # transform (5 n log2 n flop each) shared by the two real sequences of one complex transform
        n4 = 4 * ns
        gflop = dof * (3 * ns * 100.0 + 2 * 5.0 * n4 * np.log2(n4) / 2.0)
        gtf = gflop / (gen_ms * 1e-3) / 1e12 if gen_ms > 0 else 0.0
        ks["k_qtb_noise"] = dict(bound="alu", ms_per_segment=gen_ms, units=gflop, unit_name="flop (SURVEY 8(d): normals + FFT convolution)",
                                 achieved=gtf, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s", frac=gtf / FP64_PEAK_TFLOPS,
                                 bytes_written=dof * ns * 8.0, what="filter + kernel + k_qtb_noise, once per segment")
        sbytes = 2.0 * dof * ns * 8
        sgbs = sbytes / (ad_ms * 1e-3) / 1e9 if ad_ms > 0 else 0.0
        ks["k_qtb_spectra"] = dict(bound="hbm", ms_per_segment=ad_ms, units=sbytes, unit_name="algorithmic bytes (v_seg + F_c read once)",
                                   achieved=sgbs, peak=pk["hbm_gbs"], unit="GB/s", frac=sgbs / pk["hbm_gbs"], peak_source=pk["source"],
                                   what="k_qtb_spectra + reduce + adaptation, once per segment")
    return ks


def cpu_baseline(cfg, n_steps=5, budget_mol=4096):
    """The oracle as it stands, one thread, >= 5 steps of a bounded sample of the workload (the same force field,
    density, P, P', thermostat on a box of at most `budget_mol` waters); setup (initial forces) not timed."""
    import oracle as O
    O.build()
    n_mol = min(cfg["n_mol"], budget_mol)
    top = W.water_box(n_mol)
    x0, p0 = W.initial_state(top, cfg["P"], W.T_KELVIN)
    _, s_per_step = oracle_steps(dict(cfg, n_mol=n_mol), top, x0, p0, n_steps)
    N = 3 * n_mol
    return dict(value=N * cfg["P"] / s_per_step, unit="bead-atom-steps/s", cores=1, kind="oracle",
                sample=f"{n_steps} steps of a {n_mol}-water ({N}-atom) box of the {cfg['name']} workload (P={cfg['P']}, "
                       f"P'={cfg['P_contract']}, {cfg['thermostat']}), {s_per_step:.3f} s/step, setup (initial forces) not timed",
                host_cores_available=os.cpu_count())


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
    ap.add_argument("--prune-skin", type=float, default=None, help="qhp_set_pair_prune: A; <= 0 = the unpruned pre-test pair kernel; default = the library's (0.6)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--shard-beads", action="store_true", help="N > 1: bead-sharded V_s over the ranks (qhp_set_comm, NCCL all-gather of F_s; N must divide P'); "
                    "strong scaling of ONE replica instead of N independent replicas.  Unmeasured on hardware in this round.")
    ap.add_argument("--no-adqtb", action="store_true", help="skip the adQTB (C3) leg that the default C4 run appends")
    ap.add_argument("--no-amortised", action="store_true", help="skip the untimed 500-step run that measures the list-rebuild rate")
    args = ap.parse_args()
    global PRUNE_SKIN
    PRUNE_SKIN = args.prune_skin
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

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    pk = peaks()
    dfma_tf = measure_dfma_peak()

    # ---- primary workload (default C4: the configuration BASELINE.json's metric is quoted on) ------------
    cfg = workload(args.workload)
    if args.n_mol > 0:
        cfg["n_mol"] = args.n_mol
    top, sysg, x0, p0 = build_system(cfg)
    N, P, K = top["n_atoms"], cfg["P"], args.steps
    sharded = args.shard_beads and world > 1 and cfg["P_contract"] % world == 0
    if sharded:
        sysg.set_comm(rank, world)
    if args.a_block != "exact":
        sysg.set_a_block(args.a_block)
    if args.n_alt > 1:
        sysg.set_respa(args.n_alt)
        args.warmup = -(-args.warmup // args.n_alt) * args.n_alt
        args.steps = K = -(-args.steps // args.n_alt) * args.n_alt
    m = time_workload(sysg, cfg, top, x0, p0, K, args, world, local, barrier)
    amortised = None
    if not args.no_amortised and cfg["thermostat"] != "adqtb":
        # list rebuilds are rare events: their rate and cost come from a longer untimed run of the same system
        n_long = -(-500 // args.n_alt) * args.n_alt
        ca = sysg.counters()
        sysg.profile(True)
        sysg.step(n_long)
        pa = sysg.profile_read()
        sysg.profile(False)
        cb = sysg.counters()
        nreb = int(cb["rebuilds"] - ca["rebuilds"])
        amortised = dict(steps=n_long, rebuilds=nreb, rebuilds_per_step=nreb / n_long,
                         ms_per_step=pa["rebuild"]["ms"] / max(pa["rebuild"]["n"], 1),
                         ms_per_step_whole_run=sum(pa[k]["ms"] for k in ("integrate", "rebuild", "pair")) / n_long,
                         what=f"untimed {n_long}-step continuation: rebuild-chain time per step including the rebuilds that fell inside")
    kernels = kernel_blocks(cfg, N, m, pk, dfma_tf, amortised)
    e2e = None if args.no_e2e else e2e_workload(sysg, cfg, top, x0, p0, K, args, world, barrier)
    sysg.check()
    del sysg
    torch.cuda.empty_cache()

    # ---- adQTB leg (C3: 216,000 atoms, one whole 1024-step segment: noise generation, 1024 steps, spectra +
    #      adaptation), appended to the default run so that one driver run measures both halves of the metric ----
    adqtb = None
    if args.workload == "C4" and not args.no_adqtb and args.n_mol == 0 and args.n_alt == 1 and not sharded:
        c3 = workload("C3")
        top3, sys3, x3, p3 = build_system(c3)
        K3 = c3["n_seg"]
        m3 = time_workload(sys3, c3, top3, x3, p3, K3, args, world, local, barrier)
        e3 = None if args.no_e2e else e2e_workload(sys3, c3, top3, x3, p3, K3, args, world, barrier)
        sys3.check()
        adqtb = dict(workload="C3", n_atoms=top3["n_atoms"], steps=K3, value=m3["value"], unit="bead-atom-steps/s",
                     ms_per_step=m3["ms"] / K3, ns_per_day=m3["ns_day"], dt_fs=c3["dt_fs"], n_seg=c3["n_seg"],
                     gpu_launches=m3["launches"], clocks=m3["clocks"], e2e=e3,
                     kernels=kernel_blocks(c3, top3["n_atoms"], m3, pk, dfma_tf),
                     what="one whole segment: coloured-noise generation (Q2-Q4), 1024 BAOAB steps with pair forces and list "
                          "rebuilds (Q1, R7, R8), spectra + gamma adaptation (Q5-Q7)")
        del sys3
        torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- oracle on the host cores (bounded sample of the same workloads) ----------------------------------
    cpu = None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline(cfg)
        if adqtb is not None:
            adqtb["cpu_baseline"] = cpu_baseline(workload("C3"))

    pair_block = next(kernels[k] for k in ("k_pair_dense", "k_pair_staged", "k_pair") if k in kernels)
    roofline = dict(pair_block, note="achieved counts each unordered in-cutoff pair-bead once (110 flop); the kernel "
                                     "evaluates both directions (full list, no atomics), see executed_tflops; "
                                     "peak_measured = live qhp_dfma_probe")
    if sharded:                                   # one replica on all ranks: the job advanced N*P bead-atoms per step, not world times that
        m["value"] /= world
    line = dict(metric="bead_atom_steps_per_s", value=m["value"], unit="bead-atom-steps/s", n_gpus=world, steps=K,
                warmup=args.warmup, ms_per_step=m["ms"] / K, higher_is_better=True, scaling="strong" if sharded else "weak", vs_baseline=None,
                dtype="f64", data="synthetic",
                config=dict(workload=cfg["name"], n_atoms=N, P=P, P_contract=cfg["P_contract"], dt_fs=cfg["dt_fs"],
                            thermostat=cfg["thermostat"], n_alt=args.n_alt, a_block=args.a_block, ns_per_day=m["ns_day"],
                            parallelism=("bead-sharded V_s, all-gather of F_s per step" if sharded else "independent replicas (no data-path collective)") if world > 1 else "1 GPU",
                            l2="inputs larger than L2 (state + neighbour table >> 126 MB)" if N > 100000 else "inputs smaller than L2",
                            pair_beads_in_cutoff=m["c1"]["pair_beads_in_cutoff"], list_entries=m["c1"]["list_entries"]),
                clocks=m["clocks"], e2e=e2e, gpu_launches=m["launches"],
                roofline=roofline, kernels=kernels, adqtb=adqtb, cpu_baseline=cpu)
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
