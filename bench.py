#!/usr/bin/env python
"""bench.py — the headline measurement of the truncated-P2P hot path on B200 (contract: see DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

Metric (BASELINE.json): truncated P2P pair interactions/s (evaluated pairs, the paper's count)
and the fraction of the B200 FP32 FMA peak, fp32 path.  Workload at N=1: BASELINE config 4 (configs[3]),
N = 256^3 clustered particles, N_PM = 256, MAXLEAF = 32 — the configuration north_star quotes its target on.

One "step" is one pass of the whole path over the particle set, as the paper's code does once per time step
(PAPER.md L83-L89): photons_set_particles -> photons_build_leaves (ORB sort, leaf table, interaction list)
-> photons_short_range_acc (the P2P kernel, output in caller order).
  value  : evaluated pairs of all ranks / step time, inputs resident in HBM (device pointers)
  e2e    : the same through the C ABI with HOST buffers: the host->device copy of positions and the
           device->host copy of the accelerations are inside the timed region
  roofline: the dominant kernel (p2p_fp32_kernel) alone, CUDA-event time of its launches
With --gpus N each rank runs an independent replica of the workload (its own seed): the path has no
cross-rank exchange on one node ("replicas only"), scaling = "weak".

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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

from paper_2107_14008_b200 import workloads  # noqa: E402

METRIC = "truncated P2P pair interactions/s (evaluated pairs, fp32 path)"
UNIT = "pairs/s"

# B200 vector peaks: SMs x lanes x 2 flop x max SM clock
SM_COUNT = 148
FP32_LANES_PER_SM = 128
FP64_LANES_PER_SM = 64
POLY_DEGREE = 12               # the library's default (photons_params.poly_degree = 0)
PAPER_FLOPS_PER_PAIR = 51.0


def flops_per_pair(precision: str, g_mode: str, *, poly_degree: int = POLY_DEGREE, table_level: int = 2,
                   table_layout: str = "paper", equal_mass: bool = False) -> float:
    """Executed flops per evaluated pair, counted in the SASS of each kernel's hot loop (profiles/r2_sass_inner_loop.md;
    ncu's op_ffma counters read 0 for the packed FFMA2 stream): FFMA/DFMA = 2, FADD/FMUL/DADD/DMUL = 1, MUFU = 1,
    compares and selects 0.  equal_mass: the fp32 / mixed POLY / TABLE / FUSED kernels that the library takes when all masses
    are equal (photons_params.mass_path = 0) leave the multiply by G m_j out of the pair core: one FMUL per pair less."""
    if equal_mass and precision in ("fp32", "mixed") and g_mode in ("poly", "table", "fused"):
        return flops_per_pair(precision, g_mode, poly_degree=poly_degree, table_level=table_level, table_layout=table_layout) - 1.0
    if precision == "fp64":
        if g_mode == "direct":     # executed per pair on config 4 (ncu DFMA/DMUL/DADD counters): 52.6 + 12.7 + 7.8 + 3 MUFU;
            return 129.0           # the static count is 180, warp votes skip erfc/exp where no lane is inside the cut
        if table_layout == "coef":  # level 4: 15 DFMA + 7 DMUL + 4 DADD + 1 MUFU; one DFMA per level
            return 2.0 * (11 + table_level) + 7 + 4 + 1
        if table_layout == "quad":  # level 4: 16 DFMA + 10 DMUL + 4 DADD + 1 MUFU (the brackets of T[3], T[4] are read)
            return 2.0 * (12 + table_level) + 10 + 4 + 1
        # paper layout: level 4: 20 DFMA + 11 DMUL + 4 DADD + 1 MUFU; level 3: 18 + 10 + 4 + 1
        return {4: 56.0, 3: 51.0}.get(table_level, 51.0 - 4.0 * (3 - table_level))
    if g_mode == "poly":           # (8 + d) FFMA + 3 FADD + 2 FMUL + 1 MUFU.RSQ
        return 2.0 * (8 + poly_degree) + 3 + 2 + 1
    if g_mode == "table":          # level 2: 11 FFMA + 4 FADD + 8 FMUL + 1 MUFU = 35; one FFMA per level
        return 2.0 * 11 + 4 + 8 + 1 + 2.0 * (table_level - 2)
    if g_mode == "fused":          # hand-fused erfc/exp: see profiles/r2_sass_inner_loop.md
        return FUSED_FLOPS_PER_PAIR
    # direct = stock erfcf + expf: 31 FFMA + 16 FMUL + 10 FADD + 5 MUFU (3 FFMA2 + 1.5 FADD2 packed among them)
    return 2.0 * 31 + 16 + 10 + 5


FUSED_FLOPS_PER_PAIR = 2.0 * (7 + 10) + 7 + 3 + 2   # degree 10: 17 FFMA + 7 FMUL + 3 FADD + MUFU.RSQ + MUFU.EX2


def peak_tflops(precision: str, sm_mhz: float) -> float:
    lanes = FP64_LANES_PER_SM if precision == "fp64" else FP32_LANES_PER_SM
    return SM_COUNT * lanes * 2 * sm_mhz * 1e6 / 1e12


def ncu_traffic(workload: str, maxleaf: int, precision: str, g_mode: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed `ncu --set
    full` summaries (profiles/r2_traffic.csv, each row naming its capture and commit); null when this variant has
    none.  Never a number typed in here."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.csv"), newline="") as f:
            rows = {r[0]: r for r in csv.reader(f)}
    except OSError:
        return None, None
    r = rows.get(f"{workload}/{maxleaf}/{precision}/{g_mode}")
    return (float(r[1]), r[2]) if r else (None, None)


def geometry(cfg):
    r_s = 1.2 * cfg.boxsize / cfg.n_pm
    return r_s, 6.0 * r_s                   # r_cut = 6 r_s (north_star)


# close_pair_radius (in r_cut) of the fp32 kernels' exact path (A12), per workload kind: a staged run whose fp32
# partial acceleration exceeds G m / r_close^2 is redone in fp64.  The literal criterion max|da| <= 1e-5 rms needs it on
# every load: the fp32 pair core is good to ~6e-7 relative (three times the rsqrt's 2 ulp), so a target whose
# acceleration exceeds ~15 rms misses 1e-5 rms without it (config 4 at 10^4 targets: 2.1e-5 at |a| = 36 rms).  The radii
# put the trigger at a few rms: uniform-like loads (rms ~ 32 G m / spacing^2) 0.02 r_cut = 2.9 rms; clustered loads, whose
# rms is set by the dense cores, 5e-4 r_cut = 3-8 rms.  A run is redone for well under 1 % of the targets.
CLOSE_OVER_RCUT = {"uniform": 0.02, "grid": 0.02, "clustered": 5e-4}


def headline_params(cfg, **over):
    """The launch configuration this file times (also used by tests/test_gpu_parity.py at full size)."""
    _, r_cut = geometry(cfg)
    p = dict(boxsize=cfg.boxsize, n_pm=cfg.n_pm, G=cfg.G, maxleaf=cfg.maxleaf, precision="fp32", g_mode="poly",
             close_pair_radius=CLOSE_OVER_RCUT[cfg.kind] * r_cut, n_streams=1)
    p.update(over)
    return p


# ------------------------------------------------------------------------------------------ helpers

class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.th.join(timeout=2)

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        busy = [s for s, p in zip(sm, pw) if p > 0.5 * max(pw)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


def aggregate(local_ms: float, local_units: float, dist=None):
    """Whole-job figures from per-rank ones: time = MAX over ranks, units = SUM over ranks.
    Works on any torch.distributed backend (NCCL on the GPUs, gloo in the CPU test)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except OSError:
        return {}


def rank_config(cfg, rank: int):
    """Rank r's replica: the same recipe with its own seed (independent problems, no exchange)."""
    import dataclasses
    return cfg if rank == 0 else dataclasses.replace(cfg, seed=cfg.seed + 100_000 * rank)


# ----------------------------------------------------------------------------------- reference arm

def oracle_sample(cfg, pos, mass, seconds_target: float, n_threads_hint: int):
    """Time the oracle as it stands on a bounded sample: a seeded subset of targets against all N sources.
    Returns (pair tests, within-cut pairs, seconds, n_targets)."""
    import oracle
    oracle.build()
    r_s, r_cut = geometry(cfg)
    # ~1.3e8 pair tests per second per core (measured on the first run; only sets the sample size).  The oracle hands
    # out targets in chunks of 16 (schedule(dynamic, 16)): a whole number of rounds of chunks over the threads, and at
    # least four rounds, so that the measured rate does not depend on the sample size (load balance).
    quantum = 16 * max(1, n_threads_hint)
    n_t = int(seconds_target * 1.3e8 * n_threads_hint / cfg.n)
    n_t = min(cfg.n, max(4 * quantum, (n_t + quantum - 1) // quantum * quantum))
    tgt = workloads.sample_targets(cfg.n, n_t, cfg.seed)
    t0 = time.perf_counter()
    _, cnt = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G)
    dt = time.perf_counter() - t0
    return cnt["pair_tests"], cnt["pairs_in_cut"], dt, len(tgt)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    cfg = workloads.CONFIGS[args.config]
    pos, mass = workloads.make(cfg)
    cores = oracle.num_threads()
    per_step = max(2.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(cfg, pos, mass, per_step, cores)
    tests = incut = secs = 0.0
    n_t = 0
    for _ in range(args.steps):
        a, b, dt, n_t = oracle_sample(cfg, pos, mass, per_step, cores)
        tests += a; incut += b; secs += dt
    value = tests / secs
    sample = f"{n_t} seeded targets x all {cfg.n} sources per step (fp64 minimum-image direct sum, pair tests counted)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "n_particles": cfg.n, "n_pm": cfg.n_pm, "maxleaf": cfg.maxleaf,
                   "note": "CPU oracle; its unit of work is the pair TEST (every target against all N sources)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "within_cut_pairs_per_s": incut / secs},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------- our arm

def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2107_14008_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.load()

    cfg0 = workloads.CONFIGS[args.config]
    cfg = rank_config(cfg0, rank)
    r_s, r_cut = geometry(cfg)
    pos, mass = workloads.make(cfg)              # flavour F: positions on the fp32 grid (A20)
    pos32 = pos.astype(np.float32)               # exact: the caller's data are fp32
    params = headline_params(cfg, device=local, n_streams=args.streams, g_mode=args.g_mode,
                             precision=args.precision, maxleaf=args.maxleaf or cfg.maxleaf)
    if args.g_mode == "table":
        params.update(table_nodes=args.table_nodes, table_level=args.table_level, table_layout=args.table_layout)
    if args.softening_over_rcut:
        params["softening"] = args.softening_over_rcut * r_cut
    if args.warps_per_leaf:
        params["warps_per_leaf"] = args.warps_per_leaf
    if args.targets_per_lane:
        params["targets_per_lane"] = args.targets_per_lane
    if args.chunk_max:
        params["chunk_max"] = args.chunk_max
    if args.leaf_order:
        params["leaf_order"] = args.leaf_order
    if args.mass_path:
        params["mass_path"] = args.mass_path
    if args.no_close or args.precision == "fp64":
        params["close_pair_radius"] = 0.0
    n = cfg.n

    d_pos = torch.from_numpy(pos32).cuda()
    d_acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    h_pos = torch.from_numpy(pos32).pin_memory()
    h_acc = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    stream = torch.cuda.current_stream()

    ph = B.Photons(**params)
    ph.set_stream(stream)

    def step_device():
        ph.set_particles(d_pos, None, stream=stream.cuda_stream)
        ph.build_leaves()
        return ph.short_range_acc(d_acc)

    def step_host():
        ph.set_particles(h_pos, None, stream=stream.cuda_stream)
        ph.build_leaves()
        return ph.short_range_acc(h_acc)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(step, steps):
        k_ms, b_ms, st = [], [], None
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = ph.stats()["kernel_launches"]
        barrier()
        e0.record(stream)
        for _ in range(steps):
            st = step()
            k_ms.append(st["kernel_ms"]); b_ms.append(st["build_ms"])
        e1.record(stream)
        barrier()
        return e0.elapsed_time(e1), k_ms, b_ms, st, ph.stats()["kernel_launches"] - l0

    for _ in range(args.warmup):
        step_device()
    with ClockSampler(local) as clk:
        ms, k_ms, b_ms, st, launches = timed(step_device, args.steps)
    pairs = float(st["pairs_evaluated"])
    ms_max, units = aggregate(ms, pairs * args.steps, dist if world > 1 else None)
    value = units / (ms_max * 1e-3)

    # end to end through the C ABI with host buffers
    e_steps = max(1, min(args.steps, 3))
    if args.no_e2e:          # profiling runs only: the bench line then carries no end-to-end number
        e_ms_max, e2e_value = float("nan"), None
    else:
        for _ in range(min(args.warmup, 2)):
            step_host()
        e_ms, _, _, _, _ = timed(step_host, e_steps)
        e_ms_max, e_units = aggregate(e_ms, pairs * e_steps, dist if world > 1 else None)
        e2e_value = e_units / (e_ms_max * 1e-3)

    line = None
    if rank == 0:
        kernel_ms = float(np.mean(k_ms))
        # (the synthetic workloads have one particle species: mass = NULL = 1/n each)
        fpp = flops_per_pair(args.precision, args.g_mode, table_level=args.table_level, table_layout=args.table_layout,
                             equal_mass=not args.mass_path)
        clocks = clk.summary()
        peak_tf = peak_tflops(args.precision, clocks["sm_max_mhz"] or 1965.0)
        achieved_tf = pairs * fpp / (kernel_ms * 1e-3) / 1e12
        traffic, traffic_src = ncu_traffic(cfg0.name, params["maxleaf"], args.precision, args.g_mode)
        # a row stands for the kernel it was captured on: equal-mass or G m_j per pair
        eq_kernel = not args.mass_path and args.precision in ("fp32", "mixed") and args.g_mode != "direct"
        if traffic_src and args.precision != "fp64" and args.g_mode != "direct" and ("equal-mass kernel" in traffic_src) != eq_kernel:
            traffic, traffic_src = None, None
        f64 = args.precision == "fp64"
        roofline = {
            "bound": "alu", "kernel": "p2p_fp64_kernel" if f64 else "p2p_fp32_kernel", "achieved": achieved_tf, "peak": peak_tf,
            "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
            "traffic": traffic, "traffic_source": traffic_src,
            "traffic_unit": "bytes per launch (ncu dram read + write; the bound is ALU, not HBM)",
            "peak_source": f"derived: 148 SMs x {FP64_LANES_PER_SM if f64 else FP32_LANES_PER_SM} FP{'64' if f64 else '32'} lanes x 2 flop x "
                           "clocks.max.sm (DESIGN.md §7); MEASURED_PEAKS.json holds no vector-ALU peak; photons_peak_probe measures "
                           "0.89-0.91 (FFMA, FFMA2) and 0.87 (DFMA) of it (profiles/r2_peak_probe.md)",
            "flops_per_pair": fpp, "kernel_ms": kernel_ms, "kernel_pairs_per_s": pairs / (kernel_ms * 1e-3),
            "kernel_share_of_step": kernel_ms / (ms / args.steps),
            "frac_at_sampled_clock": (achieved_tf / peak_tflops(args.precision, clocks["sm_mhz"]) if clocks["sm_mhz"] else None),
            "paper_convention_tflops": pairs * PAPER_FLOPS_PER_PAIR / (kernel_ms * 1e-3) / 1e12,
        }
        # CPU baseline: the oracle on a bounded sample of the same workload, all host cores
        cpu = None
        within_cut_total = None
        if not args.no_cpu_baseline:
            import oracle
            cores = oracle.num_threads()
            tests, incut, secs, n_t = oracle_sample(cfg, pos, mass, 15.0, cores)
            cpu = {"value": tests / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"{n_t} seeded targets x all {n} sources, {secs:.1f} s (pair tests counted; "
                             f"within-cut pairs/s = {incut / secs:.3e})",
                   "within_cut_pairs_per_s": incut / secs}
            within_cut_total = incut / n_t * n       # the sample's mean in-cut neighbour count x N
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if args.precision != "fp64" else "f64", "data": "synthetic",
            "config": {"workload": cfg0.name, "n_particles": n, "n_pm": cfg.n_pm, "maxleaf": params["maxleaf"],
                       "precision": args.precision, "g_mode": args.g_mode, "close_pair_radius_over_rcut": params["close_pair_radius"] / r_cut,
                       "n_streams": args.streams, "input_flavour": "F (fp32-grid positions)",
                       "masses": "equal (one particle species, mass = NULL); " + ("G m_j per pair forced (mass_path 1)" if args.mass_path or args.precision == "fp64" or args.g_mode == "direct"
                                                                                   else "equal-mass kernels: G m applied once per staged run (mass_path 0)"),
                       "l2": "inputs exceed L2 (leaf-sorted particles + interaction list > 126 MB); no flush",
                       "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                       "step": "set_particles + build_leaves + short_range_acc"},
            "pairs_evaluated_per_step": pairs, "n_leaf_pairs": st["n_leaf_pairs"], "n_chunks": st["n_chunks"],
            "build_ms": float(np.mean(b_ms)), "kernel_ms": kernel_ms,
            # evaluated pairs/s alone rewards large leaves; these two do not
            "time_to_solution_ms": ms_max / args.steps,
            "within_cut_pairs_per_s": (within_cut_total * world / (ms_max / args.steps * 1e-3)) if within_cut_total else None,
            "e2e": None if e2e_value is None else
                   {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h_pos.numel() * 4),
                    "d2h_bytes_per_step": int(h_acc.numel() * 4), "ms_per_step": e_ms_max / e_steps},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
    ph.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ sweep (config 4)

def run_sweep(args):
    """BASELINE config 4's sweep: MAXLEAF 16/32/64/128 x g evaluated directly / from tables of 256, 512 (the
    paper's), 1024, 4096 nodes / by the polynomial, fp32 vs mixed vs fp64.  Kernel-only times (CUDA events),
    error against the oracle on sampled targets.  Prints a markdown table (see profiles/)."""
    import torch
    import oracle
    from paper_2107_14008_b200 import binding as B
    cfg = workloads.CONFIGS[args.config]
    r_s, r_cut = geometry(cfg)
    pos, mass = workloads.make(cfg)
    tgt = workloads.sample_targets(cfg.n, args.sweep_targets, cfg.seed)
    ref, cnt = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G)
    rms = float(np.sqrt((ref ** 2).sum(axis=1).mean()))
    in_cut_per_particle = cnt["pairs_in_cut"] / len(tgt)
    d_pos = torch.from_numpy(pos.astype(np.float32)).cuda()
    d_tgt = torch.from_numpy(tgt).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    close = CLOSE_OVER_RCUT[cfg.kind] * r_cut
    variants = [("fp32", "direct", {}), ("fp32", "fused", {}), ("fp32", "poly", {})]
    variants += [("fp32", "poly", dict(poly_degree=d)) for d in (10, 11, 13)]      # the default is 12
    variants += [("fp32", "table", dict(table_nodes=n, table_level=2)) for n in (256, 512, 1024, 4096)]
    variants += [("fp32", "table", dict(table_nodes=512, table_level=lv)) for lv in (0, 1, 3)]
    variants += [("mixed", "direct", {}), ("mixed", "poly", {}), ("mixed", "table", dict(table_nodes=512, table_level=2))]
    variants += [("fp64", "direct", {}), ("fp64", "table", dict(table_nodes=512, table_level=4)),
                 ("fp64", "table", dict(table_nodes=512, table_level=4, table_layout="coef")),
                 ("fp64", "table", dict(table_nodes=512, table_level=4, table_layout="quad")),
                 ("fp64", "table", dict(table_nodes=4096, table_level=3)),
                 ("fp64", "table", dict(table_nodes=4096, table_level=3, table_layout="coef"))]
    peak32 = SM_COUNT * FP32_LANES_PER_SM * 2 * 1.965e9
    print(f"# sweep on {cfg.name}: N = {cfg.n}, N_PM = {cfg.n_pm}, close_pair_radius = {close / r_cut:g} r_cut, "
          f"oracle on {len(tgt)} sampled targets (rms |a| = {rms:.4g}, {in_cut_per_particle:.0f} in-cut pairs per particle)\n")
    print("| MAXLEAF | precision | g | evaluated pairs | kernel ms | pairs/s | in-cut pairs/s | paper-convention TFLOP/s (x51) "
          "| % of fp32 peak (x51) | max err / rms |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for maxleaf in (16, 32, 64, 128):
        for prec, g, extra in variants:
            if args.sweep_quick and (maxleaf != 32 and (g == "table" and extra.get("table_nodes") != 512 or extra.get("table_level", 2) != 2)):
                continue
            if "poly_degree" in extra and maxleaf != 32:
                continue
            params = headline_params(cfg, maxleaf=maxleaf, precision=prec, g_mode=g, close_pair_radius=close if prec != "fp64" else 0.0, **extra)
            with B.Photons(**params) as ph:
                ph.set_particles(d_pos, None)
                ph.build_leaves()
                ks = [ph.short_range_acc(out)["kernel_ms"] for _ in range(2 if prec != "fp64" else 1)]
                st = ph.stats()
            a = out[d_tgt].cpu().numpy()
            err = float(np.sqrt(((a - ref) ** 2).sum(axis=1)).max() / rms)
            ms = min(ks)
            rate = st["pairs_evaluated"] / (ms * 1e-3)
            gname = (g + (f" degree {extra['poly_degree']}" if "poly_degree" in extra else "")) if g != "table" else f"table {extra['table_nodes']} / T[{extra['table_level']}]" + (" " + extra["table_layout"] if extra.get("table_layout") else "")
            print(f"| {maxleaf} | {prec} | {gname} | {st['pairs_evaluated']:.4g} | {ms:.2f} | {rate:.3e} | "
                  f"{in_cut_per_particle * cfg.n / (ms * 1e-3):.3e} | {rate * PAPER_FLOPS_PER_PAIR / 1e12:.1f} | "
                  f"{100 * rate * PAPER_FLOPS_PER_PAIR / peak32:.1f} | {err:.2e} |", flush=True)
    return 0


def run_streams_study(args):
    """a10 ("concurrency management"): the same step with target-leaf batches on 1, 2 and 4 CUDA streams:
    P2P kernel time (CUDA events around all batches), whole device-resident step, and the host-buffer step."""
    import torch
    from paper_2107_14008_b200 import binding as B
    cfg = workloads.CONFIGS[args.config]
    pos, _ = workloads.make(cfg)
    pos32 = pos.astype(np.float32)
    del pos
    d_pos = torch.from_numpy(pos32).cuda()
    h_pos = torch.from_numpy(pos32).pin_memory()
    d_acc = torch.empty((cfg.n, 3), dtype=torch.float32, device="cuda")
    h_acc = torch.empty((cfg.n, 3), dtype=torch.float32).pin_memory()
    stream = torch.cuda.current_stream()
    print(f"# streams study on {cfg.name}: N = {cfg.n}, MAXLEAF = {cfg.maxleaf}, precision {args.precision}, g {args.g_mode}; "
          f"median of {args.steps} steps after {args.warmup} warm-ups\n")
    print("| n_streams | kernel ms | build ms | device-resident step ms | host-buffer step ms |")
    print("|---|---|---|---|---|")
    for ns in (1, 2, 4, 8):
        with B.Photons(**headline_params(cfg, precision=args.precision, g_mode=args.g_mode, n_streams=ns)) as ph:
            ph.set_stream(stream)
            res = {}
            for name, src, dst in (("dev", d_pos, d_acc), ("host", h_pos, h_acc)):
                ks, bs, ts = [], [], []
                for it in range(args.warmup + args.steps):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize()
                    e0.record(stream)
                    ph.set_particles(src, None, stream=stream.cuda_stream)
                    ph.build_leaves()
                    st = ph.short_range_acc(dst)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    if it >= args.warmup:
                        ks.append(st["kernel_ms"]); bs.append(st["build_ms"]); ts.append(e0.elapsed_time(e1))
                res[name] = (float(np.median(ks)), float(np.median(bs)), float(np.median(ts)))
        print(f"| {ns} | {res['dev'][0]:.2f} | {res['dev'][1]:.2f} | {res['dev'][2]:.2f} | {res['host'][2]:.2f} |", flush=True)
    return 0


def run_m2l(args):
    """Truncated M2L: cell pairs per second of photons_m2l at order p on a periodic lattice
    of n^3 cells (jittered centres, cell = 1 PM cell so r_s = 1.2 cells), every target taking the 316 sources at Chebyshev
    distance 2..3 - the shape of an FMM interaction list ("children of the parent's neighbours"); random multipoles.
    Parity of the same call is in tests/test_gpu_m2l.py; the oracle leg times oracle/m2l.py on a bounded sample."""
    import torch
    from paper_2107_14008_b200 import binding as B
    n, p = args.m2l_cells, args.m2l_order
    rng = np.random.default_rng(77)
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    centres = (g + 0.5 + 0.2 * (rng.random((n ** 3, 3)) - 0.5)) / n
    off = np.array([(i, j, k) for i in range(-3, 4) for j in range(-3, 4) for k in range(-3, 4) if max(abs(i), abs(j), abs(k)) >= 2])
    nb = g[:, None, :] + off[None, :, :]
    shift = np.floor_divide(nb, n).astype(np.int8)            # source moved by this many box lengths
    nbw = np.mod(nb, n)
    src = (nbw[..., 0] * n * n + nbw[..., 1] * n + nbw[..., 2]).astype(np.int32).reshape(-1)
    ptr = np.arange(0, (n ** 3 + 1) * len(off), len(off), dtype=np.int64)
    nc = B.m2l_n_coeffs(p)
    M = rng.normal(size=(n ** 3, nc)) * (0.4 / n) ** np.array([sum(q) for q in _m2l_indices(p)])
    r_s = 1.2 / n
    d = [torch.from_numpy(x).cuda() for x in (centres, M, ptr, src, np.ascontiguousarray(shift.reshape(-1, 3)))]
    out = torch.empty((n ** 3, nc), dtype=torch.float64, device="cuda")
    ms = []
    for it in range(args.warmup + args.steps):
        _, t = B.m2l(d[0], d[1], d[2], d[3], d[4], p=p, r_s=r_s, boxsize=1.0, out=out)
        if it >= args.warmup:
            ms.append(t)
    n_pairs = len(src)
    k_ms = float(np.median(ms))
    flops = {4: 749.0}.get(p)          # SASS count of m2l_kernel<4> (profiles/r2_sass_inner_loop.md)
    line = {"metric": "truncated M2L cell pairs/s", "value": n_pairs / (k_ms * 1e-3), "unit": "cell pairs/s", "order_p": p, "n_cells": n ** 3,
            "n_pairs": n_pairs, "kernel_ms": k_ms, "dtype": "f64",
            "roofline": None if flops is None else {"bound": "alu", "achieved": n_pairs * flops / (k_ms * 1e-3) / 1e12, "peak": peak_tflops("fp64", 1965.0),
                                                    "unit": "TFLOP/s", "frac": n_pairs * flops / (k_ms * 1e-3) / 1e12 / peak_tflops("fp64", 1965.0),
                                                    "flops_per_pair": flops}}
    if not args.no_cpu_baseline:
        import oracle
        import time
        tsel = rng.choice(n ** 3, size=min(n ** 3, 2000), replace=False)
        pairs = np.stack([np.repeat(tsel, len(off)), src.reshape(-1, len(off))[tsel].reshape(-1)], axis=1)
        sh = shift.reshape(-1, len(off), 3)[tsel].reshape(-1, 3)
        t0 = time.perf_counter()
        ref = oracle.m2l.m2l(centres, M, pairs, p, r_s, boxsize=1.0, shifts=sh)
        dt = time.perf_counter() - t0
        got = out.cpu().numpy()
        err = float((np.abs(got[tsel] - ref[tsel]).max(axis=0) / np.abs(ref[tsel]).max(axis=0)).max())
        line["cpu_baseline"] = {"value": len(pairs) / dt, "unit": "cell pairs/s", "cores": 1, "kind": "oracle",
                                "sample": f"{len(tsel)} target cells x {len(off)} sources (numpy fp64)"}
        line["max_rel_err_vs_oracle"] = err
    print(json.dumps(line))
    return 0


def _m2l_indices(p):
    return [(nx, ny, k - nx - ny) for k in range(p + 1) for nx in range(k, -1, -1) for ny in range(k - nx, -1, -1)]


def run_table_study(args):
    """Eq. 2 study (Fig. 2): every table size x Taylor level, fp32 and fp64, on one workload:
    force error against the oracle and kernel time.  Prints a markdown table (see profiles/)."""
    import torch
    import oracle
    from paper_2107_14008_b200 import binding as B
    cfg = workloads.CONFIGS[args.config]
    r_s, r_cut = geometry(cfg)
    pos, mass = workloads.make(cfg)
    tgt = workloads.sample_targets(cfg.n, args.sweep_targets, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G)
    rms = float(np.sqrt((ref ** 2).sum(axis=1).mean()))
    d_pos = torch.from_numpy(pos.astype(np.float32)).cuda()
    d_tgt = torch.from_numpy(tgt).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    close = CLOSE_OVER_RCUT[cfg.kind] * r_cut
    print(f"# Eq. 2 table study on {cfg.name}: N = {cfg.n}, MAXLEAF = {cfg.maxleaf}, oracle on {len(tgt)} sampled targets\n")
    print("| precision | nodes | level | max table error of T (fp64, oracle/table.py) | max err / rms of the force | kernel ms | pairs/s |")
    print("|---|---|---|---|---|---|---|")
    xq = np.linspace(0.0, 3.0, 200001)
    t_exact = oracle.oracle_T(np.linspace(0.0, 3.0, 2001))
    for prec in ("fp32", "fp64"):
        for nodes in (256, 512, 1024, 4096):
            for level in range(0, 4 if prec == "fp32" else 5):
                tab_err = float(np.abs(oracle.eval_table(np.linspace(0.0, 3.0, 2001), nodes, level) - t_exact).max())
                params = headline_params(cfg, precision=prec, g_mode="table", table_nodes=nodes, table_level=level,
                                         close_pair_radius=close if prec != "fp64" else 0.0)
                with B.Photons(**params) as ph:
                    ph.set_particles(d_pos, None)
                    ph.build_leaves()
                    ks = [ph.short_range_acc(out)["kernel_ms"] for _ in range(2 if prec != "fp64" else 1)]
                    st = ph.stats()
                a = out[d_tgt].cpu().numpy()
                err = float(np.sqrt(((a - ref) ** 2).sum(axis=1)).max() / rms)
                print(f"| {prec} | {nodes} | T[{level}] | {tab_err:.2e} | {err:.2e} | {min(ks):.2f} | "
                      f"{st['pairs_evaluated'] / (min(ks) * 1e-3):.3e} |", flush=True)
    del xq
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=sorted(workloads.CONFIGS))
    ap.add_argument("--precision", default="fp32", choices=["fp32", "mixed", "fp64"])
    ap.add_argument("--g-mode", dest="g_mode", default="poly", choices=["poly", "table", "direct", "fused"])
    ap.add_argument("--table-nodes", type=int, default=512)
    ap.add_argument("--table-level", type=int, default=2)
    ap.add_argument("--table-layout", default="paper", choices=["paper", "coef", "quad"])
    ap.add_argument("--softening-over-rcut", type=float, default=0.0)
    ap.add_argument("--warps-per-leaf", type=int, default=0)
    ap.add_argument("--chunk-max", type=int, default=0, help="longest staged run in source slots (0 = the library default)")
    ap.add_argument("--targets-per-lane", type=int, default=0, help="register tiling of the fp32 kernels (0 = the default of the leaf size)")
    ap.add_argument("--leaf-order", type=int, default=0, choices=[0, 1], help="0 = ORB order (default), 1 = longest source list first")
    ap.add_argument("--mass-path", type=int, default=0, choices=[0, 1],
                    help="0 = equal masses take the kernels that apply G m once per run (default), 1 = always G m_j per pair")
    ap.add_argument("--maxleaf", type=int, default=0)
    ap.add_argument("--streams", type=int, default=1)
    ap.add_argument("--no-close", action="store_true", help="switch the exact close-pair path off")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (ncu captures)")
    ap.add_argument("--streams-study", action="store_true", help="kernel and step time for 1/2/4 streams (a10)")
    ap.add_argument("--m2l", action="store_true", help="truncated M2L kernel (SURVEY §8(f) 4) instead of the P2P bench line")
    ap.add_argument("--m2l-cells", type=int, default=48, help="cells per side of the M2L lattice")
    ap.add_argument("--m2l-order", type=int, default=4)
    ap.add_argument("--sweep", action="store_true", help="MAXLEAF x g-mode x precision table instead of the bench line")
    ap.add_argument("--table-study", action="store_true", help="Eq. 2: table size x Taylor level, fp32 and fp64")
    ap.add_argument("--sweep-targets", type=int, default=1000)
    ap.add_argument("--sweep-quick", action="store_true", help="all table sizes/levels only at MAXLEAF 32")
    args = ap.parse_args(argv)
    if args.steps < 1 or args.warmup < 0:
        ap.error("--steps >= 1 and --warmup >= 0")
    if args.precision == "fp64" and args.g_mode in ("poly", "fused"):
        args.g_mode = "direct"           # POLY and FUSED are fp32 approximations
    if args.m2l:
        return run_m2l(args)
    if args.streams_study:
        return run_streams_study(args)
    if args.sweep:
        return run_sweep(args)
    if args.table_study:
        return run_table_study(args)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
