#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract: task prompt, "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1..5}] [--impl ours|reference]

A STEP is one pass of the whole hot path over one synthetic batch.  Default
workload = BASELINE.json configs[2] ("config 3"): fp32, N = 131072, uniform positions at 5 %
volume fraction; the step is lm_set_positions + lm_hydrodynamic_velocities(F, W, tol = 1e-3), i.e.
one deterministic M.F plus the Lanczos sqrt(M).W (one pair-kernel launch per iteration) -- the
configuration the north_star quotes its fp32 target on (N >= 131072).  Configs 1, 2, 4, 5 are
selectable for measurement (`--config`), their step is set_positions + lm_mdot / lm_mdot_batch.

value   = ordered pair interactions evaluated per second (N^2 per pair-kernel launch; all right-hand
          sides of a batched launch share one pair count), whole job, device-resident inputs,
          CUDA-event time of each step on the launching stream, max over ranks.
e2e     = same metric through the *_host C-ABI calls: pinned host buffers, H2D and D2H copies inside
          the timed region.
roofline= the pair kernel against the FP32/FP64 FMA-pipe ("alu") roofline, DESIGN.md sec. 7.
cpu_baseline = the CPU fp64 oracle (oracle/, untuned) on the box's host cores, bounded row sample.

Multi-GPU (torchrun): the path does not shard in this build ("replicas only"):
every rank runs an independent replica (seed + rank); scaling = "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "rpy_pair_interactions_per_s"
UNIT = "Gpairs/s"

# Algorithmic FP-pipe lane-operations and flops per ordered pair (counted from the
# algebra of a far-field pair, never from emitted instructions; an overlapping pair needs fewer).
#   translational: d 3, r^2 3, u = s^2 and s^3 2, f 1, g 2 -> 11;  per right-hand side: d.F 3, t 1, U += fF + td 6 -> 10
#   angular      : + s^5 1, f_rr 1, g_rr 1, h d 3, g one fewer -> 16;  per right-hand side: d.F, d.T 6, t, s 2, 24 FMAs -> 32
def work_per_pair(angular: bool, nrhs: int, f64: bool):
    if angular:
        instr, fma = 16 + 32 * nrhs, 4 + 28 * nrhs
    else:
        instr, fma = 11 + 10 * nrhs, 4 + 8 * nrhs
    if f64:
        instr, fma = instr + 5, fma + 3      # fp64 refinement of the rsqrt seed
    flops = instr + fma + 1                  # FMA = 2 flops, + the rsqrt
    return instr, flops


# DRAM traffic of ONE pair-kernel launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed
# `ncu --set full` captures profiles/r1_c<N>_pair_kernel_ncu_full.md (same launch configuration); it is a
# recorded profile value, not measured by this run.  Configs 4 and 5 are dominated by the j-split partials.
NCU_DRAM_BYTES_PER_LAUNCH = {1: 64512 + 0, 2: 610816 + 0, 3: 3.16595e+06 + 3.64288e+06, 4: 1.964e+08 + 1.24312e+09, 5: 2.74117e+07 + 1.13751e+08}


def nominal_lanes(f64: bool) -> int:
    return 64 if f64 else 128                # FP64 / FP32 FMA lanes per SM (B200)


# ---------------------------------------------------------------- clocks sampler
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows = []
        self.proc = None
        self.gpu_index = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows]
        for r in rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[0])); smax.append(float(p[1])); power.append(float(p[2]))
            except ValueError:
                continue
            for name, val in zip(names, p[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------- CPU oracle legs
def oracle_rate(data, target_seconds: float):
    """Time the oracle (as it stands) on a bounded row sample of this workload: rows are independent,
    so `nrows` target rows against all N sources are exact for those rows.  Returns a dict."""
    from oracle import rpy
    cfg, N = data["cfg"], data["N"]
    F = data["forces"] if cfg.nrhs == 1 else data["forces"][0]
    T = data["torques"]
    rng = np.random.default_rng(12345)
    probe_rows = np.sort(rng.choice(N, min(N, 64), replace=False))
    t0 = time.perf_counter()
    rpy.mdot_rows(data["pos"], probe_rows, F, T, angular=cfg.angular)
    dt = max(time.perf_counter() - t0, 1e-6)
    nrows = int(min(N, max(64, probe_rows.size * target_seconds / dt)))
    rows = np.sort(rng.choice(N, nrows, replace=False))
    t0 = time.perf_counter()
    rpy.mdot_rows(data["pos"], rows, F, T, angular=cfg.angular)
    dt = time.perf_counter() - t0
    return {"pairs": float(nrows) * N, "seconds": dt, "nrows": nrows, "cores": int(rpy.mdot_rows.last_threads)}


def run_reference(args, data):
    """--impl reference: the oracle, as it stands, on the host cores, on this arm's config and metric.
    Each step is a bounded row sample (exact for its rows); rank 0 only."""
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(min(args.warmup, 1)):
        oracle_rate(data, 1.0)
    pairs = secs = 0.0
    info = None
    for _ in range(args.steps):
        info = oracle_rate(data, per_step)
        pairs += info["pairs"]
        secs += info["seconds"]
    cfg = data["cfg"]
    val = pairs / secs / 1e9
    sample = f"{info['nrows']} sampled target rows x all {data['N']} sources per step (fp64 double loop, OpenMP over rows)"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(cfg, data["N"], None),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": info["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def config_dict(cfg, N, extra):
    d = {"workload": f"BASELINE.json configs[{cfg.index - 1}] ({cfg.name})", "op": cfg.op, "N": int(N), "precision": cfg.precision,
         "include_angular": bool(cfg.angular), "nrhs": int(cfg.nrhs), "geometry": f"{cfg.geometry}={cfg.geom_param:g}", "seed": int(cfg.seed),
         "a": cfg.a, "eta": cfg.eta}
    if cfg.tol:
        d["lanczos_tol"] = cfg.tol
    if extra:
        d.update(extra)
    return d


# ---------------------------------------------------------------- the CUDA arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--N", type=int, default=None, help="override N (measurement sweeps only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "sharded"],
                    help="N > 1 ranks: independent replicas (default, weak scaling) or ONE problem row-sharded over the ranks "
                         "(lm_dist_init: all-gather of the row blocks inside every apply, strong scaling)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from paper_2510_02135_b200 import workloads

    if args.impl == "reference":
        if rank != 0:
            return 0
        run_reference(args, workloads.generate(args.config, args.N))
        return 0

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if args.warmup < 3:
        args.warmup = 3

    import paper_2510_02135_b200 as lm

    from paper_2510_02135_b200 import multi
    cfg = workloads.CONFIGS[args.config]
    sharded = args.parallelism == "sharded" and world > 1
    # replicas: every rank its own problem (seed + 1000 rank); sharded: the same problem on every rank
    data = workloads.generate(args.config, args.N, seed=cfg.seed if sharded else multi.replica_seed(cfg.seed, rank))
    N = data["N"]
    f64 = cfg.precision == "f64"
    tdt = torch.float64 if f64 else torch.float32
    dof = (6 if cfg.angular else 3) * N
    stream = torch.cuda.current_stream()

    solver = lm.Solver(cfg.precision, N, cfg.eta, cfg.a, cfg.angular)
    if sharded:
        multi.init_sharded(solver)

    # ---- device-resident inputs (value) and pinned host inputs (e2e)
    def pinned(x):
        if x is None:
            return None
        t = torch.empty(x.shape, dtype=tdt, pin_memory=True)
        t.numpy()[...] = x
        return t

    host = {k: pinned(data[k]) for k in ("pos", "forces", "torques", "noise")}
    dev = {k: (None if v is None else v.cuda()) for k, v in host.items()}
    nout = cfg.nrhs * 3 * N
    d_lin = torch.empty(nout, dtype=tdt, device="cuda")
    d_ang = torch.empty(nout, dtype=tdt, device="cuda") if cfg.angular else None
    h_lin = torch.empty(nout, dtype=tdt, pin_memory=True)
    h_ang = torch.empty(nout, dtype=tdt, pin_memory=True) if cfg.angular else None
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step_device():
        solver.set_positions(dev["pos"])
        if cfg.op == "sqrt+mdot":
            solver.hydrodynamic_velocities(dev["forces"], dev["torques"], dev["noise"], 1.0, cfg.tol, d_lin, d_ang)
        elif cfg.op == "mdot_batch":
            solver.mdot_batch(cfg.nrhs, dev["forces"], dev["torques"], d_lin, d_ang)
        else:
            solver.mdot(dev["forces"], dev["torques"], d_lin, d_ang)

    np_or_none = lambda t: None if t is None else t.numpy()

    def step_host():
        solver.set_positions_host(np_or_none(host["pos"]))
        if cfg.op == "sqrt+mdot":
            solver.hydrodynamic_velocities_host(np_or_none(host["forces"]), np_or_none(host["torques"]), np_or_none(host["noise"]), 1.0, cfg.tol,
                                                np_or_none(h_lin), np_or_none(h_ang))
        elif cfg.op == "mdot_batch":
            solver.mdot_batch_host(cfg.nrhs, np_or_none(host["forces"]), np_or_none(host["torques"]), np_or_none(h_lin), np_or_none(h_ang))
        else:
            solver.mdot_host(np_or_none(host["forces"]), np_or_none(host["torques"]), np_or_none(h_lin), np_or_none(h_ang))

    h2d = sum(v.numel() * v.element_size() for v in host.values() if v is not None)
    d2h = h_lin.numel() * h_lin.element_size() * (2 if cfg.angular else 1)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(step_fn, K):
        """K steps; each bracketed by CUDA events on the launching stream; the L2 flush between steps
        sits outside the brackets.  Returns (sum of step ms, wall t0, wall t1)."""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        barrier()
        t0 = time.time()
        for e0, e1 in evs:
            flush.zero_()
            e0.record(stream)
            step_fn()
            e1.record(stream)
        barrier()
        t1 = time.time()
        return sum(e0.elapsed_time(e1) for e0, e1 in evs), t0, t1

    for _ in range(args.warmup):
        step_device()
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    solver.set_profiling(True)
    solver.reset_stats()
    ms_total, w0, w1 = timed(step_device, args.steps)
    stats = solver.get_stats()
    solver.set_profiling(False)
    clocks = sampler.stop(w0, w1) if rank == 0 else None
    iters = solver.last_iterations() if cfg.op == "sqrt+mdot" else None

    e2e_ms = None
    if not args.no_e2e:
        for _ in range(2):
            step_host()
        solver.reset_stats()
        e2e_ms, _, _ = timed(step_host, args.steps)
        e2e_stats = solver.get_stats()

    # ---- max over ranks of the device time, sum over ranks of the pairs (replicas only)
    ms_total, pairs_all = multi.aggregate_over_ranks(ms_total, stats["pairs"], device="cuda")
    e2e_pairs_all = 0.0
    if e2e_ms is not None:
        e2e_ms, e2e_pairs_all = multi.aggregate_over_ranks(e2e_ms, e2e_stats["pairs"], device="cuda")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = pairs_all / (ms_total * 1e-3) / 1e9
    launches_pair = stats["pair_kernel_launches"]
    pair_ms_avg = stats["pair_kernel_ms"] / max(1, launches_pair)

    # ---- roofline of the dominant kernel: the pair kernel, FMA-pipe ("alu") bound
    nrhs_launch = cfg.nrhs if cfg.op == "mdot_batch" else 1
    instr, flops = work_per_pair(cfg.angular, nrhs_launch, f64)
    props = torch.cuda.get_device_properties(local_rank)
    sms = props.multi_processor_count
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    except Exception:
        sm_max_mhz = 1965.0
    if clocks and clocks.get("sm_max_mhz"):
        sm_max_mhz = float(clocks["sm_max_mhz"])
    peak = sms * nominal_lanes(f64) * sm_max_mhz * 1e6 / 1e12                 # T lane-ops/s at max clock
    pairs_per_launch = stats["pairs"] / max(1, launches_pair)                 # rank 0's share when row-sharded
    achieved = instr * pairs_per_launch / (pair_ms_avg * 1e-3) / 1e12
    probe = lm.lm_probe_fma_peak(lm.LM_F64 if f64 else lm.LM_F32, 0.3) / 1e12
    roofline = {
        "bound": "alu", "kernel": f"rpy_pair_kernel<{cfg.precision}, nrhs={nrhs_launch}, angular={int(cfg.angular)}>",
        "achieved": achieved, "peak": peak, "unit": "T FP-pipe lane-ops/s", "frac": achieved / peak,
        "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(args.config) if args.N is None else None,
        "traffic_unit": "bytes per launch (ncu dram read+write, profiles/r1_c%d_pair_kernel_ncu_full.md)" % args.config,
        "peak_source": f"derived: {sms} SMs x {nominal_lanes(f64)} lanes x {sm_max_mhz:.0f} MHz (clocks.max.sm); MEASURED_PEAKS.json has no ALU entry",
        "lane_ops_per_pair": instr, "flops_per_pair": flops, "pairs_per_launch": pairs_per_launch,
        "launch_ms_avg": pair_ms_avg, "launches_timed": launches_pair,
        "flop_frac": flops * pairs_per_launch / (pair_ms_avg * 1e-3) / 1e12 / (2 * peak),
        "measured_fma_peak": probe, "frac_of_measured_fma_peak": achieved / probe,
        "kernel_gpairs_per_s": pairs_per_launch / (pair_ms_avg * 1e-3) / 1e9,
    }
    if clocks and clocks.get("sm_mhz"):
        roofline["frac_at_observed_clock"] = achieved / (sms * nominal_lanes(f64) * clocks["sm_mhz"] * 1e6 / 1e12)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": cfg.precision, "data": "synthetic",
        "config": config_dict(cfg, N, {"l2": "256 MiB device memset between steps, outside the event brackets",
                                       "parallelism": ("row-sharded, all-gather per apply" if sharded else "replicas only") if world > 1 else "1 GPU",
                                       "pair_launches_per_step": launches_pair / args.steps, "lanczos_iterations": iters,
                                       "launch": solver.pair_launch_config(nrhs_launch)}),
        "ms_per_mdot": pair_ms_avg,
        "gpu_launches": int(stats["pair_kernel_launches"] + stats["aux_launches"]),
        "clocks": clocks,
        "roofline": roofline,
    }
    if e2e_ms is not None:
        line["e2e"] = {"value": e2e_pairs_all / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "api": "lm_set_positions_host + lm_*_host (pinned host buffers)"}
    if world == 1 and not args.no_cpu_baseline:
        info = oracle_rate(data, 12.0)
        line["cpu_baseline"] = {"value": info["pairs"] / info["seconds"] / 1e9, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                                "sample": f"{info['nrows']} sampled target rows x all {N} sources, one M.F apply, {info['seconds']:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
