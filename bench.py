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

configs = the other four BASELINE.json configs measured in the same run (a few steps each; single GPU, default
          headline only): ms per launch, roofline fraction, e2e -- so that every number of BASELINE.md sec. 4 is on
          the driver's record, not only the headline.
steady_state = small configs only (1, 2): whole applies back to back on the stream, no L2 flush -- the loop a
          time-stepping user runs; reported beside the flushed per-step figures, never instead of them.
--fig7  = the paper's Fig. 7 protocol (Mdot time vs N, open boundaries and bottom wall) as one JSON line, instead of a config.

Multi-GPU (torchrun): "replicas only" by default: every rank runs an independent replica
(seed + 1000 rank), scaling = "weak"; `--parallelism sharded` row-shards ONE problem over the ranks (lm_dist_init:
all-gather of the row blocks inside every apply), scaling = "strong".
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


def profile_traffic(config: int):
    """DRAM bytes of ONE pair-kernel launch (dram__bytes_read.sum + dram__bytes_write.sum) read at run time from the
    committed `ncu --set full` summary of the same launch configuration, profiles/r<round>_c<config>_pair_kernel_ncu_full.md
    (newest round present).  A recorded profile value -- ncu cannot run inside a timed benchmark.  (bytes, path) or (None, None)."""
    import glob
    import re
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_c{config}_pair_kernel_ncu_full.md")), reverse=True):
        text = open(path).read()
        got = {}
        for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            m = re.search(r"\|\s*" + re.escape(key) + r"\s*\|\s*(\w+)\s*\|\s*([0-9.eE+-]+)\s*\|", text)
            if m and m.group(1) in unit:
                got[key] = float(m.group(2)) * unit[m.group(1)]
        if len(got) == 2:
            return sum(got.values()), os.path.relpath(path, ROOT)
    return None, None


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
        "data": "synthetic", "config": config_dict(cfg, data["N"]),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": info["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def config_dict(cfg, N):
    """Names the workload; identical for the CUDA arm and the reference arm (run-dependent facts go to `details`)."""
    d = {"workload": f"BASELINE.json configs[{cfg.index - 1}] ({cfg.name})", "op": cfg.op, "N": int(N), "precision": cfg.precision,
         "include_angular": bool(cfg.angular), "nrhs": int(cfg.nrhs), "geometry": f"{cfg.geometry}={cfg.geom_param:g}", "seed": int(cfg.seed),
         "a": cfg.a, "eta": cfg.eta}
    if cfg.tol:
        d["lanczos_tol"] = cfg.tol
    d["l2"] = "256 MiB device memset between steps, outside the event brackets (CUDA arm)"
    return d


# ---------------------------------------------------------------- the CUDA arm
class Arm:
    """One config on this rank's GPU: device-resident and pinned-host inputs, the step functions, the timers."""

    def __init__(self, lm, torch, dist, index, N_override, rank, world, sharded):
        from paper_2510_02135_b200 import multi, workloads
        self.lm, self.torch, self.dist, self.world = lm, torch, dist, world
        cfg = self.cfg = workloads.CONFIGS[index]
        # replicas: every rank its own problem (seed + 1000 rank); sharded: the same problem on every rank
        self.data = data = workloads.generate(index, N_override, seed=cfg.seed if sharded else multi.replica_seed(cfg.seed, rank))
        N = self.N = data["N"]
        self.f64 = cfg.precision == "f64"
        tdt = torch.float64 if self.f64 else torch.float32
        self.stream = torch.cuda.current_stream()
        self.solver = lm.Solver(cfg.precision, N, cfg.eta, cfg.a, cfg.angular)
        if sharded:
            multi.init_sharded(self.solver)

        def pinned(x):
            if x is None:
                return None
            t = torch.empty(x.shape, dtype=tdt, pin_memory=True)
            t.numpy()[...] = x
            return t

        self.host = {k: pinned(data[k]) for k in ("pos", "forces", "torques", "noise")}
        self.dev = {k: (None if v is None else v.cuda()) for k, v in self.host.items()}
        nout = cfg.nrhs * 3 * N
        self.d_lin = torch.empty(nout, dtype=tdt, device="cuda")
        self.d_ang = torch.empty(nout, dtype=tdt, device="cuda") if cfg.angular else None
        self.h_lin = torch.empty(nout, dtype=tdt, pin_memory=True)
        self.h_ang = torch.empty(nout, dtype=tdt, pin_memory=True) if cfg.angular else None
        self.h2d = sum(v.numel() * v.element_size() for v in self.host.values() if v is not None)
        self.d2h = self.h_lin.numel() * self.h_lin.element_size() * (2 if cfg.angular else 1)

    def close(self):
        self.solver.close()
        self.host = self.dev = self.d_lin = self.d_ang = self.h_lin = self.h_ang = None

    def step_device(self):
        cfg, s, dev = self.cfg, self.solver, self.dev
        s.set_positions(dev["pos"])
        if cfg.op == "sqrt+mdot":
            s.hydrodynamic_velocities(dev["forces"], dev["torques"], dev["noise"], 1.0, cfg.tol, self.d_lin, self.d_ang)
        elif cfg.op == "mdot_batch":
            s.mdot_batch(cfg.nrhs, dev["forces"], dev["torques"], self.d_lin, self.d_ang)
        else:
            s.mdot(dev["forces"], dev["torques"], self.d_lin, self.d_ang)

    def step_host(self):
        cfg, s = self.cfg, self.solver
        n = lambda t: None if t is None else t.numpy()
        h = self.host
        s.set_positions_host(n(h["pos"]))
        if cfg.op == "sqrt+mdot":
            s.hydrodynamic_velocities_host(n(h["forces"]), n(h["torques"]), n(h["noise"]), 1.0, cfg.tol, n(self.h_lin), n(self.h_ang))
        elif cfg.op == "mdot_batch":
            s.mdot_batch_host(cfg.nrhs, n(h["forces"]), n(h["torques"]), n(self.h_lin), n(self.h_ang))
        else:
            s.mdot_host(n(h["forces"]), n(h["torques"]), n(self.h_lin), n(self.h_ang))

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def timed(self, step_fn, K, flush):
        """K steps; each bracketed by CUDA events on the launching stream; the L2 flush between steps
        sits outside the brackets.  Returns (sum of step ms, wall t0, wall t1)."""
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        self.barrier()
        t0 = time.time()
        for e0, e1 in evs:
            flush.zero_()
            e0.record(self.stream)
            step_fn()
            e1.record(self.stream)
        self.barrier()
        t1 = time.time()
        return sum(e0.elapsed_time(e1) for e0, e1 in evs), t0, t1

    def steady_state(self, reps=200):
        """Small configs only (working set far below the L2): `reps` applies back to back on the stream -- no L2 flush, no
        set_positions, the loop a time-stepping user runs -- under ONE event pair.  Reported beside the per-step figures,
        never instead of them: an event pair around ONE launch of a few microseconds mostly measures the stream-launch
        grid of this B200 (2.048 us per dependent stream operation, the two event records included)."""
        if self.cfg.op != "mdot" or self.N > 20000:
            return None
        torch, s, dev = self.torch, self.solver, self.dev
        for _ in range(10):
            s.mdot(dev["forces"], dev["torques"], self.d_lin, self.d_ang)
        best = None
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(self.stream)
            for _ in range(reps):
                s.mdot(dev["forces"], dev["torques"], self.d_lin, self.d_ang)
            e1.record(self.stream)
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / reps
            best = us if best is None else min(best, us)
        instr, _ = work_per_pair(self.cfg.angular, 1, self.f64)
        return {"us_per_apply": best, "gpairs_per_s": float(self.N) * self.N / (best * 1e-6) / 1e9, "applies": reps,
                "what": "whole applies (launch overhead included) back to back on one stream through the binding, no L2 flush, no set_positions "
                        "(best of 3); frac = the same lane-operations per pair over this time"}

    def measure(self, steps, warmup, flush, do_e2e, sampler=None):
        """value pass (profiling OFF: the code path a user gets, CUDA-graph replay included), a short profiled pass
        for the pair kernel's own launch time, and the e2e pass through the *_host calls."""
        s, torch = self.solver, self.torch
        for _ in range(warmup):
            self.step_device()
        torch.cuda.synchronize()
        if sampler is not None:
            sampler.start()
            time.sleep(0.3)
        s.reset_stats()
        ms_total, w0, w1 = self.timed(self.step_device, steps, flush)
        stats = s.get_stats()
        clocks = sampler.stop(w0, w1) if sampler is not None else None
        iters = s.last_iterations() if self.cfg.op == "sqrt+mdot" else None
        hist = s.lanczos_history() if self.cfg.op == "sqrt+mdot" else None
        # the pair kernel alone: every launch bracketed by CUDA events on its stream (direct launches, no graph)
        s.set_profiling(True)
        s.reset_stats()
        psteps = max(1, min(steps, 3))
        self.timed(self.step_device, psteps, flush)
        pstats = s.get_stats()
        s.set_profiling(False)
        out = dict(ms_total=ms_total, stats=stats, pstats=pstats, clocks=clocks, iters=iters, hist=hist, e2e_ms=None, e2e_stats=None)
        if do_e2e:
            for _ in range(2):
                self.step_host()
            s.reset_stats()
            out["e2e_ms"], _, _ = self.timed(self.step_host, steps, flush)
            out["e2e_stats"] = s.get_stats()
        return out


def roofline_of(arm, m, sm_max_mhz, sms, probe_lane_ops, config_index, N_override):
    cfg = arm.cfg
    nrhs_launch = cfg.nrhs if cfg.op == "mdot_batch" else 1
    instr, flops = work_per_pair(cfg.angular, nrhs_launch, arm.f64)
    ps = m["pstats"]
    launches = max(1, ps["pair_kernel_launches"])
    pair_ms_avg = ps["pair_kernel_ms"] / launches
    # lane-ops of all profiled launches (the first Lanczos apply of a config-3 step is a 2-RHS launch: 10 more per pair)
    extra = 0.0
    if cfg.op == "sqrt+mdot":
        steps_prof = max(1, round(launches / max(1, (m["iters"] or 1))))
        extra = 10.0 * steps_prof * float(arm.N) * arm.N
    pairs_per_launch = ps["pairs"] / launches
    lane_ops = instr * ps["pairs"] + extra
    peak = sms * nominal_lanes(arm.f64) * sm_max_mhz * 1e6 / 1e12                 # T lane-ops/s at max clock
    achieved = lane_ops / (ps["pair_kernel_ms"] * 1e-3) / 1e12
    traffic, traffic_src = profile_traffic(config_index) if N_override is None else (None, None)
    r = {
        "bound": "alu", "kernel": f"{arm.solver.pair_launch_config(nrhs_launch)['kernel']}<{cfg.precision}, nrhs={nrhs_launch}, angular={int(cfg.angular)}>",
        "achieved": achieved, "peak": peak, "unit": "T FP-pipe lane-ops/s", "frac": achieved / peak,
        "traffic": traffic, "traffic_unit": "bytes per launch: dram__bytes_read.sum + dram__bytes_write.sum of the committed ncu capture",
        "traffic_source": traffic_src,
        "algorithmic_bytes_per_launch": int(((arm.N + 31) // 32 * 32) * (3 + (6 if cfg.angular else 3) * nrhs_launch) * (8 if arm.f64 else 4)
                                            + 3 * arm.N * (2 if cfg.angular else 1) * nrhs_launch * (8 if arm.f64 else 4)),
        "peak_source": f"derived: {sms} SMs x {nominal_lanes(arm.f64)} lanes x {sm_max_mhz:.0f} MHz (clocks.max.sm); MEASURED_PEAKS.json has no ALU entry",
        # lane_ops_per_pair: the dominant (1-RHS) launch's count; effective_...: what `achieved` divides by -- all timed launches,
        # including the 2-RHS first launch of each Lanczos call (+10 per pair): frac = effective x pairs / time / peak
        "lane_ops_per_pair": instr, "effective_lane_ops_per_pair": lane_ops / max(ps["pairs"], 1.0), "flops_per_pair": flops, "pairs_per_launch": pairs_per_launch,
        "launch_ms_avg": pair_ms_avg, "launches_timed": ps["pair_kernel_launches"],
        "flop_frac": flops * ps["pairs"] / (ps["pair_kernel_ms"] * 1e-3) / 1e12 / (2 * peak),
        "kernel_gpairs_per_s": pairs_per_launch / (pair_ms_avg * 1e-3) / 1e9,
    }
    if probe_lane_ops:
        r["measured_fma_peak"] = probe_lane_ops / 1e12
        r["frac_of_measured_fma_peak"] = achieved / (probe_lane_ops / 1e12)
    if m["clocks"] and m["clocks"].get("sm_mhz"):
        r["frac_at_observed_clock"] = achieved / (sms * nominal_lanes(arm.f64) * m["clocks"]["sm_mhz"] * 1e6 / 1e12)
    return r


def lanczos_true_error(lm, torch, arm, y_f32):
    """Relative error of the timed step's noise part against a 300-step fp64 run of the same recurrence (outside the
    timed region): what `tol` delivered at this config (S3/S4)."""
    d, N = arm.data, arm.N
    s64 = lm.Solver("f64", N, arm.cfg.eta, arm.cfg.a, arm.cfg.angular)
    s64.set_positions(torch.from_numpy(d["pos"].astype(np.float64)).cuda())
    s64.set_max_iter(300)
    yref = torch.empty(3 * N, dtype=torch.float64, device="cuda")
    try:
        s64.sqrt_mdot_w(torch.from_numpy(d["noise"].astype(np.float64)).cuda(), 1e-9, yref, None, allow_noconv=True)
    finally:
        pass
    err = float((y_f32.double() - yref).norm() / yref.norm())
    s64.close()
    return err


def run_fig7(args):
    """--fig7: the paper's Fig. 7 protocol on this library: time of one Mdot vs N on a perturbed FCC
    lattice without overlaps, monopoles only, two number densities, for NBody with open boundaries and with a bottom
    wall.  Context, not a comparison (the paper's curves are an RTX A6000 and exist only as a figure).  Each point: applies
    back to back on one stream (the loop a user runs; inputs stay in L2 below N ~ 10^6), best of 3.  One JSON line."""
    import torch

    import paper_2510_02135_b200 as lm
    from paper_2510_02135_b200 import workloads
    cells = [2, 3, 4, 6, 8, 10, 13, 16, 20, 26, 32, 40, 51, 64]      # N = 4 n^3: 32 ... 1048576
    out = {"protocol": "perturbed FCC lattice (jitter 0.1 a, no overlaps), monopoles, applies back to back, best of 3, ms per Mdot",
           "densities": [0.01, 0.1], "rows": []}
    for prec in ("f32", "f64"):
        tdt = torch.float32 if prec == "f32" else torch.float64
        for wall in (False, True):
            for n in cells:
                N = 4 * n ** 3
                if (prec == "f64" and N > 300000) or (wall and N > 300000) or (args.N and N > args.N):
                    continue
                row = {"precision": prec, "geometry": "single_wall" if wall else "open", "N": N, "ms": []}
                for rho in out["densities"]:
                    x = workloads.fcc(n, rho, 0.1, 7)
                    if wall:
                        x[:, 2] += 1.5 - x[:, 2].min()                 # lowest layer 1.5 a above the wall at z = 0
                    pos = torch.from_numpy(x.reshape(-1)).to(tdt).cuda()
                    F = torch.randn(3 * N, dtype=tdt, device="cuda")
                    U = torch.empty_like(F)
                    s = lm.Solver(prec, N)
                    if wall:
                        s.set_wall(True, 0.0)
                    s.set_positions(pos)
                    pairs = float(N) * N * (3.4 if wall else 1.0) * (2.5 if prec == "f64" else 1.0)
                    reps = int(max(2, min(300, 3e11 / pairs)))
                    for _ in range(3):
                        s.mdot(F, None, U)
                    best = None
                    for _ in range(3):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        torch.cuda.synchronize()
                        e0.record()
                        for _ in range(reps):
                            s.mdot(F, None, U)
                        e1.record()
                        torch.cuda.synchronize()
                        ms = e0.elapsed_time(e1) / reps
                        best = ms if best is None else min(best, ms)
                    row["ms"].append(best)
                    row["kernel"] = s.pair_launch_config(1)["kernel"]
                    s.close()
                row["gpairs_per_s"] = float(N) * N / (min(row["ms"]) * 1e-3) / 1e9
                out["rows"].append(row)
    print(json.dumps({"fig7": out}))


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
    ap.add_argument("--no-configs", action="store_true", help="skip the sub-records of the other four configs")
    ap.add_argument("--small-kernel", type=int, default=1, choices=[0, 1], help="LM_OPT_SMALL_KERNEL: 1 = the one-launch kernel where the library prefers it (default), 0 = never (A/B runs)")
    ap.add_argument("--fig7", action="store_true", help="the paper's Fig. 7 protocol (Mdot time vs N, open and bottom-wall NBody) instead of a config")
    ap.add_argument("--lanczos-rule", default="estimate", choices=["estimate", "step"], help="stopping rule (DESIGN.md reading S3)")
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
    from paper_2510_02135_b200 import multi, probe

    if args.fig7:
        if rank == 0:
            run_fig7(args)
        return 0

    sharded = args.parallelism == "sharded" and world > 1
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    arm = Arm(lm, torch, dist, args.config, args.N, rank, world, sharded)
    cfg, N = arm.cfg, arm.N
    arm.solver.set_option(lm.LM_OPT_SMALL_KERNEL, args.small_kernel)
    if cfg.op == "sqrt+mdot":
        arm.solver.set_option(lm.LM_OPT_LANCZOS_RULE, lm.LM_RULE_STEP if args.lanczos_rule == "step" else lm.LM_RULE_ESTIMATE)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    m = arm.measure(args.steps, args.warmup, flush, not args.no_e2e, sampler)

    # ---- max over ranks of the device time, sum over ranks of the pairs
    ms_total, pairs_all = multi.aggregate_over_ranks(m["ms_total"], m["stats"]["pairs"], device="cuda")
    e2e_ms, e2e_pairs_all = None, 0.0
    if m["e2e_ms"] is not None:
        e2e_ms, e2e_pairs_all = multi.aggregate_over_ranks(m["e2e_ms"], m["e2e_stats"]["pairs"], device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    props = torch.cuda.get_device_properties(local_rank)
    sms = props.multi_processor_count
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    except Exception:
        sm_max_mhz = 1965.0
    clocks = m["clocks"]
    if clocks and clocks.get("sm_max_mhz"):
        sm_max_mhz = float(clocks["sm_max_mhz"])
    probes = {False: probe.fma_peak(lm.LM_F32, 0.3), True: probe.fma_peak(lm.LM_F64, 0.3)}
    roofline = roofline_of(arm, m, sm_max_mhz, sms, probes[arm.f64], args.config, args.N)
    stats = m["stats"]
    nrhs_launch = cfg.nrhs if cfg.op == "mdot_batch" else 1
    extra = {"parallelism": ("row-sharded, all-gather per apply" if sharded else "replicas only") if world > 1 else "1 GPU",
             "pair_launches_per_step": stats["pair_kernel_launches"] / args.steps, "lanczos_iterations": m["iters"],
             "launch": arm.solver.pair_launch_config(nrhs_launch)}
    if cfg.op == "sqrt+mdot":
        # what tol delivered: the noise part of the timed step against a long fp64 run (measured outside the timed region)
        y = torch.empty(3 * N, dtype=torch.float32, device="cuda")
        arm.solver.sqrt_mdot_w(arm.dev["noise"], cfg.tol, y, None)
        hist = arm.solver.lanczos_history()
        extra["lanczos_rule"] = args.lanczos_rule
        extra["lanczos_error_estimate_at_stop"] = float(hist["estimate"][-1]) if args.lanczos_rule == "estimate" else float(hist["step"][-1])
        if world == 1 and args.N is None:
            extra["lanczos_true_rel_error_vs_fp64_300_steps"] = lanczos_true_error(lm, torch, arm, y)
        del y

    line = {
        "metric": METRIC, "value": pairs_all / (ms_total * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": cfg.precision, "data": "synthetic", "config": config_dict(cfg, N), "details": extra,
        "ms_per_mdot": roofline["launch_ms_avg"],
        # time to solution of the user-visible call, which `value` (pairs/s) hides: Lanczos iterations per step and ms per step
        "lanczos_iterations": m["iters"], "ms_per_sqrt_mdot_w": (ms_total / args.steps) if cfg.op == "sqrt+mdot" else None,
        "gpu_launches": int(stats["pair_kernel_launches"] + stats["aux_launches"]),
        "clocks": clocks,
        "roofline": roofline,
    }
    if e2e_ms is not None:
        line["e2e"] = {"value": e2e_pairs_all / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                       "h2d_bytes_per_step": int(arm.h2d), "d2h_bytes_per_step": int(arm.d2h), "api": "lm_set_positions_host + lm_*_host (pinned host buffers)"}
    ss = arm.steady_state() if world == 1 else None
    if ss is not None:
        ss["frac"] = roofline["lane_ops_per_pair"] * float(N) * N / (ss["us_per_apply"] * 1e-6) / 1e12 / roofline["peak"]
        line["steady_state"] = ss
    data_headline = arm.data
    arm.close()

    # ---- the other four configs, a few steps each, so that every config's numbers are on the driver's record
    if world == 1 and args.config == 3 and args.N is None and not args.no_configs:
        sub = {}
        for index, (k, w) in {1: (20, 5), 2: (10, 3), 4: (2, 3), 5: (3, 3)}.items():
            torch.cuda.empty_cache()
            a2 = Arm(lm, torch, dist, index, None, 0, 1, False)
            m2 = a2.measure(k, w, flush, True, ClockSampler(local_rank))
            r2 = roofline_of(a2, m2, sm_max_mhz, sms, probes[a2.f64], index, None)
            c2 = a2.cfg
            sub[str(index)] = {
                "workload": f"BASELINE.json configs[{index - 1}] ({c2.name})", "steps": k, "warmup": w,
                "value": m2["stats"]["pairs"] / (m2["ms_total"] * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": m2["ms_total"] / k,
                "ms_per_launch": r2["launch_ms_avg"], "kernel_gpairs_per_s": r2["kernel_gpairs_per_s"], "lane_ops_per_pair": r2["lane_ops_per_pair"],
                "frac": r2["frac"], "flop_frac": r2["flop_frac"], "traffic": r2["traffic"], "traffic_source": r2["traffic_source"],
                "algorithmic_bytes_per_launch": r2["algorithmic_bytes_per_launch"],
                "e2e": {"value": m2["e2e_stats"]["pairs"] / (m2["e2e_ms"] * 1e-3) / 1e9, "ms_per_step": m2["e2e_ms"] / k,
                        "h2d_bytes_per_step": int(a2.h2d), "d2h_bytes_per_step": int(a2.d2h)},
                "launch": a2.solver.pair_launch_config(c2.nrhs if c2.op == "mdot_batch" else 1),
                "gpu_launches": int(m2["stats"]["pair_kernel_launches"] + m2["stats"]["aux_launches"]),
                "clocks": m2["clocks"],
            }
            ss2 = a2.steady_state()
            if ss2 is not None:
                ss2["frac"] = r2["lane_ops_per_pair"] * float(a2.N) * a2.N / (ss2["us_per_apply"] * 1e-6) / 1e12 / r2["peak"]
                sub[str(index)]["steady_state"] = ss2
            a2.close()
        line["configs"] = sub

    if world == 1 and not args.no_cpu_baseline:
        info = oracle_rate(data_headline, 12.0)
        line["cpu_baseline"] = {"value": info["pairs"] / info["seconds"] / 1e9, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                                "sample": f"{info['nrows']} sampled target rows x all {N} sources, one M.F apply, {info['seconds']:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
