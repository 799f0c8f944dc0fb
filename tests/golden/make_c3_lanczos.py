"""Writes tests/golden/c3_lanczos_tol1e-3.json: the ORACLE's Lanczos run of config 3 (fp32 inputs, N = 131072, phi = 5 %)
at the tolerance and stopping rule bench.py times (tol 1e-3, rule "estimate", readings S3/S4).

    python tests/golden/make_c3_lanczos.py [--n N] [--out FILE]

Imports ONLY oracle/ and the seeded input generator (paper_2510_02135_b200.workloads, which holds no method arithmetic):
nothing in the file it writes comes from the CUDA path.  Cost: one fp64 O(N^2) oracle apply per Lanczos iteration
(~75 applies; ~19 s each on 16 cores at N = 131072).  Stored:
  alphas, betas        alpha_k, beta_k of the whole run (fp64 recurrence, no re-orthogonalisation)
  steps, estimates     s_k (k >= 2) and the rule's error estimate e_k (k >= 3)
  iterations           the oracle's stop step
  rows, y_rows         64 evenly spaced particle indices and the final iterate y = M^{1/2} z at those rows (64 x 3)
  mz_rows              the rows of M z at the same indices (exact, for the square-root-twice check)
  y_norm               |y|
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import rpy  # noqa: E402
from paper_2510_02135_b200 import workloads  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=None, help="reduced N (same recipe) for a dry run; default: the config's N")
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "c3_lanczos_tol1e-3.json"))
    args = ap.parse_args()
    d = workloads.generate(3, N=args.n)
    cfg, N = d["cfg"], d["N"]
    tol, rule = cfg.tol, "estimate"
    z = d["noise"].astype(np.float64)
    hist = {}
    t0 = time.time()
    y, k, conv = rpy.lanczos_sqrt_mdot_w(d["pos"], z, tol, a=cfg.a, eta=cfg.eta, max_iter=200, rule=rule, history=hist)
    t1 = time.time()
    rows = np.arange(64, dtype=np.int64) * (N // 64)
    Mz, _ = rpy.mdot_rows(d["pos"], rows, z, None, a=cfg.a, eta=cfg.eta)
    out = {
        "provenance": "oracle/rpy.py lanczos_sqrt_mdot_w + mdot_rows on workloads.generate(3); written by tests/golden/make_c3_lanczos.py",
        "config": 3, "N": int(N), "tol": tol, "rule": rule, "a": cfg.a, "eta": cfg.eta, "seed": cfg.seed,
        "converged": bool(conv), "iterations": int(k), "oracle_seconds": round(t1 - t0, 1), "oracle_threads": int(rpy.mdot.last_threads),
        "alphas": [float(v) for v in hist["alphas"]], "betas": [float(v) for v in hist["betas"]],
        "steps": [float(v) for v in hist["steps"]], "estimates": [float(v) for v in hist["estimates"]],
        "rows": [int(r) for r in rows], "y_rows": y.reshape(N, 3)[rows].tolist(), "mz_rows": Mz.tolist(),
        "y_norm": float(np.linalg.norm(y)),
    }
    with open(args.out, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(f"[golden] N={N} tol={tol} rule={rule}: {k} iterations, converged={conv}, {t1 - t0:.0f} s -> {args.out}")


if __name__ == "__main__":
    main()
