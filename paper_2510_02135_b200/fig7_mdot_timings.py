"""Mdot wall time versus N on a perturbed FCC lattice -- the timing protocol of the paper's Fig. 7
("computational time required to compute deterministic particle displacements (the
Mdot operation) for ... a face-centered cubic (FCC) lattice ... slightly randomized", two number
densities rho = N/V in units of a, monopoles only), for this library's open-boundary solver.

    python -m paper_2510_02135_b200.fig7_mdot_timings [--precision f32|f64] [--max-n 1048576]

The paper's own curves exist only as an image (RTX A6000); the two densities used here (0.01 and 0.1
a^-3, both free of overlaps) are this repo's choice.  Prints a markdown table; time = CUDA-event mean
of lm_mdot (pack + pair kernel + split-j reduce), positions already set.
"""
from __future__ import annotations

import argparse

import numpy as np


def main():
    import torch

    import paper_2510_02135_b200 as lm
    from paper_2510_02135_b200 import workloads

    ap = argparse.ArgumentParser()
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--max-n", type=int, default=1048576)
    args = ap.parse_args()
    dens = (0.01, 0.1)
    print(f"| N | " + " | ".join(f"ms (rho = {d:g})" for d in dens) + " | Gpairs/s |")
    print("|---:|" + "---:|" * (len(dens) + 1))
    for n_cells in (2, 3, 4, 6, 8, 10, 13, 16, 20, 26, 32, 40, 51, 64):
        N = 4 * n_cells ** 3
        if N > args.max_n:
            break
        cells = []
        for d in dens:
            pos = workloads.fcc(n_cells, d, 0.1, seed=n_cells).astype(workloads.np_dtype(args.precision))
            s = lm.Solver(args.precision, N, 1.0, 1.0, False)
            X = torch.from_numpy(np.ascontiguousarray(pos)).cuda().reshape(-1)
            F = torch.randn(3 * N, dtype=s.torch_dtype, device="cuda")
            U = torch.empty_like(F)
            s.set_positions(X)
            for _ in range(3):
                s.mdot(F, None, U)
            torch.cuda.synchronize()
            reps = 50 if N <= 20000 else (10 if N <= 200000 else 2)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                s.mdot(F, None, U)
            e1.record()
            torch.cuda.synchronize()
            cells.append(e0.elapsed_time(e1) / reps)
            s.close()
        print(f"| {N} | " + " | ".join(f"{c:.4f}" for c in cells) + f" | {N * N / cells[-1] / 1e6:.1f} |", flush=True)


if __name__ == "__main__":
    main()
