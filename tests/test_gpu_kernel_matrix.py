"""Every kernel variant of liblm once, each compared with the CPU oracle (the selection SURVEY.md sec. 5 wanted run under
compute-sanitizer; that tool is closed on this GPU pool, see profiles/r2_sanitizer.md -- tests/test_gpu_memory_discipline.py
runs the same matrix with guard bands, poisoned neighbours and repeat-determinism instead):

  pair kernel   fp32 / fp64  x  translational / angular  x  1, 2, 4 right-hand sides  x  free space / single wall
                x  the three launch shapes: one-launch cluster kernel (rpy_small.cuh), general path SMALL shape
                (64 threads), general path LARGE shape (256 threads, TMA double buffer over several tiles, j-split partials)
  steric kernel, Lanczos on the graph-replayed path and on the direct path with the fused split-j reduce, one BD step.
"""
import numpy as np
import pytest

from oracle import bd, rpy, wall
from paper_2510_02135_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def close(a, b, tol):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return rel(a, b) <= tol and np.abs(a - b).max() <= 8 * tol * np.abs(b).max()


@pytest.fixture(scope="module")
def lm():
    import paper_2510_02135_b200 as lm
    return lm


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def dev(torch, x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


# shape -> (N, LM_OPT_SMALL_KERNEL, expected kernel, expected block)
SHAPES = {"cluster": (333, 1, "rpy_small_kernel", None), "small": (333, 0, "rpy_pair_kernel", 64), "large": (9000, 0, "rpy_pair_kernel", 256)}


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular,nrhs", [(False, 1), (False, 2), (False, 4), (True, 1), (True, 2)])
@pytest.mark.parametrize("with_wall", [False, True])
@pytest.mark.parametrize("shape", ["cluster", "small", "large"])
def test_pair_kernel_variant(lm, torch, prec, angular, nrhs, with_wall, shape):
    # (single-wall variants exist for 1 and 2 right-hand sides: lm_mdot_batch serves 4 as 2 + 2)
    N, mode, kernel, block = SHAPES[shape]
    side = 1.6 * N ** (1.0 / 3.0)                              # ~10 % volume fraction: overlapping and far pairs
    if with_wall:
        c = workloads.wall_slab_case(N, side * 1.5, -0.2, 4.0, 31 + nrhs, prec, angular, wall_z=0.5)
    else:
        c = workloads.random_case(N, side, 31 + nrhs, prec, angular)
    rng = np.random.default_rng(nrhs)
    dt = workloads.np_dtype(prec)
    F = np.stack([c["forces"]] + [rng.standard_normal((N, 3)).astype(dt) for _ in range(nrhs - 1)])
    T = np.stack([c["torques"]] + [rng.standard_normal((N, 3)).astype(dt) for _ in range(nrhs - 1)]) if angular else None
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    if with_wall:
        s.set_wall(True, c["wall_z"])
    s.set_option(lm.LM_OPT_SMALL_KERNEL, mode)
    s.set_positions(dev(torch, c["pos"]))
    cfg = s.pair_launch_config(2 if (with_wall and nrhs == 4) else nrhs)
    assert cfg["kernel"] == kernel and (block is None or cfg["block"] == block), cfg
    if shape == "large":
        assert cfg["j_splits"] > 1                              # partial sums + reduce kernel on this path
    U = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda")
    W = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    s.mdot_batch(nrhs, dev(torch, F).reshape(-1), None if T is None else dev(torch, T).reshape(-1), U, W)
    torch.cuda.synchronize()
    U = U.cpu().numpy().reshape(nrhs, N, 3)
    W = W.cpu().numpy().reshape(nrhs, N, 3) if angular else None
    for q in range(nrhs):
        if with_wall:
            Uo, Wo = wall.mdot(c["pos"], F[q], None if T is None else T[q], wall_z=c["wall_z"], angular=angular)
        else:
            Uo, Wo = rpy.mdot(c["pos"], F[q], None if T is None else T[q], angular=angular)
        assert close(U[q], Uo, TOL[prec]), (q, rel(U[q], Uo))
        if angular:
            assert close(W[q], Wo, TOL[prec]), (q, rel(W[q], Wo))
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N", [257, 5000])
def test_steric_kernel(lm, torch, prec, N):
    c = workloads.random_case(N, 1.6 * N ** (1.0 / 3.0), 5, prec, False)
    s = lm.Solver(prec, N)
    s.set_positions(dev(torch, c["pos"]))
    out = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.steric_forces(4.0, 0.1, None, out)
    torch.cuda.synchronize()
    Fo = bd.steric_forces(c["pos"], 4.0, 0.1, 2.0)
    assert close(out.cpu().numpy(), Fo, 1e-11 if prec == "f64" else 2e-5), rel(out.cpu().numpy(), Fo)
    s.close()


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
@pytest.mark.parametrize("N,graph,small", [(300, 1, 1), (300, 0, 1), (300, 1, 0), (300, 0, 0), (9000, 0, 0)])
def test_lanczos_fixed_iterations(lm, torch, prec, angular, N, graph, small):
    """Five Lanczos iterations (look-ahead; graph replay on or off) against the fp64 Lanczos oracle stopped at the same
    step, on the three driver paths: small N with the one-launch apply + fused vector step (rpy_small_kernel reading
    V[*newest], lanczos_fused_step_kernel), small N on the general kernels, and N = 9000 where the alpha kernel sums the
    j-split partials itself."""
    c = workloads.random_case(N, 2.0 * N ** (1.0 / 3.0), 9, prec, angular, with_noise=True)
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_option(lm.LM_OPT_GRAPH_REPLAY, graph)
    s.set_option(lm.LM_OPT_SMALL_KERNEL, small)
    s.set_positions(dev(torch, c["pos"]))
    s.set_max_iter(5)
    y = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    ya = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    it = s.sqrt_mdot_w(dev(torch, c["noise"]), 1e-30, y, ya, allow_noconv=True)
    torch.cuda.synchronize()
    got = np.concatenate([y.cpu().numpy()] + ([ya.cpu().numpy()] if angular else []))
    yo, ko, conv = rpy.lanczos_sqrt_mdot_w(c["pos"], c["noise"], 1e-30, angular=angular, max_iter=5)
    assert it == ko == 5 and not conv
    assert rel(got, yo) <= (1e-10 if prec == "f64" else 2e-5), rel(got, yo)
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_one_bd_step_above_a_wall(lm, torch, prec):
    """lm_bd_step_rfd: steric + wall forces, M.[F;T] sharing the first Lanczos launch, RFD drift, Adams-Bashforth update."""
    N = 200
    c = workloads.wall_slab_case(N, 14.0, 0.8, 4.0, 3, prec, False, with_noise=True)
    rng = np.random.default_rng(1)
    dt = workloads.np_dtype(prec)
    rfd = rng.standard_normal(3 * N).astype(dt)
    ext = rng.standard_normal((N, 3)).astype(dt)
    s = lm.Solver(prec, N)
    s.set_wall(True, c["wall_z"])
    X = dev(torch, c["pos"]).reshape(-1).clone()
    s.set_max_iter(300)
    s.bd_step_rfd(X, dev(torch, ext).reshape(-1), None, dev(torch, c["noise"]), dev(torch, rfd), 1e-3 if prec == "f64" else 0.05, 0.01, 0.5, 4.0, 0.1, 1e-3)
    torch.cuda.synchronize()
    new, v, info = wall.bd_step(c["pos"], None, 0.01, 0.5, wall_z=c["wall_z"], U0=4.0, b=0.1, ext_forces=ext, noise=c["noise"], rfd_noise=rfd,
                                delta=1e-3 if prec == "f64" else 0.05, sqrt_mode="dense")
    disp_gpu = X.cpu().numpy().reshape(N, 3).astype(np.float64) - c["pos"].astype(np.float64)
    disp_ora = new - c["pos"].astype(np.float64)
    # the displacement is dominated by the noise term: 3 tol (S4 iii); fp32: + the difference quotient of the drift
    assert rel(disp_gpu, disp_ora) <= 3e-3 + (0.0 if prec == "f64" else 2e-3), rel(disp_gpu, disp_ora)
    s.close()
