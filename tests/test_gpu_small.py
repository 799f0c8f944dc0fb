"""GPU parity of the one-launch small-N kernel (csrc/rpy_small.cuh; "< 50K particles", PAPER.md:435-437:
the regime where launch overhead sets the time): every cluster size x warp count the launch chooser may pick, both
precisions, translational / angular, 1-4 right-hand sides, free space and single wall, ragged N, null inputs, row
ranges -- against the CPU oracle, element by element (same gates as tests/test_gpu_parity.py)."""
import numpy as np
import pytest

from oracle import rpy, wall
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


def case(N, side, nrhs, prec, angular, seed):
    rng = np.random.default_rng(seed)
    dt = workloads.np_dtype(prec)
    pos = (rng.random((N, 3)) * side).astype(dt)
    F = rng.standard_normal((nrhs, N, 3)).astype(dt)
    T = rng.standard_normal((nrhs, N, 3)).astype(dt) if angular else None
    return pos, F, T


def run(lm, torch, prec, pos, F, T, angular, mode, wall_z=None, a=1.0, eta=1.0):
    """mdot_batch of the nrhs right-hand sides with LM_OPT_SMALL_KERNEL = mode; returns (U, W, launch config, stats)."""
    nrhs, N = F.shape[0], pos.shape[0]
    s = lm.Solver(prec, N, eta, a, angular)
    if wall_z is not None:
        s.set_wall(True, wall_z)
    s.set_option(lm.LM_OPT_SMALL_KERNEL, mode)
    s.set_positions(dev(torch, pos))
    U = torch.full((nrhs * 3 * N,), float("nan"), dtype=s.torch_dtype, device="cuda")
    W = torch.full((nrhs * 3 * N,), float("nan"), dtype=s.torch_dtype, device="cuda") if angular else None
    s.reset_stats()
    s.mdot_batch(nrhs, dev(torch, F).reshape(-1), None if T is None else dev(torch, T).reshape(-1), U, W)
    torch.cuda.synchronize()
    cfg, st = s.pair_launch_config(nrhs if nrhs in (1, 2, 4) else 1), s.get_stats()
    s.close()
    return U.cpu().numpy().reshape(nrhs, N, 3), (W.cpu().numpy().reshape(nrhs, N, 3) if angular else None), cfg, st


def oracle(pos, F, T, angular, wall_z=None, a=1.0, eta=1.0):
    if wall_z is None:
        return rpy.mdot(pos, F, T, a=a, eta=eta, angular=angular)
    return wall.mdot(pos, F, T, a=a, eta=eta, wall_z=wall_z, angular=angular)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("S,W", [(1, 1), (1, 4), (2, 2), (4, 1), (4, 8), (8, 4), (8, 8)])
def test_every_shape_matches_the_oracle(lm, torch, prec, angular, S, W):
    """Forced cluster size S and warps per CTA W; N = 777 is ragged in every unit (64 targets, 4 sources, S x W warps)."""
    pos, F, T = case(777, 11.0, 1, prec, angular, 100 + 8 * S + W)
    U, Wv, cfg, st = run(lm, torch, prec, pos, F, T, angular, (S << 8) | W)
    assert (cfg["j_splits"], cfg["block"]) == (S, 32 * W) and cfg["i_tiles"] == 13
    assert st["pair_kernel_launches"] == 1 and st["aux_launches"] == 0          # ONE kernel, nothing else
    Uo, Wo = oracle(pos, F[0], None if T is None else T[0], angular)
    assert close(U[0], Uo, TOL[prec]), rel(U[0], Uo)
    if angular:
        assert close(Wv[0], Wo, TOL[prec]), rel(Wv[0], Wo)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular,nrhs", [(False, 1), (False, 2), (False, 3), (False, 4), (False, 7), (True, 1), (True, 2), (True, 3)])
@pytest.mark.parametrize("N,side", [(1, 1.0), (3, 0.5), (63, 4.0), (65, 4.0), (1024, 40.0), (2500, 30.0)])
def test_chosen_shape_all_rhs_counts(lm, torch, prec, angular, nrhs, N, side):
    pos, F, T = case(N, side, nrhs, prec, angular, 7 * N + nrhs)
    U, Wv, cfg, st = run(lm, torch, prec, pos, F, T, angular, 1)
    if N <= 256 or (N <= 1024 and nrhs == 1 and not angular):
        assert st["aux_launches"] == 0, "these sizes take the one-launch kernel"
    for q in range(nrhs):
        Uo, Wo = oracle(pos, F[q], None if T is None else T[q], angular)
        assert close(U[q], Uo, TOL[prec]), (q, rel(U[q], Uo))
        if angular:
            assert close(Wv[q], Wo, TOL[prec]), (q, rel(Wv[q], Wo))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular,nrhs", [(False, 1), (False, 2), (True, 1), (True, 2)])
@pytest.mark.parametrize("mode", [1, (8 << 8) | 2])
def test_single_wall(lm, torch, prec, angular, nrhs, mode):
    c = workloads.wall_slab_case(900, 14.0, -0.3, 3.0, 900 + nrhs, prec, angular, wall_z=-1.25)
    rng = np.random.default_rng(5)
    F = np.stack([c["forces"]] + [rng.standard_normal(c["forces"].shape).astype(c["forces"].dtype) for _ in range(nrhs - 1)])
    T = None if not angular else np.stack([c["torques"]] + [rng.standard_normal(c["forces"].shape).astype(c["forces"].dtype) for _ in range(nrhs - 1)])
    U, Wv, cfg, st = run(lm, torch, prec, c["pos"], F, T, angular, mode, wall_z=c["wall_z"])
    # a forced shape always runs the one-launch kernel; left to the chooser, the register-heavy fp64 variants hand over early
    assert (st["aux_launches"] == 0) == (cfg["kernel"] == "rpy_small_kernel") and (mode == 1 or cfg["kernel"] == "rpy_small_kernel")
    for q in range(nrhs):
        Uo, Wo = oracle(c["pos"], F[q], None if T is None else T[q], angular, wall_z=c["wall_z"])
        assert close(U[q], Uo, TOL[prec]), (q, rel(U[q], Uo))
        if angular:
            assert close(Wv[q], Wo, TOL[prec]), (q, rel(Wv[q], Wo))


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_agrees_with_the_general_path_and_null_inputs(lm, torch, prec):
    """Same call with the small kernel off (pack, pair kernel, reduce): equal up to summation order; null forces or
    torques mean zeros; degenerate pairs (r = 0, r = 2a exactly) and a non-unit (a, eta)."""
    a, eta = 0.7, 2.5
    pos, F, T = case(1100, 14.0, 1, prec, True, 3)
    pos[1] = pos[0]                                   # coincident distinct particles (reading S5)
    pos[3] = pos[2] + np.array([2 * a, 0, 0], dtype=pos.dtype)
    Us, Ws, cfg_s, st_s = run(lm, torch, prec, pos, F, T, True, 1, a=a, eta=eta)
    Ug, Wg, cfg_g, st_g = run(lm, torch, prec, pos, F, T, True, 0, a=a, eta=eta)
    assert st_s["aux_launches"] == 0 and st_g["aux_launches"] >= 1
    assert rel(Us, Ug) <= TOL[prec] and rel(Ws, Wg) <= TOL[prec]
    Uo, Wo = oracle(pos, F[0], T[0], True, a=a, eta=eta)
    assert close(Us[0], Uo, TOL[prec]) and close(Ws[0], Wo, TOL[prec])
    N = pos.shape[0]
    s = lm.Solver(prec, N, eta, a, True)
    s.set_positions(dev(torch, pos))
    U = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    W = torch.empty_like(U)
    s.mdot(None, dev(torch, T[0]), U, W)
    torch.cuda.synchronize()
    Uo, Wo = oracle(pos, None, T[0], True, a=a, eta=eta)
    assert close(U.cpu().numpy(), Uo, TOL[prec]) and close(W.cpu().numpy(), Wo, TOL[prec])
    s.mdot(dev(torch, F[0]), None, U, W)
    torch.cuda.synchronize()
    Uo, Wo = oracle(pos, F[0], None, True, a=a, eta=eta)
    assert close(U.cpu().numpy(), Uo, TOL[prec]) and close(W.cpu().numpy(), Wo, TOL[prec])
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_row_ranges(lm, torch, prec):
    """lm_mdot_rows on the one-launch kernel: rows [b, b + n) against all sources, nothing written outside them."""
    pos, F, T = case(1500, 20.0, 1, prec, False, 11)
    N = pos.shape[0]
    s = lm.Solver(prec, N, 1.0, 1.0, False)
    s.set_positions(dev(torch, pos))
    Uo, _ = oracle(pos, F[0], None, False)
    for b, n in ((0, 1), (0, 64), (37, 900), (1499, 1), (700, 800), (5, 0), (1500, 0)):      # incl. empty row ranges: nothing written
        U = torch.full((3 * N,), 7.0, dtype=s.torch_dtype, device="cuda")
        s.mdot_rows(b, n, dev(torch, F[0]), None, U)
        torch.cuda.synchronize()
        got = U.cpu().numpy().reshape(N, 3)
        if n:
            assert close(got[b:b + n], Uo[b:b + n], TOL[prec])
        assert np.all(got[:b] == 7.0) and np.all(got[b + n:] == 7.0)
    s.close()


def test_option_values(lm, torch):
    s = lm.Solver("f32", 100, 1.0, 1.0, False)
    for bad in (-1, 2, (3 << 8) | 4, (16 << 8) | 4, (4 << 8) | 3, (4 << 8) | 16):
        with pytest.raises(lm.LmError):
            s.set_option(lm.LM_OPT_SMALL_KERNEL, bad)
    s.set_option(lm.LM_OPT_SMALL_KERNEL, 0)
    assert s.pair_launch_config(1)["block"] in (64, 256)          # the general path's shapes
    s.set_option(lm.LM_OPT_SMALL_KERNEL, (2 << 8) | 4)
    assert s.pair_launch_config(1)["block"] == 128 and s.pair_launch_config(1)["j_splits"] == 2
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_applies_can_be_captured_in_a_callers_cuda_graph(lm, torch, prec):
    """The one-launch apply makes no host decisions and synchronises nothing: a caller may capture a whole batch of
    lm_mdot calls in a CUDA graph of their own (graph kernel nodes are not subject to the 2.048 us stream-launch grid,
    DESIGN.md sec. 5) and replay it on new data."""
    pos, F, T = case(900, 13.0, 1, prec, False, 21)
    N = pos.shape[0]
    s = lm.Solver(prec, N)
    s.set_positions(dev(torch, pos))
    Fd = dev(torch, F[0]).reshape(-1).clone()
    U1 = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    U2 = torch.empty_like(U1)
    s.mdot(Fd, None, U1)                                        # warm-up outside the capture (plans, attributes)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            s.mdot(Fd, None, U1)                                # U1 = M F
            s.mdot(U1, None, U2)                                # U2 = M M F: the second node depends on the first
    for scale in (1.0, -2.5):
        Fd.copy_(dev(torch, F[0]).reshape(-1) * scale)
        g.replay()
        torch.cuda.synchronize()
        Uo, _ = oracle(pos, F[0].astype(np.float64) * scale, None, False)
        UUo, _ = oracle(pos, Uo, None, False)
        assert close(U1.cpu().numpy(), Uo, TOL[prec]) and close(U2.cpu().numpy(), UUo, 2 * TOL[prec])
    s.close()
