"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle.

Tolerances (BASELINE.json north_star): rel-L2 <= 1e-12 in fp64, <= 2e-5 in fp32 for M.F;
Lanczos gates per DESIGN.md S4.  The oracle receives the SAME already-rounded inputs (S11).
All tests here need a B200 (``-m gpu``).
"""
import math

import numpy as np
import pytest

from oracle import rpy
from paper_2510_02135_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def close(a, b, tol):
    """The M.F gate: rel-L2 <= tol (north_star) AND every element within 8 tol of the largest entry (one bad row
    in a million passes a norm)."""
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return rel(a, b) <= tol and np.abs(a - b).max() <= 8 * tol * np.abs(b).max()


def lanczos_gates(rule, prec, it, ko, y, yo, tol, tag=()):
    """S4(ii): the CUDA path and the fp64 Lanczos oracle run the SAME stopping rule.  Plain Lanczos (no
    re-orthogonalisation, S15) amplifies rounding differences geometrically once the top Ritz values have converged
    (k >~ 15-20), and the stop step is a discontinuous function of the steps, so: while the two fp64 recurrences
    still coincide (k <= 20) the stop step is the oracle's and the iterates agree to 1e-6; beyond that, and in
    fp32, the stop steps agree within max(2, k/3) (measured: up to +27 % in fp32, whose noisier steps raise the
    rule's ratio estimate) and the two results -- both within the rule's error of the exact root -- within 2 tol of
    each other (rule "estimate"; the rule of ref. [35], "step", under-states the error, its iterates at nearby steps
    differ by the true error: 12 tol at tol >= 1e-3, 50 tol below, as against the dense root)."""
    if prec == "f64" and ko <= 20:
        assert it == ko, (tag, it, ko)
        assert rel(y, yo) <= 1e-6, (tag, rel(y, yo))
    else:
        assert abs(it - ko) <= max(2, ko // 3), (tag, it, ko)
        assert rel(y, yo) <= (2 if rule == "estimate" else (12 if tol >= 1e-3 else 50)) * tol, (tag, it, ko, rel(y, yo))


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


def gpu_mdot(lm, torch, prec, pos, F, T, angular, a=1.0, eta=1.0):
    N = pos.shape[0]
    s = lm.Solver(prec, N, eta, a, angular)
    s.set_positions(dev(torch, pos))
    U = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    W = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    s.mdot(dev(torch, F), dev(torch, T), U, W)
    torch.cuda.synchronize()
    return U.cpu().numpy().reshape(N, 3), (W.cpu().numpy().reshape(N, 3) if angular else None), s


# ---------------------------------------------------------------- M.F, element by element, small and ragged sizes
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("N,side", [(1, 1.0), (2, 1.5), (3, 0.5), (37, 4.0), (129, 5.0), (511, 9.0), (513, 9.0),
                                    (1500, 20.0), (4099, 30.0), (9000, 45.0)])
def test_mdot_matches_oracle(lm, torch, prec, angular, N, side):
    """Spans one thread, one tile, tile boundaries +-1, several tiles with a ragged tail, both
    kernel variants (SMALL below ~8k, LARGE above) and split-j with its reduce pass."""
    case = workloads.random_case(N, side, seed=100 + N, precision=prec, angular=angular)
    U, W, _ = gpu_mdot(lm, torch, prec, case["pos"], case["forces"], case["torques"], angular)
    Uo, Wo = rpy.mdot(case["pos"], case["forces"], case["torques"], angular=angular)
    assert rel(U, Uo) <= TOL[prec]
    # element by element: every component within tol of the row scale
    assert np.abs(U - Uo).max() <= TOL[prec] * 8 * np.abs(Uo).max()
    if angular:
        assert rel(W, Wo) <= TOL[prec]
        assert np.abs(W - Wo).max() <= TOL[prec] * 8 * np.abs(Wo).max()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_mdot_nonunit_radius_viscosity(lm, torch, prec):
    rng = np.random.default_rng(3)
    N, a, eta = 700, 0.656, 1.0e-3          # the paper's microroller radius in um
    dt = workloads.np_dtype(prec)
    pos = (rng.random((N, 3)) * 12 * a).astype(dt)
    F, T = rng.standard_normal((N, 3)).astype(dt), rng.standard_normal((N, 3)).astype(dt)
    U, W, _ = gpu_mdot(lm, torch, prec, pos, F, T, True, a=a, eta=eta)
    Uo, Wo = rpy.mdot(pos, F, T, a=a, eta=eta, angular=True)
    assert rel(U, Uo) <= TOL[prec] and rel(W, Wo) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_degenerate_pairs(lm, torch, prec):
    """Exactly coincident distinct particles (r = 0 off the diagonal, S5), a pair exactly at
    contact r = 2a (S2), and near-contact on both sides."""
    dt = workloads.np_dtype(prec)
    pos = np.array([[0, 0, 0], [0, 0, 0], [2, 0, 0], [2, 0, 1.9999], [2, 2.0001, 0], [10, 10, 10]], dtype=dt)
    rng = np.random.default_rng(1)
    F, T = rng.standard_normal((6, 3)).astype(dt), rng.standard_normal((6, 3)).astype(dt)
    U, W, _ = gpu_mdot(lm, torch, prec, pos, F, T, True)
    Uo, Wo = rpy.mdot(pos, F, T, angular=True)
    assert np.isfinite(U).all() and np.isfinite(W).all()
    assert rel(U, Uo) <= TOL[prec] and rel(W, Wo) <= TOL[prec]


def test_self_mobility_on_gpu(lm, torch):
    """P1 through the CUDA path: N = 1 gives F/(6 pi eta a) and T/(8 pi eta a^3)."""
    a, eta = 1.7, 0.4
    F, T = np.array([[0.3, -2.0, 1.5]]), np.array([[1.0, 0.25, -0.5]])
    U, W, _ = gpu_mdot(lm, torch, "f64", np.array([[4.0, -1.0, 2.0]]), F, T, True, a=a, eta=eta)
    np.testing.assert_allclose(U, F / (6 * math.pi * eta * a), rtol=1e-14)
    np.testing.assert_allclose(W, T / (8 * math.pi * eta * a ** 3), rtol=1e-14)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_null_forces_or_torques_mean_zero(lm, torch, prec):
    case = workloads.random_case(300, 8.0, 5, prec, True)
    U1, W1, _ = gpu_mdot(lm, torch, prec, case["pos"], None, case["torques"], True)
    Uo, Wo = rpy.mdot(case["pos"], None, case["torques"], angular=True)
    assert rel(U1, Uo) <= TOL[prec] and rel(W1, Wo) <= TOL[prec]
    U2, W2, _ = gpu_mdot(lm, torch, prec, case["pos"], case["forces"], None, True)
    Uo, Wo = rpy.mdot(case["pos"], case["forces"], None, angular=True)
    assert rel(U2, Uo) <= TOL[prec] and rel(W2, Wo) <= TOL[prec]


# ---------------------------------------------------------------- multi-RHS
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 5, 7])
def test_mdot_batch(lm, torch, prec, angular, nrhs):
    N = 1300
    dt = workloads.np_dtype(prec)
    rng = np.random.default_rng(nrhs)
    pos = (rng.random((N, 3)) * 18).astype(dt)
    F = rng.standard_normal((nrhs, N, 3)).astype(dt)
    T = rng.standard_normal((nrhs, N, 3)).astype(dt) if angular else None
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_positions(dev(torch, pos))
    U = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda")
    W = torch.empty_like(U) if angular else None
    s.mdot_batch(nrhs, dev(torch, F), dev(torch, T), U, W)
    torch.cuda.synchronize()
    U = U.cpu().numpy().reshape(nrhs, N, 3)
    for q in range(nrhs):
        Uo, Wo = rpy.mdot(pos, F[q], T[q] if angular else None, angular=angular)
        assert close(U[q], Uo, TOL[prec])
        if angular:
            assert close(W.cpu().numpy().reshape(nrhs, N, 3)[q], Wo, TOL[prec])


# ---------------------------------------------------------------- the five configs
def test_config1_full(lm, torch):
    d = workloads.generate(1)
    U, _, s = gpu_mdot(lm, torch, "f64", d["pos"], d["forces"], None, False)
    Uo, _ = rpy.mdot(d["pos"], d["forces"])
    assert close(U, Uo, 1e-12)


def test_config2_full(lm, torch):
    d = workloads.generate(2)
    U, W, s = gpu_mdot(lm, torch, "f32", d["pos"], d["forces"], d["torques"], True)
    Uo, Wo = rpy.mdot(d["pos"], d["forces"], d["torques"], angular=True)
    assert close(U, Uo, 2e-5) and close(W, Wo, 2e-5)


def _sampled_rows(N, n, seed):
    rows = np.random.default_rng(seed).choice(N, n, replace=False)
    rows[:4] = [0, 1, N - 2, N - 1]              # first / last rows: tile edges
    return np.sort(rows)


def test_config3_full_size_sampled_rows(lm, torch):
    """Full N = 131072 in the launch configuration bench.py times; the oracle computes 192 target
    rows exactly (rows are independent)."""
    d = workloads.generate(3)
    U, _, s = gpu_mdot(lm, torch, "f32", d["pos"], d["forces"], None, False)
    rows = _sampled_rows(d["N"], 192, 3)
    Uo, _ = rpy.mdot_rows(d["pos"], rows, d["forces"])
    assert rel(U[rows], Uo) <= 2e-5
    assert np.abs(U[rows] - Uo).max() <= 2e-5 * 8 * np.abs(Uo).max()


def test_config4_full_size_sampled_rows(lm, torch):
    d = workloads.generate(4)
    N = d["N"]
    s = lm.Solver("f32", N)
    s.set_positions(dev(torch, d["pos"]))
    U = torch.empty(4 * 3 * N, dtype=torch.float32, device="cuda")
    s.mdot_batch(4, dev(torch, d["forces"]), None, U)
    torch.cuda.synchronize()
    U = U.cpu().numpy().reshape(4, N, 3)
    rows = _sampled_rows(N, 48, 4)
    for q in range(4):
        Uo, _ = rpy.mdot_rows(d["pos"], rows, d["forces"][q])
        assert close(U[q][rows], Uo, 2e-5)


def test_config5_full_size_sampled_rows(lm, torch):
    d = workloads.generate(5)
    U, W, s = gpu_mdot(lm, torch, "f64", d["pos"], d["forces"], d["torques"], True)
    rows = _sampled_rows(d["N"], 96, 5)
    Uo, Wo = rpy.mdot_rows(d["pos"], rows, d["forces"], d["torques"], angular=True)
    assert close(U[rows], Uo, 1e-12) and close(W[rows], Wo, 1e-12)


# ---------------------------------------------------------------- Lanczos sqrt(M).W
def gpu_sqrt(lm, torch, prec, pos, noise, tol, angular, max_iter=None, allow_noconv=False, rule=None):
    N = pos.shape[0]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    if max_iter:
        s.set_max_iter(max_iter)
    if rule is not None:
        s.set_option(lm.LM_OPT_LANCZOS_RULE, {"estimate": lm.LM_RULE_ESTIMATE, "step": lm.LM_RULE_STEP}[rule])
    s.set_positions(dev(torch, pos))
    y = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    ya = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    it = s.sqrt_mdot_w(dev(torch, noise), tol, y, ya, allow_noconv=allow_noconv)
    out = y.cpu().numpy() if not angular else np.concatenate([y.cpu().numpy(), ya.cpu().numpy()])
    return out, it, s


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
def test_lanczos_iterates_match_oracle_step_by_step(lm, torch, prec, angular):
    """Algorithmic parity: stop both sides after exactly k steps (tol unreachable, max_iter = k) and
    compare the iterates y_k.  Lanczos without re-orthogonalisation amplifies rounding differences
    roughly geometrically in k, so the bound loosens with k (S4)."""
    case = workloads.random_case(400, 14.0, 21, prec, angular, with_noise=True)
    bounds = {"f64": {3: 1e-12, 6: 1e-11, 10: 1e-9, 14: 1e-7}, "f32": {3: 2e-6, 6: 5e-6, 10: 2e-5, 14: 1e-4}}[prec]
    for k, bound in bounds.items():
        y, it, _ = gpu_sqrt(lm, torch, prec, case["pos"], case["noise"], 1e-30, angular, max_iter=k, allow_noconv=True)
        yo, ko, conv = rpy.lanczos_sqrt_mdot_w(case["pos"], case["noise"], 1e-30, angular=angular, max_iter=k)
        assert it == ko == k and not conv
        assert rel(y, yo) <= bound, (k, rel(y, yo))


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
@pytest.mark.parametrize("rule", ["estimate", "step"])
def test_lanczos_stopping_rule_vs_oracle_lanczos_and_dense(lm, torch, prec, angular, rule):
    """Gates of DESIGN.md S4 for both rules of reading S3.  (i) With the same rule on both sides the CUDA path stops
    at the oracle's step in fp64 and within a few steps in fp32, and the two results agree to O(tol).  (ii) Against
    the exact dense root: rule "estimate" (default) delivers the requested tolerance within a factor 3 (measured here:
    0.3 ... 2.1 tol); rule "step"
    (ref. [35]) under-states the error: <= 10 tol at tol >= 1e-3, <= 50 tol at 1e-5 on this small problem."""
    case = workloads.random_case(400, 14.0, 21, prec, angular, with_noise=True)
    exact = rpy.dense_sqrt_mdot_w(case["pos"], case["noise"], angular=angular)
    tols = (1e-2, 1e-3, 1e-5) if prec == "f64" else (1e-2, 1e-3, 1e-4)
    for tol in tols:
        y, it, s = gpu_sqrt(lm, torch, prec, case["pos"], case["noise"], tol, angular, rule=rule)
        yo, ko, conv = rpy.lanczos_sqrt_mdot_w(case["pos"], case["noise"], tol, angular=angular, rule=rule)
        assert conv
        lanczos_gates(rule, prec, it, ko, y, yo, tol, tol)
        slack = 3.0 if rule == "estimate" else (10.0 if tol >= 1e-3 else 50.0)
        assert rel(y, exact) <= slack * tol, (tol, it, rel(y, exact))
        # the history the library reports is the one it stopped on
        hist = s.lanczos_history()
        assert len(hist["alpha"]) == it and np.isnan(hist["step"][0]) and np.all(hist["step"][1:] > 0)
        if rule == "estimate":
            assert hist["estimate"][-1] <= tol and np.all(hist["estimate"][2:-1] > tol)
            assert hist["estimate"][-1] == pytest.approx(rpy.step_error_estimate(hist["step"][1:]), rel=1e-12)
        else:
            assert hist["step"][-1] <= tol and np.all(hist["step"][1:-1] > tol) and np.all(np.isnan(hist["estimate"]))
        s.close()


def _memo_apply(pos):
    """The oracle's O(N^2) apply with a cache keyed on the input vector: the Lanczos oracle called again with a
    larger max_iter (or another stopping rule) replays the same sequence of applies, each ~20 s at N = 131072."""
    cache = {}

    def apply(v):
        key = hash(v.tobytes())
        if key not in cache:
            cache[key] = rpy.apply_vec(pos, v)
        return cache[key]
    return apply


def test_lanczos_large_n_path_fixed_k_iterates_vs_oracle_config3(lm, torch):
    """The driver path config 3 and bench.py run (N = 131072: direct launches, no look-ahead, the alpha kernel
    summing the 37 j-split partials) against the fp64 Lanczos oracle: fixed k (max_iter = k, tol unreachable) for
    k = 2, 4, 6 -- six full O(N^2) oracle applies.  Gates as test_lanczos_iterates_match_oracle_step_by_step."""
    d = workloads.generate(3)
    apply = _memo_apply(d["pos"])
    for k, bound in ((2, 2e-6), (4, 3e-6), (6, 5e-6)):
        y, it, s = gpu_sqrt(lm, torch, "f32", d["pos"], d["noise"], 1e-30, False, max_iter=k, allow_noconv=True)
        cfgl = s.pair_launch_config(1)
        assert cfgl["j_splits"] > 1                         # the fused split-j reduce is on this path
        yo, ko, conv = rpy.lanczos_sqrt_mdot_w(d["pos"], d["noise"], 1e-30, max_iter=k, apply=apply)
        assert it == ko == k and not conv
        assert rel(y, yo) <= bound, (k, rel(y, yo))
        assert np.abs(y - yo).max() <= 8 * bound * np.abs(yo).max()
        s.close()


def test_hydrodynamic_velocities_config3_vs_oracle(lm, torch):
    """lm_hydrodynamic_velocities -- the call bench.py times -- at config 3: with max_iter = 3 the result is
    M.F + prefactor * y_3; the oracle gives M.F on sampled rows (exact for those rows) and y_3 from three full
    applies.  Also checks that the shared first launch (M.F riding along with the first Lanczos apply, a 2-RHS
    launch) and the separate launches give the same answer."""
    d = workloads.generate(3)
    N, pref = d["N"], 0.37
    s = lm.Solver("f32", N)
    s.set_positions(dev(torch, d["pos"]))
    s.set_max_iter(3)
    F, z = dev(torch, d["forces"]), dev(torch, d["noise"])
    H = torch.empty(3 * N, dtype=torch.float32, device="cuda")
    H2 = torch.empty_like(H)
    s.reset_stats()
    with pytest.raises(lm.LmError) as ei:
        s.hydrodynamic_velocities(F, None, z, pref, 1e-30, H)
    assert ei.value.code == lm.LM_E_NOCONV                  # the result is still written
    assert s.get_stats()["pair_kernel_launches"] == 3       # 1 shared 2-RHS launch + 2, not 1 + 3
    s.set_option(lm.LM_OPT_SHARE_FIRST_APPLY, 0)
    s.reset_stats()
    with pytest.raises(lm.LmError):
        s.hydrodynamic_velocities(F, None, z, pref, 1e-30, H2)
    assert s.get_stats()["pair_kernel_launches"] == 4
    torch.cuda.synchronize()
    H, H2 = H.cpu().numpy().reshape(N, 3), H2.cpu().numpy().reshape(N, 3)
    assert rel(H, H2) <= 2e-6
    y3, k3, _ = rpy.lanczos_sqrt_mdot_w(d["pos"], d["noise"], 1e-30, max_iter=3, apply=_memo_apply(d["pos"]))
    rows = _sampled_rows(N, 192, 33)
    Uo, _ = rpy.mdot_rows(d["pos"], rows, d["forces"])
    want = Uo + pref * y3.reshape(N, 3)[rows]
    assert close(H[rows], want, 2e-5) and close(H2[rows], want, 2e-5)
    s.close()


@pytest.mark.parametrize("rule,tol", [("step", 1e-3), ("estimate", 1e-2)])
def test_lanczos_large_n_path_stopping_rule_vs_oracle(lm, torch, rule, tol):
    """N = 65536 at phi = 5 % (config 3's recipe at half size; still the direct-launch path) with the stopping rule on
    both sides.  The oracle runs the whole fp64 recurrence (~30-40 O(N^2) applies, shared between the two rules
    through the apply cache).  Gates S4(ii), lanczos_gates above: stop step within max(2, k/3), results within 2 tol
    ("estimate") of each other; for the rule of ref. [35] ("step") the iterates of nearby steps differ by the true
    error, measured ~10 tol here, so its gate is the step count and 12 tol."""
    N = 65536
    d = workloads.generate(3, N)
    if not hasattr(test_lanczos_large_n_path_stopping_rule_vs_oracle, "apply"):
        test_lanczos_large_n_path_stopping_rule_vs_oracle.apply = _memo_apply(d["pos"])
    y, it, s = gpu_sqrt(lm, torch, "f32", d["pos"], d["noise"], tol, False, rule=rule)
    assert s.pair_launch_config(1)["j_splits"] > 1
    yo, ko, conv = rpy.lanczos_sqrt_mdot_w(d["pos"], d["noise"], tol, rule=rule, apply=test_lanczos_large_n_path_stopping_rule_vs_oracle.apply)
    assert conv
    lanczos_gates(rule, "f32", it, ko, y, yo, tol, rule)
    s.close()


def test_lanczos_config3_true_error_of_the_default_rule(lm, torch):
    """What tol means at the headline config: the tol = 1e-3 iterate (default rule, fp32) against a 300-step fp64
    run of the same CUDA recurrence -- itself checked against the oracle step by step above -- is within 3 tol;
    the rule of ref. [35] stops ~3x earlier at 15-20 tol (asserted only to be worse, S3/S4)."""
    d = workloads.generate(3)
    N = d["N"]
    s64 = lm.Solver("f64", N)
    s64.set_positions(dev(torch, d["pos"].astype(np.float64)))
    s64.set_max_iter(300)
    yref = torch.empty(3 * N, dtype=torch.float64, device="cuda")
    s64.sqrt_mdot_w(dev(torch, d["noise"].astype(np.float64)), 1e-9, yref, None, allow_noconv=True)
    yref = yref.cpu().numpy()
    s64.close()
    y, it, s = gpu_sqrt(lm, torch, "f32", d["pos"], d["noise"], 1e-3, False)
    e_est = rel(y, yref)
    s.close()
    ys, its, s = gpu_sqrt(lm, torch, "f32", d["pos"], d["noise"], 1e-3, False, rule="step")
    e_step = rel(ys, yref)
    s.close()
    assert 40 <= it <= 100 and e_est <= 3e-3, (it, e_est)
    assert its < it and e_step > e_est, (its, e_step)


def test_lanczos_square_root_twice_config3_size(lm, torch):
    """P10(ii) at the full config-3 size, no dense matrix: sqrt(M) sqrt(M) z = M z."""
    d = workloads.generate(3)
    N = d["N"]
    s = lm.Solver("f32", N)
    s.set_positions(dev(torch, d["pos"]))
    z = dev(torch, d["noise"])
    y1 = torch.empty_like(z)
    y2 = torch.empty_like(z)
    Mz = torch.empty_like(z)
    errs = {}
    for tol in (1e-2, 3e-3):      # (at this N the default rule needs ~70 steps for 1e-3 and > 100 for 3e-4, in fp64 too)
        it1 = s.sqrt_mdot_w(z, tol, y1)
        it2 = s.sqrt_mdot_w(y1, tol, y2)
        s.mdot(z, None, Mz)
        torch.cuda.synchronize()
        assert 5 < it1 < 100 and 5 < it2 < 100
        errs[tol] = rel(y2.cpu().numpy(), Mz.cpu().numpy())
    # two applications, each within ~2 tol of the exact root (default rule, S4)
    assert errs[1e-2] <= 6 * 1e-2, errs
    assert errs[3e-3] <= 6 * 3e-3 and errs[3e-3] < errs[1e-2], errs


def test_lanczos_exact_cases_and_noconv(lm, torch):
    # N = 1: M = I/(6 pi), sqrt(M) z = z / sqrt(6 pi), found in one step (breakdown: beta = 0)
    z = np.array([0.5, -1.0, 2.0])
    y, it, _ = gpu_sqrt(lm, torch, "f64", np.zeros((1, 3)), z, 1e-8, False)
    np.testing.assert_allclose(y, z / math.sqrt(6 * math.pi), rtol=1e-13)
    assert it == 1
    # zero noise -> zero output, zero iterations
    y, it, _ = gpu_sqrt(lm, torch, "f32", np.zeros((5, 3), dtype=np.float32), np.zeros(15, dtype=np.float32), 1e-3, False)
    assert it == 0 and not y.any()
    # max_iter reached: LM_E_NOCONV but the iterate is written
    case = workloads.random_case(200, 6.0, 2, "f64", False, with_noise=True)
    y, it, s = gpu_sqrt(lm, torch, "f64", case["pos"], case["noise"], 1e-12, False, max_iter=4, allow_noconv=True)
    assert it == 4 and "max_iter" in s.last_error()
    yo, ko, conv = rpy.lanczos_sqrt_mdot_w(case["pos"], case["noise"], 1e-12, max_iter=4)
    assert not conv and rel(y, yo) <= 1e-9
    with pytest.raises(lm.LmError) as ei:
        gpu_sqrt(lm, torch, "f64", case["pos"], case["noise"], 1e-12, False, max_iter=4)
    assert ei.value.code == lm.LM_E_NOCONV


def test_fluctuation_dissipation_ks(lm, torch):
    """eq. (12): M_SVD^{-1/2} (M^{1/2} W) ~ N(0,1) over many realisations (KS test),
    and <y y^T> ~ M, with the samples drawn by the CUDA Lanczos path and M from the oracle."""
    from scipy import stats
    rng = np.random.default_rng(12)
    N = 6
    pos = rng.random((N, 3)) * 3.5
    M = rpy.dense(pos, angular=True)
    Uu, sv, Vt = np.linalg.svd(M)
    Minvhalf = Uu @ np.diag(sv ** -0.5) @ Vt
    s = lm.Solver("f64", N, 1.0, 1.0, True)
    s.set_positions(dev(torch, pos))
    nsamp, dof = 1200, 6 * N
    Wn = rng.standard_normal((nsamp, dof))
    Y = np.empty((nsamp, dof))
    yl = torch.empty(3 * N, dtype=torch.float64, device="cuda")
    ya = torch.empty(3 * N, dtype=torch.float64, device="cuda")
    for k in range(nsamp):
        s.sqrt_mdot_w(dev(torch, Wn[k]), 1e-8, yl, ya)
        Y[k] = np.concatenate([yl.cpu().numpy(), ya.cpu().numpy()])
    white = Y @ Minvhalf.T
    assert stats.kstest(white.reshape(-1), "norm").pvalue > 0.01
    assert np.abs(Y.T @ Y / nsamp - M).max() < 6.0 * np.abs(M).max() / math.sqrt(nsamp)
    # each sample also matches the exact root applied to the same noise
    exact = Wn @ (Uu @ np.diag(np.sqrt(sv)) @ Vt).T
    assert rel(Y, exact) <= 1e-6


# ---------------------------------------------------------------- hydrodynamic_velocities and host entry points
@pytest.mark.parametrize("prec,angular", [("f64", True), ("f32", False)])
def test_hydrodynamic_velocities_is_mdot_plus_noise(lm, torch, prec, angular):
    case = workloads.random_case(600, 15.0, 9, prec, angular, with_noise=True)
    N, tol, pref = 600, 1e-3, 0.37
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_positions(dev(torch, case["pos"]))
    F, T, z = dev(torch, case["forces"]), dev(torch, case["torques"]), dev(torch, case["noise"])
    mk = lambda: torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    U, W, yl, ya, Hl, Ha = mk(), (mk() if angular else None), mk(), (mk() if angular else None), mk(), (mk() if angular else None)
    s.mdot(F, T, U, W)
    s.sqrt_mdot_w(z, tol, yl, ya)
    s.hydrodynamic_velocities(F, T, z, pref, tol, Hl, Ha)
    torch.cuda.synchronize()
    want = U.double() + pref * yl.double()
    assert rel(Hl.cpu().numpy(), want.cpu().numpy()) <= (1e-13 if prec == "f64" else 3e-7)
    if angular:
        want = W.double() + pref * ya.double()
        assert rel(Ha.cpu().numpy(), want.cpu().numpy()) <= 1e-13
    # against the oracle: M.F + pref * Lanczos
    Uo, Wo = rpy.mdot(case["pos"], case["forces"], case["torques"], angular=angular)
    yo, _, _ = rpy.lanczos_sqrt_mdot_w(case["pos"], case["noise"], tol, angular=angular)
    assert rel(Hl.cpu().numpy(), Uo.reshape(-1) + pref * yo[:3 * N]) <= 2 * tol
    # noise = None: deterministic part only
    s.hydrodynamic_velocities(F, T, None, 0.0, tol, Hl, Ha)
    torch.cuda.synchronize()
    assert torch.equal(Hl, U)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_host_entry_points_equal_device_entry_points(lm, torch, prec):
    case = workloads.random_case(900, 16.0, 33, prec, True, with_noise=True)
    N = 900
    s = lm.Solver(prec, N, 1.0, 1.0, True)
    s.set_positions_host(case["pos"])
    U, W = np.empty((N, 3), dtype=s.np_dtype), np.empty((N, 3), dtype=s.np_dtype)
    s.mdot_host(case["forces"], case["torques"], U, W)
    Ud, Wd, _ = gpu_mdot(lm, torch, prec, case["pos"], case["forces"], case["torques"], True)
    assert np.array_equal(U, Ud) and np.array_equal(W, Wd)
    yl, ya = np.empty(3 * N, dtype=s.np_dtype), np.empty(3 * N, dtype=s.np_dtype)
    it = s.sqrt_mdot_w_host(case["noise"], 1e-3, yl, ya)
    yd, itd, _ = gpu_sqrt(lm, torch, prec, case["pos"], case["noise"], 1e-3, True)
    assert it == itd and np.array_equal(np.concatenate([yl, ya]), yd)
    Hl, Ha = np.empty(3 * N, dtype=s.np_dtype), np.empty(3 * N, dtype=s.np_dtype)
    s.hydrodynamic_velocities_host(case["forces"], case["torques"], case["noise"], 2.0, 1e-3, Hl, Ha)
    assert rel(Hl, U.reshape(-1).astype(np.float64) + 2.0 * yl) <= (1e-13 if prec == "f64" else 3e-7)
    F4 = np.stack([case["forces"]] * 2)
    U4 = np.empty((2, N, 3), dtype=s.np_dtype)
    W4 = np.empty((2, N, 3), dtype=s.np_dtype)
    s.mdot_batch_host(2, F4, np.stack([case["torques"]] * 2), U4, W4)
    assert rel(U4[1], Ud) <= TOL[prec]


# ---------------------------------------------------------------- API guarantees
def test_error_codes(lm, torch):
    with pytest.raises(lm.LmError) as ei:
        lm.Solver("f32", 0)
    assert ei.value.code == lm.LM_E_INVALID
    for bad in (dict(eta=-1.0), dict(a=0.0)):
        with pytest.raises(lm.LmError):
            lm.Solver("f32", 10, **bad)
    s = lm.Solver("f32", 10)
    x = torch.zeros(30, dtype=torch.float32, device="cuda")
    out = torch.zeros(30, dtype=torch.float32, device="cuda")
    with pytest.raises(lm.LmError) as ei:
        s.mdot(x, None, out)
    assert ei.value.code == lm.LM_E_NOPOS
    s.set_positions(x)
    with pytest.raises(lm.LmError) as ei:
        s.mdot(x, x, out)                        # torques without include_angular
    assert ei.value.code == lm.LM_E_ANGULAR
    with pytest.raises(lm.LmError) as ei:
        s.mdot(None, None, out)
    assert ei.value.code == lm.LM_E_NULL
    with pytest.raises(lm.LmError) as ei:
        s.sqrt_mdot_w(x, 0.0, out)
    assert ei.value.code == lm.LM_E_INVALID
    sa = lm.Solver("f32", 10, include_angular=True)
    sa.set_positions(x)
    with pytest.raises(lm.LmError) as ei:
        sa.mdot(x, x, out, None)                 # angular solver needs ang_out
    assert ei.value.code == lm.LM_E_ANGULAR
    with pytest.raises(lm.LmError):
        s.set_max_iter(0)
    with pytest.raises(TypeError):
        s.mdot(x.double(), None, out)


def test_stats_and_launch_config(lm, torch):
    d = workloads.generate(1)
    U, _, s = gpu_mdot(lm, torch, "f64", d["pos"], d["forces"], None, False)
    st = s.get_stats()
    assert st["pair_kernel_launches"] == 1 and st["pairs"] == 1024.0 ** 2
    cfg = s.pair_launch_config(1)
    assert cfg["i_tiles"] * cfg["j_splits"] >= 32         # small N is split over j to fill the SMs
    s.set_profiling(True)
    s.reset_stats()
    s.mdot(dev(torch, d["forces"]), None, dev(torch, np.empty_like(d["forces"])))
    st = s.get_stats()
    assert st["pair_kernel_launches"] == 1 and st["pair_kernel_ms"] > 0
    from paper_2510_02135_b200 import probe
    assert probe.fma_peak(lm.LM_F32, 0.05) > 1e13


# ---------------------------------------------------------------- several noise vectors per call
@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
@pytest.mark.parametrize("nvec", [2, 3, 4, 7])
def test_sqrt_mdot_w_batch_each_vector_matches_oracle(lm, torch, prec, angular, nvec):
    """Lockstep recurrences on the multi-RHS kernel: every vector must satisfy the single-vector gates (S4)
    against the fp64 Lanczos oracle and the exact dense root, with its own stopping step; groups 4/2/1
    (angular 2/1) and a zero vector in the batch."""
    N, tol = 300, 1e-3
    case = workloads.random_case(N, 12.0, 40 + nvec, prec, angular, with_noise=True)
    dof = (6 if angular else 3) * N
    rng = np.random.default_rng(100 + nvec)
    W = rng.standard_normal((nvec, dof)).astype(workloads.np_dtype(prec))
    W[0] = case["noise"]
    if nvec >= 3:
        W[2] = 0.0                                         # M^{1/2} 0 = 0, zero iterations
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_positions(dev(torch, case["pos"]))
    lin = torch.empty(nvec * 3 * N, dtype=s.torch_dtype, device="cuda")
    ang = torch.empty(nvec * 3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    iters = s.sqrt_mdot_w_batch(nvec, dev(torch, W).reshape(-1), tol, lin, ang)
    torch.cuda.synchronize()
    lin = lin.cpu().numpy().reshape(nvec, 3 * N)
    ang = ang.cpu().numpy().reshape(nvec, 3 * N) if angular else None
    for q in range(nvec):
        y = lin[q] if not angular else np.concatenate([lin[q], ang[q]])
        if nvec >= 3 and q == 2:
            assert iters[q] == 0 and np.all(y == 0.0)
            continue
        yo, ko, conv = rpy.lanczos_sqrt_mdot_w(case["pos"], W[q], tol, angular=angular)
        exact = rpy.dense_sqrt_mdot_w(case["pos"], W[q], angular=angular)
        assert conv
        lanczos_gates("estimate", prec, iters[q], ko, y, yo, tol, q)
        assert rel(y, exact) <= 3 * tol, (q, rel(y, exact))
    # the single-vector call gives the same answer for vector 0 (up to the pair kernel's summation order)
    y1, it1, _ = gpu_sqrt(lm, torch, prec, case["pos"], W[0], tol, angular)
    y0 = lin[0] if not angular else np.concatenate([lin[0], ang[0]])
    assert abs(it1 - iters[0]) <= (1 if prec == "f64" else max(2, it1 // 4)), (it1, iters[0])
    assert rel(y0, y1) <= (1e-5 if prec == "f64" else 2 * tol), rel(y0, y1)
    s.close()


def test_sqrt_mdot_w_batch_noconv_and_errors(lm, torch):
    case = workloads.random_case(200, 8.0, 50, "f64", False, with_noise=True)
    N = 200
    s = lm.Solver("f64", N, 1.0, 1.0, False)
    s.set_positions(dev(torch, case["pos"]))
    W = np.random.default_rng(5).standard_normal((2, 3 * N))
    lin = torch.empty(2 * 3 * N, dtype=torch.float64, device="cuda")
    s.set_max_iter(3)
    with pytest.raises(lm.LmError) as e:
        s.sqrt_mdot_w_batch(2, dev(torch, W).reshape(-1), 1e-12, lin)
    assert e.value.code == lm.LM_E_NOCONV
    its = s.sqrt_mdot_w_batch(2, dev(torch, W).reshape(-1), 1e-12, lin, allow_noconv=True)
    assert its == [3, 3]
    for q in range(2):                                        # the last iterate IS written: 3 plain Lanczos steps
        yo, ko, _ = rpy.lanczos_sqrt_mdot_w(case["pos"], W[q], 1e-12, max_iter=3)
        assert ko == 3 and rel(lin.cpu().numpy().reshape(2, -1)[q], yo) <= 1e-11
    with pytest.raises(lm.LmError) as e:
        s.sqrt_mdot_w_batch(0, dev(torch, W).reshape(-1)[:0], 1e-3, lin[:0])
    assert e.value.code in (lm.LM_E_INVALID, lm.LM_E_NULL)
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("small_kernel", [0, 1])
def test_repeated_small_applies_replay_a_graph_on_current_data(lm, torch, prec, small_kernel):
    """Short applies called again with the same buffers are replayed as a CUDA graph: the
    replay must read the buffers' CURRENT contents (forces changed in place, positions re-set), and calls with
    other buffers, other right-hand-side counts or a row range must not be served by a stale graph.  With the
    one-launch kernel off this size takes the graph-replayed general path (as N ~ 5000 ... 14000 always does); with
    it on, the same sequence of calls runs on rpy_small_kernel."""
    N = 700
    c = workloads.random_case(N, 15.0, 77, prec, False)
    s = lm.Solver(prec, N)
    s.set_option(lm.LM_OPT_SMALL_KERNEL, small_kernel)
    X, F = dev(torch, c["pos"]).reshape(-1), dev(torch, c["forces"]).reshape(-1).clone()
    U = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.set_positions(X)
    pos, f = np.asarray(c["pos"], np.float64), np.asarray(c["forces"], np.float64)
    for it in range(5):                                   # direct, capture, replay, replay, replay
        s.mdot(F, None, U)
        torch.cuda.synchronize()
        assert rel(U.cpu().numpy(), rpy.mdot(pos, f)[0]) <= TOL[prec], it
        F.mul_(-1.5)                                      # same buffer, new contents
        f = f * -1.5
    X2 = (X * 1.25).contiguous()
    s.set_positions(X2)                                   # same packed buffer inside the handle, new contents
    s.mdot(F, None, U)
    torch.cuda.synchronize()
    assert rel(U.cpu().numpy(), rpy.mdot(X2.cpu().numpy().reshape(N, 3), f)[0]) <= TOL[prec]
    U2 = torch.empty_like(U)                              # another output buffer: not the captured call
    s.mdot(F, None, U2)
    s.mdot_rows(100, 50, F, None, U2)                     # a row range in between
    s.mdot(F, None, U)
    s.mdot(F, None, U)
    torch.cuda.synchronize()
    ref = rpy.mdot(X2.cpu().numpy().reshape(N, 3), f)[0]
    assert rel(U2.cpu().numpy(), ref) <= TOL[prec] and rel(U.cpu().numpy(), ref) <= TOL[prec]
    s.close()


@pytest.mark.parametrize("a,eta", [(1e-6, 1e-3), (1e-9, 1.0), (3.7e4, 2.5e-2)])
def test_fp32_in_any_unit_system(lm, torch, a, eta):
    """SI micrometre spheres in water (a = 1e-6 m, eta = 1e-3 Pa s), nanometres, and a large odd radius: the
    internal power-of-two length unit keeps the fp32 angular blocks, the steric force and the Lanczos root in
    range; same gates as for a = eta = 1."""
    N = 600
    rng = np.random.default_rng(12)
    pos = (rng.random((N, 3)) * 13.0 * a).astype(np.float32)
    F = (rng.standard_normal((N, 3)) * 1e-12).astype(np.float32)
    T = (rng.standard_normal((N, 3)) * 1e-12 * a).astype(np.float32)
    W = rng.standard_normal(6 * N).astype(np.float32)
    s = lm.Solver("f32", N, eta, a, True)
    s.set_positions(dev(torch, pos))
    U = torch.empty(3 * N, dtype=torch.float32, device="cuda")
    Om = torch.empty_like(U)
    s.mdot(dev(torch, F), dev(torch, T), U, Om)
    torch.cuda.synchronize()
    Uo, Oo = rpy.mdot(pos, F, T, a=a, eta=eta, angular=True)
    assert rel(U.cpu().numpy(), Uo) <= 2e-5 and rel(Om.cpu().numpy(), Oo) <= 2e-5
    # The Lanczos root is checked on the translational solver: with include_angular the 6N x 6N matrix mixes
    # blocks ~ 1/(eta a) and ~ 1/(eta a^3), so in such units its symmetric root spans ~ a^-1 orders of magnitude
    # inside one vector -- a property of the method in those units (include/lm.h), not of the kernels.
    st = lm.Solver("f32", N, eta, a, False)
    st.set_positions(dev(torch, pos))
    it = st.sqrt_mdot_w(dev(torch, W[: 3 * N]), 1e-3, U, None)
    torch.cuda.synchronize()
    y = U.cpu().numpy()
    exact = rpy.dense_sqrt_mdot_w(pos, W[: 3 * N], a=a, eta=eta)
    assert np.all(np.isfinite(y)) and 2 <= it < 100
    assert rel(y, exact) <= 1e-2
    st.close()
    from oracle import bd
    Fs = torch.empty(3 * N, dtype=torch.float32, device="cuda")
    U0, b = 4 * 4.11e-21, 0.1 * a
    s.steric_forces(U0, b, None, Fs)
    torch.cuda.synchronize()
    assert rel(Fs.cpu().numpy(), bd.steric_forces(pos, U0, b, 2 * a)) <= 2e-5
    s.close()


def test_seeded_sweep_of_sizes_and_shapes(lm, torch):
    """40 seeded random (N, precision, angular, nrhs, density) combinations: ragged tails, every launch shape and
    split count the chooser produces in this range, far-only and overlap-heavy geometries."""
    rng = np.random.default_rng(2024)
    for case_id in range(40):
        N = int(rng.choice([rng.integers(1, 70), rng.integers(70, 1200), rng.integers(1200, 9000)]))
        prec = "f32" if rng.random() < 0.5 else "f64"
        angular = bool(rng.random() < 0.5)
        nrhs = int(rng.choice([1, 2, 3, 4] if not angular else [1, 2, 3]))
        side = float(N ** (1 / 3) * rng.choice([0.8, 2.0, 6.0]))     # heavy overlap ... dilute
        dt = workloads.np_dtype(prec)
        pos = (rng.random((N, 3)) * side).astype(dt)
        F = rng.standard_normal((nrhs, N, 3)).astype(dt)
        T = rng.standard_normal((nrhs, N, 3)).astype(dt) if angular else None
        s = lm.Solver(prec, N, 1.0, 1.0, angular)
        s.set_positions(dev(torch, pos))
        U = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda")
        W = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
        s.mdot_batch(nrhs, dev(torch, F).reshape(-1), None if T is None else dev(torch, T).reshape(-1), U, W)
        torch.cuda.synchronize()
        U = U.cpu().numpy().reshape(nrhs, N, 3)
        W = W.cpu().numpy().reshape(nrhs, N, 3) if angular else None
        for q in range(nrhs):
            Uo, Wo = rpy.mdot(pos, F[q], None if T is None else T[q], angular=angular)
            tag = (case_id, N, prec, angular, nrhs, q, side)
            assert close(U[q], Uo, TOL[prec]), tag
            if angular:
                assert close(W[q], Wo, TOL[prec]), tag
        s.close()


def test_handles_release_their_device_memory(lm, torch):
    """lm_destroy frees everything a handle allocated (packed arrays, Lanczos basis, graphs, staging, BD buffers)."""
    N = 4000
    c = workloads.random_case(N, 40.0, 5, "f32", True, with_noise=True)
    def cycle():
        s = lm.Solver("f32", N, 1.0, 1.0, True)
        X = dev(torch, c["pos"]).reshape(-1).clone()
        s.set_positions(X)
        U = torch.empty(3 * N, dtype=torch.float32, device="cuda"); W = torch.empty_like(U)
        for _ in range(3):
            s.mdot(dev(torch, c["forces"]), dev(torch, c["torques"]), U, W)
        s.sqrt_mdot_w(dev(torch, c["noise"]), 1e-2, U, W)
        s.bd_step(X, dev(torch, c["forces"]).reshape(-1), None, dev(torch, c["noise"]), 1e-3, 1.0, 4.0, 0.1, 1e-2)
        s.thermal_drift_rfd(dev(torch, c["noise"][: 3 * N]), 1e-2, U, W)
        s.close()
        del X, U, W
    cycle()
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        cycle()
    torch.cuda.synchronize(); torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 8 * 2 ** 20, (free0, free1)        # < 8 MiB drift over 20 handles (one handle holds ~60 MiB)
