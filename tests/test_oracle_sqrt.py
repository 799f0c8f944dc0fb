"""Pins for the oracle's square-root functions (oracle/rpy.py: O3 dense, O4 Lanczos) -- CPU only.

P10(i)   Lanczos vs the exact dense principal root (gates S4), for both stopping rules of reading S3
P10(v)   the stopping quantity (step_error_estimate): closed form on geometric step sequences (the remaining
         path length of an iterate that moves along a line), dips, the cap, and "never before the step rule"
P10(ii)  square-root-twice invariant  sqrt(M) sqrt(M) z = M z, no dense matrix needed
P10(iv)  eq. (12): M^{-1/2} (M^{1/2} W) ~ N(0,1), Kolmogorov-Smirnov; <y y^T> = M
plus closed forms for the small tridiagonal problem.
"""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import rpy


def test_tridiag_sqrt_e1_closed_forms():
    assert rpy.tridiag_sqrt_e1([2.25], []) == pytest.approx([1.5])
    # 2x2 SPD: sqrt(T) = (T + sqrt(det) I) / sqrt(tr + 2 sqrt(det))   (Cayley-Hamilton)
    al, be = [3.0, 2.0], [1.2]
    det = al[0] * al[1] - be[0] ** 2
    den = math.sqrt(al[0] + al[1] + 2 * math.sqrt(det))
    np.testing.assert_allclose(rpy.tridiag_sqrt_e1(al, be), [(al[0] + math.sqrt(det)) / den, be[0] / den], rtol=1e-14)
    # |T^{1/2} e_1|^2 = e_1^T T e_1 = alpha_1 for any SPD tridiagonal
    rng = np.random.default_rng(0)
    al = 2.0 + rng.random(9)
    be = 0.5 * rng.random(8)
    c = rpy.tridiag_sqrt_e1(al, be)
    assert c @ c == pytest.approx(al[0], rel=1e-13)


@pytest.mark.parametrize("angular", [False, True])
def test_dense_root_is_the_symmetric_psd_root(angular):
    rng = np.random.default_rng(1)
    N = 10
    pos = rng.random((N, 3)) * 4.0
    M = rpy.dense(pos, angular=angular)
    dof = M.shape[0]
    S = np.stack([rpy.dense_sqrt_mdot_w(pos, np.eye(dof)[k], angular=angular) for k in range(dof)], 1)
    np.testing.assert_allclose(S, S.T, atol=1e-14)
    np.testing.assert_allclose(S @ S, M, atol=1e-14)
    assert np.linalg.eigvalsh(0.5 * (S + S.T)).min() > 0
    # it is NOT the Cholesky factor (S4 / O3: Lanczos converges to the symmetric root)
    assert np.abs(S - np.linalg.cholesky(M)).max() > 1e-3


def test_lanczos_is_exact_after_dof_steps():
    rng = np.random.default_rng(2)
    N = 3
    pos = rng.random((N, 3)) * 3.0
    z = rng.standard_normal(3 * N)
    y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol=1e-14, max_iter=3 * N)
    np.testing.assert_allclose(y, rpy.dense_sqrt_mdot_w(pos, z), rtol=1e-9, atol=1e-12)
    assert k <= 3 * N


@pytest.mark.parametrize("angular,side", [(False, 12.0), (True, 12.0), (False, 5.0)])
def test_p10i_lanczos_vs_dense_root(angular, side):
    rng = np.random.default_rng(3)
    N = 300
    pos = rng.random((N, 3)) * side
    z = rng.standard_normal((6 if angular else 3) * N)
    exact = rpy.dense_sqrt_mdot_w(pos, z, angular=angular)
    M = rpy.dense(pos, angular=angular)
    err = lambda y: np.linalg.norm(y - exact) / np.linalg.norm(exact)
    # rule "step" (ref. [35]): it bounds the CHANGE between iterates, which under-states the true error
    # (measured x2.5-x8 at tol 1e-3, up to x60 at 1e-7 on these dense, overlapping clouds) -- S4's loose gates
    errs, ksteps = {}, {}
    for tol, slack in ((1e-3, 10.0), (1e-5, 50.0), (1e-6, 100.0)):
        y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol, angular=angular, apply=lambda v: M @ v, rule="step")
        errs[tol], ksteps[tol] = err(y), k
        assert conv and 2 <= k < 100
        assert errs[tol] <= slack * tol, (tol, k, errs[tol])
    assert errs[1e-5] <= 1e-3            # asking for tol/100 delivers a true error below tol
    assert errs[1e-6] < errs[1e-5] < errs[1e-3]
    # rule "estimate" (the default, reading S3): tol is the relative ERROR, met within a factor 2, never stopping
    # before the step rule would, and not wastefully late (the error is not below tol/50)
    for tol in (1e-2, 1e-3, 1e-5):
        y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol, angular=angular, apply=lambda v: M @ v, max_iter=150)
        assert conv and 3 <= k < 150
        assert tol / 50 <= err(y) <= 2.0 * tol, (tol, k, err(y))
        if tol in ksteps:
            assert k >= ksteps[tol]
    # the matrix-free operator (C double loop) gives the same iterate as the dense matvec
    y2, k2, _ = rpy.lanczos_sqrt_mdot_w(pos, z, 1e-3, angular=angular)
    ym, km, _ = rpy.lanczos_sqrt_mdot_w(pos, z, 1e-3, angular=angular, apply=lambda v: M @ v)
    # Lanczos without re-orthogonalisation amplifies the 1e-16 summation-order difference between
    # the two operators (up to ~1e-4 by k ~ 40 on the ill-conditioned side-5 cloud, where the stop step then
    # moves by two); both stay within tol
    assert abs(k2 - km) <= max(1, km // 15)
    assert np.linalg.norm(y2 - ym) <= 0.5 * 1e-3 * np.linalg.norm(ym)


def test_p10v_step_error_estimate_closed_forms():
    """An iterate that moves along a straight line with steps s_i = C rho^i still has s_{k+1} + s_{k+2} + ... =
    s_k rho / (1 - rho) to go.  The estimate is that tail computed from max(s_k, s_{k-1}) = s_k / rho, i.e.
    s_k / (1 - rho) (the current step included: conservative by one step) for rho >= 1/2, and s_{k-1} below."""
    for rho in (0.5, 0.7, 0.9, 0.97):
        for k in (3, 4, 9, 22, 40):
            s = [0.3 * rho ** i for i in range(2, k + 1)]
            assert rpy.step_error_estimate(s) == pytest.approx(s[-1] / (1.0 - rho), rel=1e-12), (rho, k)
    for rho in (0.05, 0.3):                                   # fast convergence: no amplification, never below a step
        s = [0.3 * rho ** i for i in range(2, 12)]
        assert rpy.step_error_estimate(s) == pytest.approx(s[-2], rel=1e-12)
    # stagnation or growth: rho is capped at 0.98 -> the step times 49
    assert rpy.step_error_estimate([1e-3] * 30) == pytest.approx(49e-3, rel=1e-9)
    assert rpy.step_error_estimate([1e-3 * 1.1 ** i for i in range(30)]) == pytest.approx(49 * 1e-3 * 1.1 ** 29, rel=1e-9)
    # one dip (a new Ritz value appears and the next step is tiny) does not pull the estimate under its neighbour
    s = [0.3 * 0.9 ** i for i in range(2, 30)]
    ref = rpy.step_error_estimate(s[:-1])
    dipped = s[:-1] + [s[-1] * 1e-3]
    assert rpy.step_error_estimate(dipped) >= 0.8 * ref * 0.9
    # window: only the last 2 x 10 steps matter
    assert rpy.step_error_estimate([5.0] * 7 + s[-20:]) == pytest.approx(rpy.step_error_estimate(s[-20:]), rel=1e-12)
    # the trailing window is min(10, (k - 1) // 2) steps: k = 3 uses rho = s_3 / s_2
    assert rpy.step_error_estimate([0.2, 0.15]) == pytest.approx(0.2 * 3.0, rel=1e-12)
    with pytest.raises(ValueError):
        rpy.step_error_estimate([0.1])


@pytest.mark.parametrize("name", ["phi1", "phi10", "phi30", "clusters", "angular", "tiny"])
def test_p10v_estimate_rule_delivers_the_requested_error(name):
    """Default rule on dilute ... dense ... clustered ... angular clouds (condition numbers 1e2 ... 1e4): the true
    relative error against the exact dense root is within [tol/50, 2 tol] -- the rule of ref. [35] ("step") is x1.3 ...
    x12 over tol on the same inputs -- and the history it reports is what it stopped on."""
    rng = np.random.default_rng(7)
    side = lambda N, phi: (N * 4.0 * math.pi / (3.0 * phi)) ** (1.0 / 3.0)
    angular = name == "angular"
    N = {"tiny": 12, "angular": 250}.get(name, 500)
    if name == "clusters":
        pos = rng.normal(0.0, 3.0, (N, 3)) + (rng.random((5, 3)) * 50.0).repeat(N // 5, 0)
    elif name == "tiny":
        pos = rng.random((N, 3)) * 3.0
    else:
        pos = rng.random((N, 3)) * side(N, {"phi1": 0.01, "phi10": 0.10, "phi30": 0.30, "angular": 0.10}[name])
    z = rng.standard_normal((6 if angular else 3) * N)
    M = rpy.dense(pos, angular=angular)
    lam, Q = np.linalg.eigh(M)
    exact = Q @ (np.sqrt(lam) * (Q.T @ z))
    for tol in (1e-2, 1e-3, 1e-4):
        hist = {}
        y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol, angular=angular, apply=lambda v: M @ v, history=hist)
        e = np.linalg.norm(y - exact) / np.linalg.norm(exact)
        assert conv and tol / 50 <= e <= 2.0 * tol, (name, tol, k, e)
        assert len(hist["steps"]) == k - 1 and len(hist["estimates"]) == k - 2
        assert hist["estimates"][-1] <= tol and all(v > tol for v in hist["estimates"][:-1])
        assert hist["estimates"][-1] == rpy.step_error_estimate(hist["steps"])
        ys, ks, _ = rpy.lanczos_sqrt_mdot_w(pos, z, tol, angular=angular, apply=lambda v: M @ v, rule="step")
        assert ks <= k


def test_p10ii_square_root_twice():
    rng = np.random.default_rng(4)
    N = 800
    pos = rng.random((N, 3)) * 20.0
    z = rng.standard_normal(3 * N)
    tol = 1e-5                             # two roots, each within ~tol of exact (default rule): a few tol together
    y1, _, c1 = rpy.lanczos_sqrt_mdot_w(pos, z, tol)
    y2, _, c2 = rpy.lanczos_sqrt_mdot_w(pos, y1, tol)
    Mz = rpy.apply_vec(pos, z)
    assert c1 and c2
    assert np.linalg.norm(y2 - Mz) / np.linalg.norm(Mz) < 4 * tol


def test_p10iv_fluctuation_dissipation_ks_and_covariance():
    """eq. (12): whiten Lanczos samples with the exact inverse root from the SVD of the dense M."""
    rng = np.random.default_rng(5)
    N = 6
    pos = rng.random((N, 3)) * 3.5
    M = rpy.dense(pos, angular=True)
    dof = 6 * N
    Uu, sv, Vt = np.linalg.svd(M)
    Minvhalf = Uu @ np.diag(sv ** -0.5) @ Vt
    nsamp = 1500
    Y = np.empty((nsamp, dof))
    for s in range(nsamp):
        Y[s], _, conv = rpy.lanczos_sqrt_mdot_w(pos, rng.standard_normal(dof), 1e-8, angular=True,
                                                apply=lambda v: M @ v)
        assert conv
    white = Y @ Minvhalf.T
    assert stats.kstest(white.reshape(-1), "norm").pvalue > 0.01
    C = Y.T @ Y / nsamp
    assert np.abs(C - M).max() < 6.0 * np.abs(M).max() / math.sqrt(nsamp)


def test_zero_noise_and_max_iter():
    pos = np.random.default_rng(6).random((5, 3)) * 3
    y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, np.zeros(15), 1e-3)
    assert k == 0 and conv and not y.any()
    y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, np.ones(15), 1e-15, max_iter=3)
    assert k == 3 and not conv
