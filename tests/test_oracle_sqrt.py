"""Pins for the oracle's square-root functions (oracle/rpy.py: O3 dense, O4 Lanczos) -- CPU only.

P10(i)   Lanczos vs the exact dense principal root (gates S4)
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
    # S3/S4: the stopping rule bounds the CHANGE between iterates, which under-states the true
    # error (measured x2.5-x8 at tol 1e-3, up to x60 at 1e-7 on these dense, overlapping clouds)
    errs = {}
    for tol, slack in ((1e-3, 10.0), (1e-5, 50.0), (1e-6, 100.0)):
        y, k, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol, angular=angular, apply=lambda v: M @ v)
        errs[tol] = np.linalg.norm(y - exact) / np.linalg.norm(exact)
        assert conv and 2 <= k < 100
        assert errs[tol] <= slack * tol, (tol, k, errs[tol])
    assert errs[1e-5] <= 1e-3            # asking for tol/100 delivers a true error below tol
    assert errs[1e-6] < errs[1e-5] < errs[1e-3]
    # the matrix-free operator (C double loop) gives the same iterate as the dense matvec
    y2, k2, _ = rpy.lanczos_sqrt_mdot_w(pos, z, 1e-3, angular=angular)
    ym, km, _ = rpy.lanczos_sqrt_mdot_w(pos, z, 1e-3, angular=angular, apply=lambda v: M @ v)
    assert abs(k2 - km) <= 1
    # Lanczos without re-orthogonalisation amplifies the 1e-16 summation-order difference between
    # the two operators (up to ~1e-4 on the ill-conditioned side-5 cloud); both stay within tol
    assert np.linalg.norm(y2 - ym) <= 0.5 * 1e-3 * np.linalg.norm(ym)


def test_p10ii_square_root_twice():
    rng = np.random.default_rng(4)
    N = 800
    pos = rng.random((N, 3)) * 20.0
    z = rng.standard_normal(3 * N)
    y1, _, c1 = rpy.lanczos_sqrt_mdot_w(pos, z, 1e-7)
    y2, _, c2 = rpy.lanczos_sqrt_mdot_w(pos, y1, 1e-7)
    Mz = rpy.apply_vec(pos, z)
    assert c1 and c2
    assert np.linalg.norm(y2 - Mz) / np.linalg.norm(Mz) < 1e-5


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
