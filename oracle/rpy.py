"""Oracle front end: ctypes binding to ``rpy_oracle.c`` plus the dense / Lanczos square-root oracles.

TEST INFRASTRUCTURE, NOT PRODUCT CODE (see ``rpy_oracle.c`` header).  Everything here is fp64.

Functions and the passage each follows
--------------------------------------
pair_scalars      SURVEY.md sec. 8(c) O1 (PAPER.md:173 names the RPY kernels; eq. (8))
mdot, mdot_rows   O2: U = M.[F;T], eq. (7), plain double loop in C
dense             eq. (7) assembled densely (PAPER.md:196-198 uses the full matrix in its tests)
dense_sqrt_mdot_w O3: principal symmetric square root by eigendecomposition
lanczos_sqrt_mdot_w  O4: Lanczos iteration of ref. [35], step by step
step_error_estimate  the stopping quantity of O4 (reading S3: the paper states no rule)
tridiag_sqrt_e1   the small T_k^{1/2} e_1 problem inside O4

Pins: tests/test_oracle_pins.py (mdot family), tests/test_oracle_sqrt.py (square roots).
No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rpy_oracle.c")
_LIB = os.path.join(_HERE, "librpy_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile rpy_oracle.c with gcc -O2 -fopenmp (no fast-math).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        lib.rpy_pair_scalars.argtypes = [ctypes.c_double] * 3 + [dp]
        lib.rpy_pair_scalars.restype = None
        lib.rpy_mdot.argtypes = [ctypes.c_int64, ctypes.c_double, ctypes.c_double, dp, dp, dp, dp, dp]
        lib.rpy_mdot.restype = ctypes.c_int
        lib.rpy_mdot_rows.argtypes = [ctypes.c_int64, ctypes.c_double, ctypes.c_double, dp, dp, dp,
                                      ctypes.c_int64, ip, dp, dp]
        lib.rpy_mdot_rows.restype = ctypes.c_int
        lib.rpy_dense.argtypes = [ctypes.c_int64, ctypes.c_double, ctypes.c_double, dp, ctypes.c_int, dp]
        lib.rpy_dense.restype = None
        _lib = lib
    return _lib


def _d(arr):
    return None if arr is None else arr.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _as3n(v, N, name):
    if v is None:
        return None
    v = np.ascontiguousarray(np.asarray(v, dtype=np.float64).reshape(-1))
    if v.size != 3 * N:
        raise ValueError(f"{name} must have 3N = {3 * N} entries, got {v.size}")
    return v


def pair_scalars(r: float, a: float = 1.0, eta: float = 1.0) -> np.ndarray:
    """(f_tt, g_tt, f_rr, g_rr, g_c) at centre distance r -- O1."""
    out = np.zeros(5)
    _load().rpy_pair_scalars(float(r), float(a), float(eta), _d(out))
    return out


def mdot(pos, forces=None, torques=None, a: float = 1.0, eta: float = 1.0, angular: bool = False):
    """U = M.[F;T] (O2).  Returns (U, Omega) as (N,3) arrays; Omega is None unless ``angular``.

    ``forces`` / ``torques`` = None means zeros ("one or both of forces and torques").
    Inputs of any float dtype are promoted exactly to fp64 (S11)."""
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1))
    N = pos.size // 3
    F = _as3n(forces, N, "forces")
    T = _as3n(torques, N, "torques")
    if T is not None and not angular:
        raise ValueError("torques given but angular=False")
    U = np.zeros(3 * N)
    W = np.zeros(3 * N) if angular else None
    mdot.last_threads = _load().rpy_mdot(N, a, eta, _d(pos), _d(F), _d(T), _d(U), _d(W))
    return U.reshape(N, 3), (W.reshape(N, 3) if angular else None)


mdot.last_threads = 0


def mdot_rows(pos, rows, forces=None, torques=None, a: float = 1.0, eta: float = 1.0, angular: bool = False):
    """O2 for the target rows ``rows`` only, against all N sources (exact for those rows)."""
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1))
    N = pos.size // 3
    rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    if rows.size and (rows.min() < 0 or rows.max() >= N):
        raise ValueError("row index out of range")
    F = _as3n(forces, N, "forces")
    T = _as3n(torques, N, "torques")
    U = np.zeros(3 * rows.size)
    W = np.zeros(3 * rows.size) if angular else None
    mdot_rows.last_threads = _load().rpy_mdot_rows(
        N, a, eta, _d(pos), _d(F), _d(T), rows.size,
        rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), _d(U), _d(W))
    return U.reshape(-1, 3), (W.reshape(-1, 3) if angular else None)


mdot_rows.last_threads = 0


def dense(pos, a: float = 1.0, eta: float = 1.0, angular: bool = False) -> np.ndarray:
    """Dense grand mobility (eq. (7)), dof x dof, dof = 3N or 6N: [linear | angular] ordering."""
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1))
    N = pos.size // 3
    dof = (6 if angular else 3) * N
    M = np.zeros((dof, dof))
    _load().rpy_dense(N, a, eta, _d(pos), int(angular), _d(M))
    return M


def apply_vec(pos, v, a: float = 1.0, eta: float = 1.0, angular: bool = False) -> np.ndarray:
    """M.v for a dof-vector v = [3N linear | 3N angular] (S10), returned in the same layout."""
    v = np.asarray(v, dtype=np.float64).reshape(-1)
    N = np.asarray(pos).size // 3
    if angular:
        U, W = mdot(pos, v[:3 * N], v[3 * N:], a, eta, True)
        return np.concatenate([U.reshape(-1), W.reshape(-1)])
    U, _ = mdot(pos, v, None, a, eta, False)
    return U.reshape(-1)


def dense_sqrt_mdot_w(pos, noise, a: float = 1.0, eta: float = 1.0, angular: bool = False) -> np.ndarray:
    """O3: the exact principal square root applied to ``noise``: M = Q L Q^T, y = Q L^{1/2} Q^T W."""
    M = dense(pos, a, eta, angular)
    lam, Q = np.linalg.eigh(M)
    lam = np.clip(lam, 0.0, None)
    w = np.asarray(noise, dtype=np.float64).reshape(-1)
    return Q @ (np.sqrt(lam) * (Q.T @ w))


def tridiag_sqrt_e1(alpha, beta) -> np.ndarray:
    """c = T^{1/2} e_1 for T = tridiag(beta; alpha; beta), negative eigenvalues clamped to 0 (O4)."""
    k = len(alpha)
    Tm = np.diag(np.asarray(alpha, dtype=np.float64))
    for i in range(k - 1):
        Tm[i, i + 1] = Tm[i + 1, i] = beta[i]
    lam, S = np.linalg.eigh(Tm)
    lam = np.clip(lam, 0.0, None)
    return S @ (np.sqrt(lam) * S[0, :])


def step_error_estimate(steps, window: int = 10, rho_max: float = 0.98) -> float:
    """Error estimate of the newest Lanczos iterate from the relative steps s_2..s_k (reading S3).

    ``steps`` = [s_2, ..., s_k], s_i = |y_i - y_{i-1}| / |y_{i-1}|, k >= 3.  The paper fixes no stopping rule
    (PAPER.md:147); the rule of ref. [35] takes s_k itself as the error, which under-states it by the factor
    rho/(1 - rho) when the steps shrink slowly (ratio rho per iteration): the iterate still has to travel
    s_{k+1} + s_{k+2} + ... ~ s_k (rho + rho^2 + ...) = s_k rho / (1 - rho).  Here

        m   = max(1, min(window, (k - 1) // 2))                  trailing window, in steps
        rho = min( (sum of the last m steps / sum of the m steps before them)^(1/m), rho_max )
        e_k = max(s_k, s_{k-1}) * max(1, rho / (1 - rho))

    max(s_k, s_{k-1}): one small step is no evidence (the steps dip whenever a new Ritz value appears);
    max(1, .): never less than the step rule of ref. [35]; rho_max bounds the amplification (x49)."""
    s = [float(v) for v in steps]
    n = len(s)                                   # n = k - 1 steps
    if n < 2:
        raise ValueError("needs at least the two steps s_2, s_3")
    m = max(1, min(int(window), n // 2))
    recent = sum(s[n - m:])
    before = sum(s[n - 2 * m:n - m])
    if before > 0.0:
        rho = min((recent / before) ** (1.0 / m), rho_max)
    else:
        rho = 0.0                                # the earlier steps were exactly zero: nothing left to extrapolate
    return max(s[-1], s[-2]) * max(1.0, rho / (1.0 - rho))


def lanczos_sqrt_mdot_w(pos, noise, tol: float, a: float = 1.0, eta: float = 1.0, angular: bool = False,
                        max_iter: int = 100, apply=None, rule: str = "estimate", history: dict | None = None):
    """O4: Lanczos approximation of M^{1/2} z (ref. [35]), in the order written
    in SURVEY.md sec. 8(c) O4.  No re-orthogonalisation.  Returns (y, iterations, converged).

        v_1 = z/|z|, beta_0 = 0
        k = 1,2,..:  w = M v_k - beta_{k-1} v_{k-1};  alpha_k = w.v_k;  w -= alpha_k v_k;
                     beta_k = |w|;  v_{k+1} = w / beta_k
                     c_k = T_k^{1/2} e_1;  y_k = |z| V_k c_k;  s_k = |y_k - y_{k-1}| / |y_{k-1}|
                     stop (reading S3; the paper states no rule):
                       rule "estimate" (default): k >= 3 and step_error_estimate(s_2..s_k) <= tol
                       rule "step" (ref. [35] as SURVEY O4 writes it): k >= 2 and s_k <= tol
                     or beta_k ~ 0 (invariant subspace: y_k is exact).
    ``apply`` overrides the operator (default: the O(N^2) oracle apply).  ``history``, if given, receives
    "steps" = [s_2..s_k], "estimates" = [e_3..e_k], "alphas" = [alpha_1..alpha_k] and "betas" = [beta_1..] (the lists the
    loop below fills anyway: test diagnostics, no arithmetic of their own)."""
    if rule not in ("estimate", "step"):
        raise ValueError("rule must be 'estimate' or 'step'")
    z = np.asarray(noise, dtype=np.float64).reshape(-1)
    if apply is None:
        def apply(v):
            return apply_vec(pos, v, a, eta, angular)
    steps, estimates = [], []
    if history is not None:
        history["steps"], history["estimates"] = steps, estimates
    znorm = np.linalg.norm(z)
    if znorm == 0.0:
        return np.zeros_like(z), 0, True
    V = [z / znorm]
    alphas, betas = [], []
    if history is not None:
        history["alphas"], history["betas"] = alphas, betas
    y_prev = None
    for k in range(1, max_iter + 1):
        w = apply(V[k - 1])
        if k > 1:
            w = w - betas[k - 2] * V[k - 2]
        alpha = float(w @ V[k - 1])
        w = w - alpha * V[k - 1]
        beta = float(np.linalg.norm(w))
        alphas.append(alpha)
        c = tridiag_sqrt_e1(alphas, betas)
        y = znorm * (np.stack(V, axis=1) @ c)
        if y_prev is not None:
            steps.append(float(np.linalg.norm(y - y_prev) / np.linalg.norm(y_prev)))
            if rule == "step":
                if steps[-1] <= tol:
                    return y, k, True
            elif k >= 3:
                estimates.append(step_error_estimate(steps))
                if estimates[-1] <= tol:
                    return y, k, True
        if beta <= 1e-14 * abs(alpha):          # invariant subspace: y_k is exact
            return y, k, True
        betas.append(beta)
        V.append(w / beta)
        y_prev = y
    return y, max_iter, False
