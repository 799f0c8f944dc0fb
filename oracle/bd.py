"""Oracle for the free-space Brownian-dynamics step built on the mobility hot path.

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  fp64, numpy, plain loops over particles; imports only
``oracle.rpy`` (never the CUDA package).

Functions and the passage each follows
--------------------------------------
steric_potential   eq. (13):  U(r) = U0 (1 + (d - r)/b), r < d;  U0 exp((d - r)/b), r >= d
steric_forces      F_i = - grad_i sum_{j != i} U(|x_i - x_j|)  (pairwise repulsion; particle-particle d = 2a,
                   PAPER.md:218).  Coincident particles (r = 0) have no direction: they add nothing (reading S16).
ab_displacement    the deterministic part of eq. (14):  dt (3/2 v^n - 1/2 v^{n-1}); the first
                   step has no history and is forward Euler, dt v^0 (the paper is silent: reading S17).
noise_prefactor    sqrt(2 k_B T dt), eq. (14) (and eq. (9) PAPER.md:78 with the M^{1/2} of reading S7)
bd_step            X^{n+1} = X^n + dt (3/2 M^n F^n - 1/2 M^{n-1} F^{n-1}) + sqrt(2 k_B T dt) (M^n)^{1/2} W^n;
                   the thermal drift terms of eq. (14) vanish for open boundaries.
                   F^n = steric forces at X^n + external forces; torques are external (PAPER.md:226:
                   "F represents a combined vector of forces and torques").

thermal_drift_rfd  eq. (11), one realisation (no average):
                   (1/delta) [ M(X + delta W/2) W - M(X - delta W/2) W ],  W of length 3N acting as forces
                   (the mobility depends on positions only); rows = linear (and angular) velocities.
                   For open boundaries its mean over W is the divergence of M, which is zero.

Pins: tests/test_oracle_bd.py (B1-B11; B11 pins the ``rows=`` branch of steric_forces).  No function here is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np

from . import rpy


def steric_potential(r, U0: float, b: float, d: float):
    """eq. (13): soft repulsive pair potential."""
    r = np.asarray(r, dtype=np.float64)
    return np.where(r < d, U0 * (1.0 + (d - r) / b), U0 * np.exp((d - r) / b))


def steric_forces(pos, U0: float, b: float, d: float, rows=None) -> np.ndarray:
    """Forces from eq. (13), all ordered pairs j != i, row by row.  (N,3), or (len(rows),3) for the
    listed target rows only (rows are independent, so a sample is exact for its rows)."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    N = x.shape[0]
    targets = range(N) if rows is None else [int(i) for i in rows]
    if any(i < 0 or i >= N for i in targets):      # as rpy.mdot_rows: no silent wrap-around of a negative index
        raise ValueError("row index out of range")
    F = np.zeros((len(targets), 3))
    for out, i in enumerate(targets):
        rv = x[i] - x                              # r_vec = x_i - x_j, points from j to i
        r = np.sqrt(np.sum(rv * rv, axis=1))
        ok = r > 0.0                               # skips j = i and exactly coincident particles
        rr = r[ok]
        # -dU/dr: U0/b inside the core, (U0/b) exp((d - r)/b) outside
        mag = np.where(rr < d, U0 / b, (U0 / b) * np.exp((d - rr) / b))
        F[out] = np.sum((mag / rr)[:, None] * rv[ok], axis=0)
    return F


def ab_displacement(v_n, v_nm1, dt: float):
    """dt (3/2 v^n - 1/2 v^{n-1}); forward Euler dt v^n when there is no history (v_nm1 is None)."""
    v_n = np.asarray(v_n, dtype=np.float64)
    if v_nm1 is None:
        return dt * v_n
    return dt * (1.5 * v_n - 0.5 * np.asarray(v_nm1, dtype=np.float64))


def noise_prefactor(kT: float, dt: float) -> float:
    return math.sqrt(2.0 * kT * dt)


def bd_step(pos, v_prev, dt: float, kT: float, a: float = 1.0, eta: float = 1.0, U0: float = 0.0, b: float = 0.1,
            ext_forces=None, ext_torques=None, noise=None, angular: bool = False, sqrt_mode: str = "dense",
            tol: float = 1e-3, max_iter: int = 100):
    """One step of eq. (14).  Returns (new positions (N,3), v_n (N,3) to pass as ``v_prev`` next time, info).

    ``sqrt_mode``: "dense" = exact symmetric root of the dense M (small N); "lanczos" = the Lanczos
    oracle with the stopping rule of rpy.lanczos_sqrt_mdot_w.  ``noise`` is W^n (dof entries) or None.
    """
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    N = x.shape[0]
    d = 2.0 * a                                    # particle-particle contact distance
    F = np.zeros((N, 3))
    if U0 != 0.0:
        F += steric_forces(x, U0, b, d)
    if ext_forces is not None:
        F += np.asarray(ext_forces, dtype=np.float64).reshape(N, 3)
    T = None if ext_torques is None else np.asarray(ext_torques, dtype=np.float64).reshape(N, 3)
    U, _ = rpy.mdot(x, F, T, a=a, eta=eta, angular=angular)
    info = {"iterations": 0}
    new = x + ab_displacement(U, v_prev, dt)
    if noise is not None and kT > 0.0:
        if sqrt_mode == "dense":
            y = rpy.dense_sqrt_mdot_w(x, noise, a=a, eta=eta, angular=angular)
        else:
            y, k, _ = rpy.lanczos_sqrt_mdot_w(x, noise, tol, a=a, eta=eta, angular=angular, max_iter=max_iter)
            info["iterations"] = k
        new = new + noise_prefactor(kT, dt) * np.asarray(y).reshape(-1)[: 3 * N].reshape(N, 3)
    return new, U, info


def thermal_drift_rfd(pos, W, delta: float, a: float = 1.0, eta: float = 1.0, angular: bool = False):
    """One random-finite-difference sample of the thermal drift, eq. (11).  Returns (lin (N,3), ang (N,3) or None)."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    w = np.asarray(W, dtype=np.float64).reshape(-1, 3)
    Up, Op = rpy.mdot(x + 0.5 * delta * w, w, None, a=a, eta=eta, angular=angular)
    Um, Om = rpy.mdot(x - 0.5 * delta * w, w, None, a=a, eta=eta, angular=angular)
    lin = (Up - Um) / delta
    ang = (Op - Om) / delta if angular else None
    return lin, ang
