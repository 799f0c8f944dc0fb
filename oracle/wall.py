"""Oracle front end for the single-wall (Swan-Brady) mobility: ctypes binding to ``wall_oracle.c``.

TEST INFRASTRUCTURE, NOT PRODUCT CODE (see the ``wall_oracle.c`` header).  Everything here is fp64.

Functions and the passage each follows
--------------------------------------
pair_correction   the four 3x3 blocks by which the wall corrects the free-space pair mobility (PAPER.md:173 names the
                  Swan-Brady kernel, ref. [37]; reading S18 and appendix A: Faxen operators on the image part
                  of the half-space Green's function = eq. (8) PAPER.md:73 for spheres that do not cut the wall)
damping           raised heights and the damping factors b_i ("damping matrix approach"; reading S19)
mdot, mdot_rows   U = B M(x~) B [F;T]  (eq. (7) PAPER.md:66-69 for the geometry ("open","open","single_wall"))
dense             the same matrix assembled densely
apply_vec         M~.v for a dof-vector [3N linear | 3N angular] (reading S10)
dense_sqrt_mdot_w the exact principal square root applied to W
lanczos_sqrt_mdot_w  rpy.lanczos_sqrt_mdot_w with the wall operator
thermal_drift_rfd eq. (11), one realisation: (1/delta)[M(X + delta W/2) - M(X - delta W/2)] W
divergence_fd     (d/dX).M by central differences of the dense matrix: what the mean of the RFD must equal
wall_steric_forces eq. (13) PAPER.md:214-219 between a particle and the wall: r = height of the centre, d = a
bd_step           eq. (14) PAPER.md:224-228 above a wall: X^{n+1} = X^n + dt (3/2 v^n - 1/2 v^{n-1}) + sqrt(2 kT dt) (M^n)^{1/2} W^n
                  with v^n = M^n F^n + kT (d/dX).M^n, the drift taken as ONE random-finite-difference sample of eq. (11)
                  ("we also include the thermal drift term in the deterministic part of the time stepping
                  scheme"); F^n = particle-particle and particle-wall steric forces (eq. 13) + external forces

Pins: tests/test_oracle_wall.py.  No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from . import rpy

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = [os.path.join(_HERE, "wall_oracle.c"), os.path.join(_HERE, "rpy_oracle.c")]
_LIB = os.path.join(_HERE, "libwall_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp (no fast-math) of wall_oracle.c + rpy_oracle.c.  Returns the .so path."""
    if force or not os.path.exists(_LIB) or any(os.path.getmtime(_LIB) < os.path.getmtime(s) for s in _SRCS):
        subprocess.run(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB] + _SRCS + ["-lm"], check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        lib.wall_pair_correction.argtypes = [dp, dp, ctypes.c_double, ctypes.c_double, dp, dp, dp, dp]
        lib.wall_pair_correction.restype = None
        lib.wall_mdot_rows.argtypes = [ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, dp, dp, ctypes.c_int64, ip, dp, dp]
        lib.wall_mdot_rows.restype = ctypes.c_int
        lib.wall_dense.argtypes = [ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, ctypes.c_int, dp]
        lib.wall_dense.restype = None
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


def pair_correction(xi, xj, a: float = 1.0, eta: float = 1.0):
    """Wall correction blocks (uF, uT, wF, wT), each 3x3, for particle i <- particle j.  ``xi``, ``xj``: positions with
    z = height above the wall, both >= a (no damping, no free-space part here)."""
    xi = np.ascontiguousarray(np.asarray(xi, dtype=np.float64).reshape(3))
    xj = np.ascontiguousarray(np.asarray(xj, dtype=np.float64).reshape(3))
    out = [np.zeros(9) for _ in range(4)]
    _load().wall_pair_correction(_d(xi), _d(xj), float(a), float(eta), *[_d(o) for o in out])
    return tuple(o.reshape(3, 3) for o in out)


def damping(pos, a: float = 1.0, wall_z: float = 0.0):
    """Reading S19.  Returns (x~ with heights above the wall raised to >= a, b) with b_i = min(1, max(h_i, 0)/a)."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3).copy()
    h = x[:, 2] - wall_z
    b = np.clip(h / a, 0.0, 1.0)
    x[:, 2] = np.maximum(h, a)
    return x, b


def mdot_rows(pos, rows, forces=None, torques=None, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False):
    """U = M~.[F;T] for the target rows ``rows`` (None: all) against all N sources.  Returns (U, Omega or None)."""
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1))
    N = pos.size // 3
    F = _as3n(forces, N, "forces")
    T = _as3n(torques, N, "torques")
    if T is not None and not angular:
        raise ValueError("torques given but angular=False")
    if rows is None:
        n, rp = N, None
    else:
        rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
        if rows.size and (rows.min() < 0 or rows.max() >= N):
            raise ValueError("row index out of range")
        n, rp = rows.size, rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
    U = np.zeros(3 * n)
    W = np.zeros(3 * n) if angular else None
    mdot_rows.last_threads = _load().wall_mdot_rows(N, float(a), float(eta), float(wall_z), _d(pos), _d(F), _d(T), n, rp, _d(U), _d(W))
    return U.reshape(-1, 3), (W.reshape(-1, 3) if angular else None)


mdot_rows.last_threads = 0


def mdot(pos, forces=None, torques=None, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False):
    return mdot_rows(pos, None, forces, torques, a, eta, wall_z, angular)


def dense(pos, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False) -> np.ndarray:
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1))
    N = pos.size // 3
    dof = (6 if angular else 3) * N
    M = np.zeros((dof, dof))
    _load().wall_dense(N, float(a), float(eta), float(wall_z), _d(pos), int(angular), _d(M))
    return M


def apply_vec(pos, v, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False) -> np.ndarray:
    v = np.asarray(v, dtype=np.float64).reshape(-1)
    N = np.asarray(pos).size // 3
    if angular:
        U, W = mdot(pos, v[:3 * N], v[3 * N:], a, eta, wall_z, True)
        return np.concatenate([U.reshape(-1), W.reshape(-1)])
    U, _ = mdot(pos, v, None, a, eta, wall_z, False)
    return U.reshape(-1)


def dense_sqrt_mdot_w(pos, noise, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False) -> np.ndarray:
    lam, Q = np.linalg.eigh(dense(pos, a, eta, wall_z, angular))
    lam = np.clip(lam, 0.0, None)
    return Q @ (np.sqrt(lam) * (Q.T @ np.asarray(noise, dtype=np.float64).reshape(-1)))


def lanczos_sqrt_mdot_w(pos, noise, tol: float, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False,
                        max_iter: int = 100, rule: str = "estimate", history=None):
    return rpy.lanczos_sqrt_mdot_w(pos, noise, tol, max_iter=max_iter, rule=rule, history=history,
                                   apply=lambda v: apply_vec(pos, v, a, eta, wall_z, angular))


def thermal_drift_rfd(pos, W, delta: float, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False):
    """One random-finite-difference sample of eq. (11); W (3N) acts as forces.  Returns (lin (N,3), ang (N,3) or None)."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    w = np.asarray(W, dtype=np.float64).reshape(-1, 3)
    Up, Op = mdot(x + 0.5 * delta * w, w, None, a, eta, wall_z, angular)
    Um, Om = mdot(x - 0.5 * delta * w, w, None, a, eta, wall_z, angular)
    return (Up - Um) / delta, ((Op - Om) / delta if angular else None)


def divergence_fd(pos, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, angular: bool = False, step: float = 1e-5) -> np.ndarray:
    """(d/dX).M~ : component r = sum_c dM~[r, c] / dX_c over the 3N position coordinates c (orientations do not enter
    the mobility of spheres), by central differences of the dense matrix.  Length dof."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1)
    out = np.zeros((6 if angular else 3) * (x.size // 3))
    for c in range(x.size):
        xp, xm = x.copy(), x.copy()
        xp[c] += step
        xm[c] -= step
        out += (dense(xp, a, eta, wall_z, angular)[:, c] - dense(xm, a, eta, wall_z, angular)[:, c]) / (2.0 * step)
    return out


def wall_steric_forces(pos, U0: float, b: float, a: float = 1.0, wall_z: float = 0.0) -> np.ndarray:
    """eq. (13) between each particle and the wall: r = height of the centre above the wall, d = a;
    F_z = -dU/dr = U0/b for r < d, (U0/b) exp((d - r)/b) for r >= d.  (N,3), only z non-zero."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    r = x[:, 2] - wall_z
    F = np.zeros_like(x)
    F[:, 2] = np.where(r < a, U0 / b, (U0 / b) * np.exp((a - r) / b))
    return F


def bd_step(pos, v_prev, dt: float, kT: float, a: float = 1.0, eta: float = 1.0, wall_z: float = 0.0, U0: float = 0.0, b: float = 0.1,
            ext_forces=None, ext_torques=None, noise=None, rfd_noise=None, delta: float = 1e-3, angular: bool = False,
            sqrt_mode: str = "dense", tol: float = 1e-3, max_iter: int = 100):
    """One step of eq. (14) above a wall.  Returns (new positions (N,3), v^n (N,3) to pass as ``v_prev`` next time, info).
    The first step (v_prev None) is forward Euler (reading S17).  ``rfd_noise``: the 3N vector W~ of eq. (11) for
    this step's drift sample, or None for no drift term; ``noise``: W^n (dof entries) or None."""
    from . import bd
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    N = x.shape[0]
    F = np.zeros((N, 3))
    if U0 != 0.0:
        F += bd.steric_forces(x, U0, b, 2.0 * a) + wall_steric_forces(x, U0, b, a, wall_z)
    if ext_forces is not None:
        F += np.asarray(ext_forces, dtype=np.float64).reshape(N, 3)
    T = None if ext_torques is None else np.asarray(ext_torques, dtype=np.float64).reshape(N, 3)
    v, _ = mdot(x, F, T, a, eta, wall_z, angular)
    if rfd_noise is not None and kT > 0.0:
        v = v + kT * thermal_drift_rfd(x, rfd_noise, delta, a, eta, wall_z, angular)[0]
    info = {"iterations": 0}
    new = x + bd.ab_displacement(v, v_prev, dt)
    if noise is not None and kT > 0.0:
        if sqrt_mode == "dense":
            y = dense_sqrt_mdot_w(x, noise, a, eta, wall_z, angular)
        else:
            y, k, _ = lanczos_sqrt_mdot_w(x, noise, tol, a, eta, wall_z, angular, max_iter=max_iter)
            info["iterations"] = k
        new = new + bd.noise_prefactor(kT, dt) * np.asarray(y).reshape(-1)[: 3 * N].reshape(N, 3)
    return new, v, info
