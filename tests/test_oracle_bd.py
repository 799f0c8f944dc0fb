"""Pins for oracle/bd.py (free-space Brownian-dynamics step, eqs. (13)-(14) PAPER.md:214-226) -- CPU only.

B1  eq. (13): the potential and its slope are continuous at r = d (value U0, slope -U0/b), typed here
    from the printed formula, not from the oracle
B2  steric force = -grad of the total energy sum_{i<j} U(r_ij): central finite differences of an
    energy function written out here from eq. (13)
B3  Newton's third law: total force and total torque of the pair forces vanish
B4  two-particle closed forms inside and outside the core
B5  eq. (14) deterministic part: the 3/2, -1/2 weights integrate v(t) = t exactly and give second-order
    convergence on dx/dt = -x (first order if the weights were wrong)
B6  noise prefactor: one isolated sphere performs free diffusion with D = k_B T / (6 pi eta a)
    (eq. (9) PAPER.md:78 with the self mobility PAPER.md:165): displacement = sqrt(2 D dt) W exactly
B7  two equal spheres under equal forces: one Euler step moves them by dt times the closed-form
    sedimentation velocity (textbook RPY)
B8  Lanczos and dense noise modes agree within the gates of S4
B9  eq. (11): the RFD sample equals the directional derivative sum_k W_k dM/dX_k W built coordinate by
    coordinate from central differences of the DENSE matrix (a different route: pins 1/delta and the
    +-delta/2 arguments), to O(delta^2); and its mean over many W vanishes for open boundaries
     within the statistical error
"""
import math

import numpy as np
import pytest

from oracle import bd


def energy(x, U0, b, d):
    """sum over unordered pairs of eq. (13), typed from PAPER.md:214-216."""
    x = np.asarray(x, dtype=np.float64).reshape(-1, 3)
    E = 0.0
    for i in range(len(x)):
        for j in range(i + 1, len(x)):
            r = math.dist(x[i], x[j])
            E += U0 * (1.0 + (d - r) / b) if r < d else U0 * math.exp((d - r) / b)
    return E


def test_b1_potential_continuous_with_continuous_slope_at_contact():
    U0, b, d = 4.0, 0.1, 2.0
    h = 1e-7
    lo, hi = bd.steric_potential(d - h, U0, b, d), bd.steric_potential(d + h, U0, b, d)
    assert float(lo) == pytest.approx(U0, rel=1e-5) and float(hi) == pytest.approx(U0, rel=1e-5)
    slope_in = (bd.steric_potential(d - h, U0, b, d) - bd.steric_potential(d - 2 * h, U0, b, d)) / h
    slope_out = (bd.steric_potential(d + 2 * h, U0, b, d) - bd.steric_potential(d + h, U0, b, d)) / h
    assert float(slope_in) == pytest.approx(-U0 / b, rel=1e-5)
    assert float(slope_out) == pytest.approx(-U0 / b, rel=1e-5)
    assert float(bd.steric_potential(0.0, U0, b, d)) == pytest.approx(U0 * (1 + d / b))
    assert float(bd.steric_potential(d + 3 * b, U0, b, d)) == pytest.approx(U0 * math.exp(-3.0))


def test_b2_force_is_minus_gradient_of_the_energy():
    rng = np.random.default_rng(5)
    N, U0, b, d = 12, 1.7, 0.3, 2.0
    x = rng.random((N, 3)) * 4.5                     # mixes r < d and r >= d pairs
    F = bd.steric_forces(x, U0, b, d)
    h = 1e-6
    for i in (0, 3, 7, 11):
        for k in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, k] += h
            xm[i, k] -= h
            fd = -(energy(xp, U0, b, d) - energy(xm, U0, b, d)) / (2 * h)
            assert F[i, k] == pytest.approx(fd, rel=2e-7, abs=1e-8)


def test_b3_newtons_third_law():
    rng = np.random.default_rng(6)
    x = rng.random((40, 3)) * 6.0
    F = bd.steric_forces(x, 4.0, 0.1, 2.0)
    scale = np.abs(F).max()
    assert np.abs(F.sum(0)).max() <= 1e-12 * scale * 40
    assert np.abs(np.cross(x, F).sum(0)).max() <= 1e-11 * scale * 40 * 6


def test_b4_two_particle_closed_forms_and_coincident_particles():
    U0, b, d = 4.0, 0.1, 2.0
    for r, mag in ((1.5, U0 / b), (2.5, U0 / b * math.exp(-5.0)), (2.0, U0 / b)):
        x = np.array([[0.0, 0.0, 0.0], [0.0, r, 0.0]])
        F = bd.steric_forces(x, U0, b, d)
        np.testing.assert_allclose(F[0], [0.0, -mag, 0.0], rtol=1e-14, atol=0)   # pushed away from the neighbour
        np.testing.assert_allclose(F[1], [0.0, +mag, 0.0], rtol=1e-14, atol=0)
    x = np.zeros((2, 3))                              # coincident: no direction, no force (S16)
    assert np.all(bd.steric_forces(x, U0, b, d) == 0.0)


def test_b5_adams_bashforth_weights():
    # exact for v(t) = t:  x(t) = t^2/2
    dt, x, vprev = 0.1, 0.0, None
    for n in range(20):
        t = n * dt
        if vprev is None:
            x = 0.5 * dt * dt                         # exact start so that only the AB weights are tested
        else:
            x = x + float(bd.ab_displacement(t, vprev, dt))
        vprev = t
    assert x == pytest.approx(0.5 * (20 * dt) ** 2, rel=1e-13)
    # first step without history is forward Euler
    assert float(bd.ab_displacement(3.0, None, 0.25)) == 0.75

    # second-order convergence on dx/dt = -x, x(0) = 1, to t = 1
    def run(nsteps):
        dt = 1.0 / nsteps
        x, vprev = 1.0, None
        for _ in range(nsteps):
            v = -x
            x, vprev = x + float(bd.ab_displacement(v, vprev, dt)), v
        return abs(x - math.exp(-1.0))
    e1, e2 = run(200), run(400)
    assert 3.0 < e1 / e2 < 5.0                        # ~4: second order (Euler start costs O(dt^2) once)


def test_b6_single_sphere_free_diffusion_step():
    a, eta, kT, dt = 0.7, 1.3, 0.41, 0.02
    W = np.array([0.3, -1.2, 2.0])
    D = kT / (6 * math.pi * eta * a)
    for mode in ("dense", "lanczos"):
        new, U, _ = bd.bd_step(np.zeros((1, 3)), None, dt, kT, a=a, eta=eta, noise=W, sqrt_mode=mode, tol=1e-12)
        np.testing.assert_allclose(new[0], math.sqrt(2 * D * dt) * W, rtol=1e-13)
        assert np.all(U == 0.0)
    assert bd.noise_prefactor(kT, dt) == pytest.approx(math.sqrt(2 * kT * dt))


def test_b7_two_sphere_sedimentation_euler_step():
    a, eta, dt, r, f = 1.0, 1.0, 0.5, 3.0, 2.0
    x = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
    mu0 = 1.0 / (6 * math.pi * eta * a)
    # forces along the line of centres / perpendicular to it (r >= 2a)
    for direction, factor in (([1.0, 0, 0], 1 + 1.5 * a / r - a ** 3 / r ** 3), ([0, 0, 1.0], 1 + 0.75 * a / r + 0.5 * a ** 3 / r ** 3)):
        F = np.tile(np.array(direction) * f, (2, 1))
        new, U, _ = bd.bd_step(x, None, dt, 0.0, a=a, eta=eta, ext_forces=F)
        np.testing.assert_allclose(new - x, dt * mu0 * factor * F, rtol=1e-13, atol=1e-16)
    # second step uses the 3/2, -1/2 weights with the stored velocity
    F = np.tile(np.array([0, 0, 1.0]), (2, 1))
    x1, v0, _ = bd.bd_step(x, None, dt, 0.0, ext_forces=F)
    x2, v1, _ = bd.bd_step(x1, v0, dt, 0.0, ext_forces=F)
    np.testing.assert_allclose(x2 - x1, dt * (1.5 * v1 - 0.5 * v0), rtol=1e-13)


def test_b8_noise_modes_agree_and_steric_pushes_overlaps_apart():
    rng = np.random.default_rng(8)
    N = 60
    x = rng.random((N, 3)) * 9.0
    W = rng.standard_normal(3 * N)
    kw = dict(dt=0.01, kT=1.0, U0=4.0, b=0.1, noise=W)
    xd, _, _ = bd.bd_step(x, None, sqrt_mode="dense", **kw)
    xl, _, info = bd.bd_step(x, None, sqrt_mode="lanczos", tol=1e-8, **kw)
    assert info["iterations"] >= 2
    assert np.linalg.norm(xl - xd) <= 1e-6 * np.linalg.norm(xd - x)
    # deterministic step with the steric force only: the closest overlapping pair separates
    x2 = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [30.0, 0.0, 0.0]])
    new, _, _ = bd.bd_step(x2, None, 1e-3, 0.0, U0=4.0, b=0.1)
    assert np.linalg.norm(new[1] - new[0]) > 1.0


def test_b9_rfd_is_the_directional_derivative_and_averages_to_zero():
    from oracle import rpy
    rng = np.random.default_rng(9)
    N = 5
    x = rng.random((N, 3)) * 4.0                       # overlapping and non-overlapping pairs
    W = rng.standard_normal((N, 3))
    delta = 1e-4
    lin, ang = bd.thermal_drift_rfd(x, W, delta, angular=True)
    # sum_k W_k dM/dX_k, coordinate by coordinate, from the dense 6N x 6N matrix
    h = 1e-6
    dM = np.zeros((6 * N, 6 * N))
    for p in range(N):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[p, c] += h
            xm[p, c] -= h
            dM += W[p, c] * (rpy.dense(xp, angular=True) - rpy.dense(xm, angular=True)) / (2 * h)
    ref = dM @ np.concatenate([W.reshape(-1), np.zeros(3 * N)])
    np.testing.assert_allclose(lin.reshape(-1), ref[: 3 * N], rtol=2e-5, atol=1e-9)
    np.testing.assert_allclose(ang.reshape(-1), ref[3 * N:], rtol=2e-5, atol=1e-9)
    # mean over realisations -> div M = 0; a single sample is O(|dM|) ~ 1e-2
    S = 4000
    acc = np.zeros((N, 3))
    sq = np.zeros((N, 3))
    for _ in range(S):
        l, _ = bd.thermal_drift_rfd(x, rng.standard_normal((N, 3)), 1e-3)
        acc += l
        sq += l * l
    mean, sem = acc / S, np.sqrt(sq / S) / math.sqrt(S)
    assert np.sqrt(sq / S).max() > 1e-3                 # the samples themselves are not small
    assert np.all(np.abs(mean) <= 5 * sem)


def test_b10_steric_force_dimensional_scaling():
    """eq. (13): U depends on r only through (d - r)/b, so scaling all lengths (positions, d, b) by lam at fixed
    U0 scales every force by 1/lam, and the force is linear in U0."""
    rng = np.random.default_rng(10)
    x = rng.random((30, 3)) * 6.0
    F = bd.steric_forces(x, 4.0, 0.1, 2.0)
    for lam in (0.656e-6, 3.0, 1.0e5):
        np.testing.assert_allclose(bd.steric_forces(lam * x, 4.0, 0.1 * lam, 2.0 * lam), F / lam, rtol=1e-10)
    np.testing.assert_allclose(bd.steric_forces(x, 10.0, 0.1, 2.0), 2.5 * F, rtol=1e-13)


def test_b11_row_sampled_steric_forces_equal_the_full_call():
    """``rows=`` (the row-sampled oracle used at N = 131072 by the GPU tests) returns exactly the listed rows of the
    full call -- rows are independent --, in the order listed, duplicates included; an index outside [0, N) is an
    error, never a silent wrap-around of a negative index.  Against the energy gradient too (B2's route), so the
    sampled path is pinned by something other than the full path."""
    rng = np.random.default_rng(11)
    N, U0, b, d = 60, 4.0, 0.1, 2.0
    x = rng.random((N, 3)) * 5.0
    full = bd.steric_forces(x, U0, b, d)
    rows = np.array([0, 17, 17, 59, 3, 0])
    part = bd.steric_forces(x, U0, b, d, rows=rows)
    assert part.shape == (6, 3)
    assert np.array_equal(part, full[rows])
    assert bd.steric_forces(x, U0, b, d, rows=[]).shape == (0, 3)
    assert np.array_equal(bd.steric_forces(x, U0, b, d, rows=range(N)), full)
    for bad in ([N], [-1], [0, N + 5]):
        with pytest.raises((IndexError, ValueError)):
            bd.steric_forces(x, U0, b, d, rows=bad)
    h = 1e-6
    for out, i in enumerate(rows[:4]):
        for k in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, k] += h
            xm[i, k] -= h
            fd = -(energy(xp, U0, b, d) - energy(xm, U0, b, d)) / (2 * h)
            assert part[out, k] == pytest.approx(fd, rel=2e-7, abs=1e-7)
