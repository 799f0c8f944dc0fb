"""GPU parity for the free-space Brownian-dynamics step: lm_steric_forces (eq. 13) and lm_bd_step (eq. 14)
against oracle/bd.py, through the C ABI.  Needs a B200 (``-m gpu``).

Tolerances: steric forces rel-L2 <= 1e-12 (fp64) / 2e-5 (fp32), the M.F gates -- the fp32 exponential is
MUFU ex2 (rel. error ~2^-22 plus ~1.5e-6 from the argument); the cut-off drops terms below exp(-20) / exp(-40).
BD displacements inherit the M.F gates (deterministic part) and the Lanczos gates of DESIGN.md S4 (noise part).
"""
import math

import numpy as np
import pytest

from oracle import bd
from paper_2510_02135_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


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


def case(N, side, seed, prec, angular=False):
    return workloads.random_case(N, side, seed=seed, precision=prec, angular=angular, with_noise=True)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N,side", [(1, 1.0), (2, 1.5), (3, 0.5), (37, 4.0), (129, 5.0), (513, 9.0), (1500, 16.0), (3001, 25.0)])
@pytest.mark.parametrize("with_ext", [False, True])
def test_steric_forces_match_oracle(lm, torch, prec, N, side, with_ext):
    """One thread, one group, unit boundaries +-1, several tiles and j-splits with a ragged tail; cubes that
    start at the origin, where the ghost sources of the padded tail sit."""
    c = case(N, side, 11, prec)
    U0, b = 4.0, 0.1
    s = lm.Solver(prec, N, 1.0, 1.0, False)
    s.set_positions(dev(torch, c["pos"]))
    ext = c["forces"] if with_ext else None
    F = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.steric_forces(U0, b, dev(torch, ext), F)
    torch.cuda.synchronize()
    Fo = bd.steric_forces(c["pos"], U0, b, 2.0)
    if with_ext:
        Fo = Fo + np.asarray(ext, np.float64).reshape(N, 3)
    got = F.cpu().numpy().reshape(N, 3)
    if N == 1 and not with_ext:
        assert np.all(got == 0.0)
        return
    scale = np.abs(Fo).max()
    assert np.abs(got - Fo).max() <= 8 * TOL[prec] * max(scale, U0 / b)
    if np.linalg.norm(Fo) > 0:
        assert rel(got, Fo) <= TOL[prec] * max(1.0, (U0 / b) * math.sqrt(N) / np.linalg.norm(Fo))
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_steric_nonunit_radius_coincident_particles_and_softness(lm, torch, prec):
    rng = np.random.default_rng(3)
    N, a = 200, 0.656                                   # the paper's colloid radius in micrometres
    pos = (rng.random((N, 3)) * 6.0).astype(workloads.np_dtype(prec))
    pos[17] = pos[5]                                    # exactly coincident pair: exerts nothing on each other
    for U0, b in ((4 * 4.11e-3, 0.1 * a), (1.0, 0.5 * a)):
        s = lm.Solver(prec, N, 1.0e-3, a, False)
        s.set_positions(dev(torch, pos))
        F = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
        s.steric_forces(U0, b, None, F)
        torch.cuda.synchronize()
        Fo = bd.steric_forces(pos, U0, b, 2 * a)
        assert rel(F.cpu().numpy(), Fo) <= TOL[prec]
        s.close()


def test_steric_full_size_sampled_rows(lm, torch):
    """Config-3 geometry (N = 131072, phi = 5 %), the launch configuration a BD step uses; sampled rows."""
    data = workloads.generate(3)
    N = data["N"]
    s = lm.Solver("f32", N, 1.0, 1.0, False)
    s.set_positions(dev(torch, data["pos"]))
    F = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.steric_forces(4.0, 0.1, None, F)
    torch.cuda.synchronize()
    rows = np.sort(np.random.default_rng(0).choice(N, 256, replace=False))
    rows[:2] = [0, N - 1]
    Fo = bd.steric_forces(data["pos"], 4.0, 0.1, 2.0, rows=rows)
    got = F.cpu().numpy().reshape(N, 3)[rows]
    assert np.abs(got - Fo).max() <= 8 * 2e-5 * 40.0
    assert rel(got, Fo) <= 2e-5
    # Newton's third law at full size: the total force vanishes to rounding
    tot = F.double().reshape(N, 3).sum(0).abs().max().item()
    assert tot <= 1e-4 * 40.0 * math.sqrt(N)
    s.close()


def run_gpu(lm, torch, prec, c, nsteps, dt, kT, U0, b, tol, angular, ext=True, noise=True, host=False, max_iter=100):
    N = c["pos"].shape[0]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_max_iter(max_iter)
    X = c["pos"].copy().reshape(-1) if host else dev(torch, c["pos"]).reshape(-1).clone()
    conv = (lambda v: None if v is None else np.ascontiguousarray(v).reshape(-1)) if host else (lambda v: None if v is None else dev(torch, v).reshape(-1))
    F = conv(c["forces"]) if ext else None
    T = conv(c["torques"]) if (ext and angular) else None
    traj = []
    for n in range(nsteps):
        W = conv(noise_for(c, n)) if noise else None
        (s.bd_step_host if host else s.bd_step)(X, F, T, W, dt, kT, U0, b, tol)
        traj.append(X.copy() if host else X.cpu().numpy().copy())
    s.close()
    return traj


def noise_for(c, n):
    w = np.asarray(c["noise"])
    return np.roll(w, 7 * n).astype(w.dtype)              # a different, reproducible W^n per step


def run_oracle(c, nsteps, dt, kT, U0, b, tol, angular, ext=True, noise=True, mode="lanczos"):
    x, vprev, traj = np.asarray(c["pos"], np.float64), None, []
    for n in range(nsteps):
        x, vprev, _ = bd.bd_step(x, vprev, dt, kT, U0=U0, b=b, ext_forces=c["forces"] if ext else None,
                                 ext_torques=c["torques"] if (ext and angular) else None, noise=noise_for(c, n) if noise else None,
                                 angular=angular, sqrt_mode=mode, tol=tol)
        traj.append(x.reshape(-1).copy())
    return traj


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
def test_bd_deterministic_trajectory_matches_oracle(lm, torch, prec, angular):
    """kT = 0: Euler start then the 3/2, -1/2 weights, steric + external forces (and torques)."""
    c = case(700, 14.0, 21, prec, angular)
    dt, U0, b = 2e-3, 4.0, 0.1
    g = run_gpu(lm, torch, prec, c, 4, dt, 0.0, U0, b, 1e-3, angular, noise=False)
    o = run_oracle(c, 4, dt, 0.0, U0, b, 1e-3, angular, noise=False)
    x0 = np.asarray(c["pos"], np.float64).reshape(-1)
    for n in range(4):
        # displacement from the start, so that the gate applies to what the step computes
        assert rel(g[n] - x0, o[n] - x0) <= (5e-11 if prec == "f64" else 5e-3), n   # fp32: one ulp of x ~ 1e-6 against a ~1e-3 step
        assert np.abs(g[n] - o[n]).max() <= (1e-12 if prec == "f64" else 2e-6) * np.abs(x0).max()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_bd_stochastic_step_matches_oracle(lm, torch, prec):
    c = case(500, 13.0, 22, prec)
    dt, kT, U0, b = 1e-2, 1.0, 4.0, 0.1
    tol = 1e-5 if prec == "f64" else 1e-3
    g = run_gpu(lm, torch, prec, c, 2, dt, kT, U0, b, tol, False, max_iter=400)
    x0 = np.asarray(c["pos"], np.float64).reshape(-1)
    if prec == "f64":
        o = run_oracle(c, 2, dt, kT, U0, b, tol, False, mode="dense")
        for n in range(2):
            assert rel(g[n] - x0, o[n] - x0) <= 3 * tol       # vs the exact root (S4 iii, default rule)
    else:
        o = run_oracle(c, 2, dt, kT, U0, b, tol, False, mode="lanczos")
        od = run_oracle(c, 2, dt, kT, U0, b, tol, False, mode="dense")
        for n in range(2):
            assert rel(g[n] - x0, o[n] - x0) <= 3 * tol        # same rule, fp32 vs fp64 (S4 ii)
            assert rel(g[n] - x0, od[n] - x0) <= 3 * tol       # vs the exact root (S4 iii)


def test_bd_single_sphere_diffuses_with_stokes_einstein(lm, torch):
    a, eta, kT, dt = 0.7, 1.3, 0.41, 0.02
    s = lm.Solver("f64", 1, eta, a, False)
    X = torch.zeros(3, dtype=torch.float64, device="cuda")
    W = torch.tensor([0.3, -1.2, 2.0], dtype=torch.float64, device="cuda")
    s.bd_step(X, None, None, W, dt, kT, 0.0, 0.1, 1e-10)
    D = kT / (6 * math.pi * eta * a)
    np.testing.assert_allclose(X.cpu().numpy(), math.sqrt(2 * D * dt) * W.cpu().numpy(), rtol=1e-12)
    s.close()


def test_bd_reset_host_variant_and_errors(lm, torch):
    c = case(300, 10.0, 23, "f64")
    dt, U0, b = 1e-3, 4.0, 0.1
    g = run_gpu(lm, torch, "f64", c, 3, dt, 0.5, U0, b, 1e-4, False)
    gh = run_gpu(lm, torch, "f64", c, 3, dt, 0.5, U0, b, 1e-4, False, host=True)
    for n in range(3):
        np.testing.assert_array_equal(g[n], gh[n])
    N = 300
    s = lm.Solver("f64", N, 1.0, 1.0, False)
    X = dev(torch, c["pos"]).reshape(-1).clone()
    F = dev(torch, c["forces"]).reshape(-1)
    out = torch.empty_like(X)
    with pytest.raises(lm.LmError) as e:
        s.steric_forces(U0, b, None, out)                    # positions not set
    assert e.value.code == lm.LM_E_NOPOS
    s.bd_step(X, F, None, None, dt, 0.0, U0, b, 1e-3)        # Euler
    x1 = X.clone()
    s.bd_step(X, F, None, None, dt, 0.0, U0, b, 1e-3)        # AB2
    s.bd_reset()
    X2 = x1.clone()
    s.bd_step(X2, F, None, None, dt, 0.0, U0, b, 1e-3)       # Euler again from the same state
    o1, v0, _ = bd.bd_step(c["pos"], None, dt, 0.0, U0=U0, b=b, ext_forces=c["forces"])
    oe, _, _ = bd.bd_step(o1, None, dt, 0.0, U0=U0, b=b, ext_forces=c["forces"])
    oa, _, _ = bd.bd_step(o1, v0, dt, 0.0, U0=U0, b=b, ext_forces=c["forces"])
    x0 = np.asarray(c["pos"]).reshape(-1)
    assert rel(X2.cpu().numpy() - x0, oe.reshape(-1) - x0) <= 1e-10
    assert rel(X.cpu().numpy() - x0, oa.reshape(-1) - x0) <= 1e-10
    assert rel(oe, oa) > 1e-9                                # the two really differ
    for bad in (dict(dt=0.0), dict(dt=-1.0), dict(kT=-1.0), dict(b=0.0)):
        kw = dict(dt=dt, kT=0.0, U0=U0, b=b)
        kw.update(bad)
        with pytest.raises(lm.LmError) as e:
            s.bd_step(X, F, None, None, kw["dt"], kw["kT"], kw["U0"], kw["b"], 1e-3)
        assert e.value.code == lm.LM_E_INVALID
    with pytest.raises(lm.LmError) as e:
        s.bd_step(X, F, F, None, dt, 0.0, U0, b, 1e-3)       # torques without include_angular
    assert e.value.code == lm.LM_E_ANGULAR
    with pytest.raises(lm.LmError) as e:
        s.steric_forces(U0, -1.0, None, out)
    assert e.value.code in (lm.LM_E_INVALID, lm.LM_E_NOPOS)
    s.close()


@pytest.mark.parametrize("prec,angular,delta", [("f64", False, 1e-3), ("f64", True, 1e-3), ("f32", False, 0.05), ("f32", True, 0.05)])
def test_thermal_drift_rfd_matches_oracle_and_default_is_zero(lm, torch, prec, angular, delta):
    """eq. (11): the difference quotient divides the M.F rounding error by delta, so the gate is the M.F
    gate times |M W| / (delta |RFD|)."""
    from oracle import rpy
    c = case(900, 15.0, 31, prec, angular)
    N = 900
    W = c["noise"][: 3 * N]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_positions(dev(torch, c["pos"]))
    lin = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    ang = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    s.thermal_drift_rfd(dev(torch, W), delta, lin, ang)
    torch.cuda.synchronize()
    lo, ao = bd.thermal_drift_rfd(c["pos"], W, delta, angular=angular)
    U, Om = rpy.mdot(c["pos"], W, None, angular=angular)
    # the displaced positions are rounded to the run precision on the GPU: that alone perturbs M W by ~eps |x| |dM W|
    eps_x = np.finfo(workloads.np_dtype(prec)).eps * np.abs(c["pos"]).max()
    gate = 4 * TOL[prec] * np.linalg.norm(U) / (delta * np.linalg.norm(lo)) + 4 * eps_x / delta
    assert rel(lin.cpu().numpy(), lo) <= gate
    if angular:
        gate_a = 4 * TOL[prec] * np.linalg.norm(Om) / (delta * np.linalg.norm(ao)) + 4 * eps_x / delta
        assert rel(ang.cpu().numpy(), ao) <= gate_a
    # the handle's own positions are untouched: M.F afterwards is M.F at X
    U2 = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.mdot(dev(torch, W), None, U2, ang)
    torch.cuda.synchronize()
    assert rel(U2.cpu().numpy(), U) <= TOL[prec]
    # library default for open boundaries: zero drift
    s.thermal_drift(lin, ang)
    torch.cuda.synchronize()
    assert float(lin.abs().max()) == 0.0 and (ang is None or float(ang.abs().max()) == 0.0)
    with pytest.raises(lm.LmError) as e:
        s.thermal_drift_rfd(dev(torch, W), 0.0, lin, ang)
    assert e.value.code == lm.LM_E_INVALID
    s.close()


def test_bd_step_leaves_the_handle_at_the_new_positions(lm, torch):
    from oracle import rpy
    c = case(400, 11.0, 24, "f64")
    N = 400
    s = lm.Solver("f64", N)
    X = dev(torch, c["pos"]).reshape(-1).clone()
    F = dev(torch, c["forces"]).reshape(-1)
    s.bd_step(X, F, None, None, 1e-2, 0.0, 4.0, 0.1, 1e-3)
    U = torch.empty(3 * N, dtype=torch.float64, device="cuda")
    s.mdot(F, None, U)                                    # no lm_set_positions in between
    torch.cuda.synchronize()
    Uo, _ = rpy.mdot(X.cpu().numpy().reshape(N, 3), c["forces"])
    assert rel(U.cpu().numpy(), Uo) <= 1e-12
    s.close()
