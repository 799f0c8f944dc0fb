"""GPU parity of the single-wall geometry:
the CUDA path through the C ABI (lm_set_wall + the ordinary entry points) against oracle/wall.py, element by element on
the same seeded inputs.  Gates as for the free-space path (tests/test_gpu_parity.py): rel-L2 <= 1e-12 (fp64) / 2e-5
(fp32) plus the element-wise bound."""
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
    return torch


def dev(torch, x):
    return None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()


def gpu_wall_mdot(lm, torch, prec, pos, F, T, angular, a=1.0, eta=1.0, wall_z=0.0, nrhs=1):
    N = pos.shape[0]
    s = lm.Solver(prec, N, eta, a, angular)
    s.set_wall(True, wall_z)
    s.set_positions(dev(torch, pos))
    U = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda")
    W = torch.empty(nrhs * 3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    if nrhs == 1:
        s.mdot(dev(torch, F), dev(torch, T), U, W)
    else:
        s.mdot_batch(nrhs, dev(torch, F).reshape(-1), None if T is None else dev(torch, T).reshape(-1), U, W)
    torch.cuda.synchronize()
    return U.cpu().numpy().reshape(nrhs, N, 3), (W.cpu().numpy().reshape(nrhs, N, 3) if angular else None), s


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("N,side,zlo,zhi", [(1, 1.0, 1.5, 1.5), (2, 1.5, 1.0, 2.0), (3, 0.5, 0.2, 0.9), (37, 4.0, -0.3, 3.0), (129, 6.0, 1.0, 4.0),
                                            (513, 12.0, 0.5, 2.5), (1500, 25.0, 1.0, 2.0), (4097, 40.0, 0.0, 6.0), (9001, 50.0, 0.9, 30.0)])
def test_wall_mdot_matches_oracle(lm, torch, prec, angular, N, side, zlo, zhi):
    c = workloads.wall_slab_case(N, side, zlo, zhi, N, prec, angular, wall_z=-1.25)
    U, W, s = gpu_wall_mdot(lm, torch, prec, c["pos"], c["forces"], c["torques"], angular, wall_z=c["wall_z"])
    Uo, Wo = wall.mdot(c["pos"], c["forces"], c["torques"], wall_z=c["wall_z"], angular=angular)
    assert close(U[0], Uo, TOL[prec]), rel(U[0], Uo)
    if angular:
        assert close(W[0], Wo, TOL[prec]), rel(W[0], Wo)
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_wall_is_not_the_free_space_result_and_can_be_switched_off(lm, torch, prec):
    c = workloads.wall_slab_case(700, 15.0, 0.5, 3.0, 3, prec, True)
    U, W, s = gpu_wall_mdot(lm, torch, prec, c["pos"], c["forces"], c["torques"], True)
    Uf, Wf = rpy.mdot(c["pos"], c["forces"], c["torques"], angular=True)
    assert rel(U[0], Uf) > 0.05
    s.set_wall(False, 0.0)
    with pytest.raises(lm.LmError) as e:                      # lm_set_wall invalidates the positions
        s.mdot(dev(torch, c["forces"]), dev(torch, c["torques"]), dev(torch, np.empty_like(c["forces"])), dev(torch, np.empty_like(c["forces"])))
    assert e.value.code == lm.LM_E_NOPOS
    s.set_positions(dev(torch, c["pos"]))
    U2 = torch.empty(3 * 700, dtype=s.torch_dtype, device="cuda")
    W2 = torch.empty_like(U2)
    s.mdot(dev(torch, c["forces"]), dev(torch, c["torques"]), U2, W2)
    torch.cuda.synchronize()
    assert close(U2.cpu().numpy(), Uf, TOL[prec]) and close(W2.cpu().numpy(), Wf, TOL[prec])
    with pytest.raises(lm.LmError):
        s.set_wall(True, float("nan"))
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("a,eta", [(0.656, 1.0e-3), (1e-6, 1e-3), (37.0, 2.5)])
def test_wall_any_unit_system(lm, torch, prec, a, eta):
    rng = np.random.default_rng(4)
    N = 600
    dt = workloads.np_dtype(prec)
    pos = np.column_stack([rng.random(N) * 20 * a, rng.random(N) * 20 * a, 5 * a + (0.3 + 3 * rng.random(N)) * a]).astype(dt)
    F = (rng.standard_normal((N, 3))).astype(dt)
    T = (rng.standard_normal((N, 3)) * a).astype(dt)
    U, W, s = gpu_wall_mdot(lm, torch, prec, pos, F, T, True, a=a, eta=eta, wall_z=5 * a)
    Uo, Wo = wall.mdot(pos, F, T, a=a, eta=eta, wall_z=5 * a, angular=True)
    assert close(U[0], Uo, TOL[prec]) and close(W[0], Wo, TOL[prec]), (rel(U[0], Uo), rel(W[0], Wo))
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("nrhs", [2, 3, 4, 5])
def test_wall_mdot_batch(lm, torch, prec, angular, nrhs):
    N = 1300
    dt = workloads.np_dtype(prec)
    c = workloads.wall_slab_case(N, 22.0, 0.4, 3.0, 10 + nrhs, prec, angular)
    rng = np.random.default_rng(nrhs)
    F = rng.standard_normal((nrhs, N, 3)).astype(dt)
    T = rng.standard_normal((nrhs, N, 3)).astype(dt) if angular else None
    U, W, s = gpu_wall_mdot(lm, torch, prec, c["pos"], F, T, angular, nrhs=nrhs)
    for q in range(nrhs):
        Uo, Wo = wall.mdot(c["pos"], F[q], T[q] if angular else None, angular=angular)
        assert close(U[q], Uo, TOL[prec])
        if angular:
            assert close(W[q], Wo, TOL[prec])
    s.close()


def test_wall_microroller_size_sampled_rows(lm, torch):
    """The paper's single-wall problem size (N = 2^15, a = 0.656, torque-driven rollers above a wall) on
    the synthetic monolayer of workloads.microroller_monolayer, fp32 with the angular blocks: 96 sampled rows."""
    d = workloads.microroller_monolayer()
    N, a = d["N"], d["a"]
    U, W, s = gpu_wall_mdot(lm, torch, "f32", d["pos"], d["forces"], d["torques"], True, a=a, eta=1.0e-3)
    rows = np.sort(np.random.default_rng(6).choice(N, 96, replace=False))
    Uo, Wo = wall.mdot_rows(d["pos"], rows, d["forces"], d["torques"], a=a, eta=1.0e-3, angular=True)
    assert close(U[0][rows], Uo, 2e-5) and close(W[0][rows], Wo, 2e-5), (rel(U[0][rows], Uo), rel(W[0][rows], Wo))
    s.close()


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
def test_wall_lanczos_and_hydrodynamic_velocities(lm, torch, prec, angular):
    N, tol, pref = 400, 1e-3, 0.7
    c = workloads.wall_slab_case(N, 16.0, 0.3, 3.0, 31, prec, angular, with_noise=True, wall_z=0.5)
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_wall(True, c["wall_z"])
    s.set_positions(dev(torch, c["pos"]))
    y = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    ya = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    # fixed-k iterates against the fp64 Lanczos oracle run on the wall operator
    for k, bound in ((3, 1e-12 if prec == "f64" else 3e-6), (8, 1e-10 if prec == "f64" else 1e-5)):
        s.set_max_iter(k)
        s.sqrt_mdot_w(dev(torch, c["noise"]), 1e-30, y, ya, allow_noconv=True)
        torch.cuda.synchronize()
        got = np.concatenate([y.cpu().numpy(), ya.cpu().numpy()]) if angular else y.cpu().numpy()
        yo, ko, _ = wall.lanczos_sqrt_mdot_w(c["pos"], c["noise"], 1e-30, wall_z=c["wall_z"], angular=angular, max_iter=k)
        assert rel(got, yo) <= bound, (k, rel(got, yo))
    # the stopping rule against the exact dense root of the damped wall mobility
    s.set_max_iter(100)
    it = s.sqrt_mdot_w(dev(torch, c["noise"]), tol, y, ya)
    torch.cuda.synchronize()
    got = np.concatenate([y.cpu().numpy(), ya.cpu().numpy()]) if angular else y.cpu().numpy()
    exact = wall.dense_sqrt_mdot_w(c["pos"], c["noise"], wall_z=c["wall_z"], angular=angular)
    assert 3 <= it < 100 and rel(got, exact) <= 3 * tol, (it, rel(got, exact))
    # lm_hydrodynamic_velocities = M.[F;T] + pref M^{1/2} W (shared first launch)
    H = torch.empty_like(y)
    Ha = torch.empty_like(y) if angular else None
    s.hydrodynamic_velocities(dev(torch, c["forces"]), dev(torch, c["torques"]), dev(torch, c["noise"]), pref, tol, H, Ha)
    torch.cuda.synchronize()
    Uo, Wo = wall.mdot(c["pos"], c["forces"], c["torques"], wall_z=c["wall_z"], angular=angular)
    assert rel(H.cpu().numpy(), Uo.reshape(-1) + pref * exact[:3 * N]) <= 3 * tol
    if angular:
        assert rel(Ha.cpu().numpy(), Wo.reshape(-1) + pref * exact[3 * N:]) <= 3 * tol
    s.close()


@pytest.mark.parametrize("prec,angular,nvec", [("f64", False, 4), ("f32", False, 5), ("f64", True, 3)])
def test_wall_sqrt_mdot_w_batch(lm, torch, prec, angular, nvec):
    """Several noise vectors above a wall: the wall variants of the pair kernel serve 1 and 2 right-hand sides, so a batch of
    4 or more must be grouped 2 + 2 (+ 1), not refused; every vector against the exact dense root of the damped wall mobility."""
    N, tol = 300, 1e-3
    c = workloads.wall_slab_case(N, 14.0, 0.3, 3.0, 61, prec, angular, with_noise=True, wall_z=0.25)
    dof = (6 if angular else 3) * N
    W = np.random.default_rng(200 + nvec).standard_normal((nvec, dof)).astype(workloads.np_dtype(prec))
    W[0] = c["noise"]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_wall(True, c["wall_z"])
    s.set_positions(dev(torch, c["pos"]))
    lin = torch.empty(nvec * 3 * N, dtype=s.torch_dtype, device="cuda")
    ang = torch.empty(nvec * 3 * N, dtype=s.torch_dtype, device="cuda") if angular else None
    iters = s.sqrt_mdot_w_batch(nvec, dev(torch, W).reshape(-1), tol, lin, ang)
    torch.cuda.synchronize()
    lin = lin.cpu().numpy().reshape(nvec, 3 * N)
    ang = ang.cpu().numpy().reshape(nvec, 3 * N) if angular else None
    for q in range(nvec):
        y = lin[q] if not angular else np.concatenate([lin[q], ang[q]])
        exact = wall.dense_sqrt_mdot_w(c["pos"], W[q], wall_z=c["wall_z"], angular=angular)
        assert 3 <= iters[q] < 100 and rel(y, exact) <= 3 * tol, (q, iters[q], rel(y, exact))
    s.close()


def test_wall_default_thermal_drift_is_refused(lm, torch):
    """lm_thermal_drift is the zero default of open boundaries; above a wall the divergence is not zero
    (PAPER.md:87), so the call must say so instead of returning zeros."""
    N = 64
    c = workloads.wall_slab_case(N, 8.0, 0.5, 3.0, 5, "f64", False)
    s = lm.Solver("f64", N)
    s.set_wall(True, 0.0)
    s.set_positions(dev(torch, c["pos"]))
    lin = torch.full((3 * N,), 5.0, dtype=torch.float64, device="cuda")
    with pytest.raises(lm.LmError) as e:
        s.thermal_drift(lin)
    assert e.value.code == lm.LM_E_INVALID and "lm_thermal_drift_rfd" in str(e.value)
    torch.cuda.synchronize()
    assert bool((lin == 5.0).all())
    s.set_wall(False, 0.0)
    s.set_positions(dev(torch, c["pos"]))
    s.thermal_drift(lin)
    torch.cuda.synchronize()
    assert float(lin.abs().max()) == 0.0
    s.close()


@pytest.mark.parametrize("prec,angular,delta", [("f64", False, 1e-3), ("f64", True, 1e-3), ("f32", False, 0.05), ("f32", True, 0.05)])
def test_wall_thermal_drift_rfd(lm, torch, prec, angular, delta):
    """eq. (11) with the wall mobility, same W on both sides; and its non-zero mean for one sphere:
    the average over the six unit vectors +-e_c... (W = e_c, c = 0..2 summed) equals d mu_perp/dh."""
    N = 500
    c = workloads.wall_slab_case(N, 18.0, 0.3, 3.0, 41, prec, angular, with_noise=True)
    W = c["noise"][:3 * N]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_wall(True, 0.0)
    s.set_positions(dev(torch, c["pos"]))
    lin = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    ang = torch.empty_like(lin) if angular else None
    s.thermal_drift_rfd(dev(torch, W), delta, lin, ang)
    torch.cuda.synchronize()
    lo, ao = wall.thermal_drift_rfd(c["pos"], W, delta, angular=angular)
    # a difference quotient: rounding is amplified by |U| / (delta |dU|)
    gate = 1e-9 if prec == "f64" else 2e-3
    assert rel(lin.cpu().numpy(), lo) <= gate, rel(lin.cpu().numpy(), lo)
    if angular:
        assert rel(ang.cpu().numpy(), ao) <= gate * 5
    s.close()
    if prec == "f64" and not angular:
        h = 1.7
        s1 = lm.Solver("f64", 1)
        s1.set_wall(True, 0.0)
        s1.set_positions(dev(torch, np.array([[0.0, 0.0, h]])))
        tot = np.zeros(3)
        out = torch.empty(3, dtype=torch.float64, device="cuda")
        for cdir in range(3):
            e = np.zeros(3)
            e[cdir] = 1.0
            s1.thermal_drift_rfd(dev(torch, e), 1e-4, out)
            tot += out.cpu().numpy()
        eps = 1.0 / h
        want = (1 / (6 * np.pi)) * (9 / 8 * eps - 3 / 2 * eps ** 3 + 5 / 8 * eps ** 5) / h
        np.testing.assert_allclose(tot, [0, 0, want], rtol=1e-6, atol=1e-10)
        s1.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_wall_steric_forces(lm, torch, prec):
    """eq. (13): particle-particle (d = 2a, at the TRUE positions, not the raised ones) + particle-wall (d = a)."""
    N, a, U0, b = 900, 0.8, 4.0, 0.08
    c = workloads.wall_slab_case(N, 14.0, -0.1, 2.5, 51, prec, False, wall_z=1.0)
    s = lm.Solver(prec, N, 1.0, a, False)
    s.set_wall(True, c["wall_z"])
    s.set_positions(dev(torch, c["pos"]))
    out = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    s.steric_forces(U0, b, dev(torch, c["forces"]).reshape(-1), out)
    torch.cuda.synchronize()
    want = bd.steric_forces(c["pos"], U0, b, 2 * a) + wall.wall_steric_forces(c["pos"], U0, b, a, c["wall_z"]) + c["forces"].astype(np.float64)
    assert close(out.cpu().numpy(), want, 1e-12 if prec == "f64" else 2e-5), rel(out.cpu().numpy(), want)
    s.close()


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
def test_wall_bd_step_with_drift_matches_oracle(lm, torch, prec, angular):
    """eq. (14) above a wall: steric forces between particles and with the wall, external forces and
    torques, the drift term as one RFD sample, the Lanczos noise -- three steps (Euler, then Adams-Bashforth) against
    oracle/wall.bd_step (dense root), same W^n and W~^n on both sides; host variant bit-identical."""
    N, dt, kT, U0, b, tol = 300, 2e-3, 0.4, 4.0, 0.1, (1e-6 if prec == "f64" else 1e-3)
    delta = 1e-3 if prec == "f64" else 0.05
    c = workloads.wall_slab_case(N, 14.0, 0.6, 2.5, 71, prec, angular, with_noise=True, wall_z=-2.0)
    dtp = workloads.np_dtype(prec)
    rng = np.random.default_rng(72)
    Wn = [np.roll(c["noise"], 5 * n) for n in range(3)]
    Wt = [rng.standard_normal(3 * N).astype(dtp) for n in range(3)]
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_wall(True, c["wall_z"])
    s.set_max_iter(300)
    X = dev(torch, c["pos"]).reshape(-1).clone()
    F, T = dev(torch, c["forces"]).reshape(-1), (dev(torch, c["torques"]).reshape(-1) if angular else None)
    traj = []
    for n in range(3):
        s.bd_step_rfd(X, F, T, dev(torch, Wn[n]), dev(torch, Wt[n]), delta, dt, kT, U0, b, tol)
        traj.append(X.cpu().numpy().copy())
    s.close()
    sh = lm.Solver(prec, N, 1.0, 1.0, angular)
    sh.set_wall(True, c["wall_z"])
    sh.set_max_iter(300)
    Xh = c["pos"].copy().reshape(-1)
    for n in range(3):
        sh.bd_step_rfd_host(Xh, c["forces"].reshape(-1), c["torques"].reshape(-1) if angular else None, Wn[n], Wt[n], delta, dt, kT, U0, b, tol)
        np.testing.assert_array_equal(Xh, traj[n])
    sh.close()
    x, vprev = np.asarray(c["pos"], np.float64), None
    x0 = x.reshape(-1).copy()
    for n in range(3):
        x, vprev, _ = wall.bd_step(x, vprev, dt, kT, wall_z=c["wall_z"], U0=U0, b=b, ext_forces=c["forces"], ext_torques=c["torques"] if angular else None,
                                   noise=Wn[n], rfd_noise=Wt[n], delta=delta, angular=angular, sqrt_mode="dense")
        # the displacement is dominated by the noise term (tolerance 3 tol, S4 iii); fp32: difference quotient of the drift
        gate = 3 * tol + (0.0 if prec == "f64" else 2e-3)
        assert rel(traj[n] - x0, x.reshape(-1) - x0) <= gate, (n, rel(traj[n] - x0, x.reshape(-1) - x0))
    # deterministic part alone (no noise): tight
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_wall(True, c["wall_z"])
    X = dev(torch, c["pos"]).reshape(-1).clone()
    x, vprev = np.asarray(c["pos"], np.float64), None
    for n in range(2):
        s.bd_step_rfd(X, F, T, None, dev(torch, Wt[n]), delta, dt, kT, U0, b, tol)
        x, vprev, _ = wall.bd_step(x, vprev, dt, kT, wall_z=c["wall_z"], U0=U0, b=b, ext_forces=c["forces"], ext_torques=c["torques"] if angular else None,
                                   rfd_noise=Wt[n], delta=delta, angular=angular)
        assert rel(X.cpu().numpy() - x0, x.reshape(-1) - x0) <= (1e-9 if prec == "f64" else 2e-3), (n, rel(X.cpu().numpy() - x0, x.reshape(-1) - x0))
    s.close()
