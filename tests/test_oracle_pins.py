"""Pins for the CPU oracle's M.F family (oracle/rpy_oracle.c) -- CPU only, no CUDA code involved.

Every check compares the oracle with something fixed by the paper or by mathematics, not with a
retyped copy of its own formulas:

P1  self mobility 1/(6 pi eta a) and 1/(8 pi eta a^3)
P2  continuity of the five pair scalars across r = 2a
P3  Oseen limit  8 pi eta r M_uF -> I + rr^T
P4  two-sphere sedimentation closed forms (textbook Rotne-Prager)
P5  dense M symmetric positive definite, translational and full 6N
P6  divergence-free => zero thermal drift in bulk
P7  the integral DEFINITION eq. (8) / eq. (4) evaluated by quadrature over
    the two spheres, for the tt, rt and rr blocks, in both the overlap and the far branch
P8  handedness of the translation-rotation coupling (S6)
P9  brute force: independent numpy double loop; dense M @ [F;T]; row-sampled == full
G   golden typo guards (tests/golden, surveyor-computed)
"""
import math
import os

import numpy as np
import pytest

from oracle import rpy

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_rows(name):
    rows = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("a,eta", [(1.0, 1.0), (0.656, 1.0e-3), (2.5, 3.0)])
def test_p1_self_mobility(a, eta):
    F = np.array([[0.3, -2.0, 1.5]])
    T = np.array([[1.0, 0.25, -0.5]])
    U, W = rpy.mdot(np.array([[4.0, -1.0, 2.0]]), F, T, a=a, eta=eta, angular=True)
    np.testing.assert_allclose(U, F / (6 * math.pi * eta * a), rtol=1e-15)
    np.testing.assert_allclose(W, T / (8 * math.pi * eta * a ** 3), rtol=1e-15)
    consts = {r[0]: float(r[1]) for r in _read_rows("closed_form_constants.txt")}
    s = rpy.pair_scalars(0.0)
    assert s[0] == pytest.approx(consts["self_tt"], rel=1e-14)
    assert s[2] == pytest.approx(consts["self_rr"], rel=1e-14)
    assert s[1] == 0.0 and s[3] == 0.0 and s[4] == 0.0


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("a,eta", [(1.0, 1.0), (0.37, 2.2)])
def test_p2_continuity_at_2a(a, eta):
    lo = rpy.pair_scalars(2 * a * (1 - 1e-9), a, eta)
    hi = rpy.pair_scalars(2 * a * (1 + 1e-9), a, eta)
    at = rpy.pair_scalars(2 * a, a, eta)
    scale = 1.0 / (8 * math.pi * eta * a ** 3) * np.array([a * a, a * a, 1, 1, a])
    assert np.all(np.abs(lo - hi) < 1e-8 * scale)
    assert np.all(np.abs(at - hi) < 1e-8 * scale)
    # first derivatives of the tt scalars are continuous too (C^1 at contact): a wrong
    # coefficient in either branch that happens to keep the value would show here
    h = 1e-6 * a
    for k in (0, 1):
        dlo = (rpy.pair_scalars(2 * a - h, a, eta)[k] - rpy.pair_scalars(2 * a - 2 * h, a, eta)[k]) / h
        dhi = (rpy.pair_scalars(2 * a + 2 * h, a, eta)[k] - rpy.pair_scalars(2 * a + h, a, eta)[k]) / h
        assert abs(dlo - dhi) < 1e-4 * abs(dhi)


# ---------------------------------------------------------------- P3
def test_p3_oseen_limit():
    a, eta = 1.0, 1.3
    for r in (1e2, 1e3, 1e4):
        s = rpy.pair_scalars(r, a, eta)
        assert abs(8 * math.pi * eta * r * s[0] - 1.0) < 1.0 * (a / r) ** 2
        assert abs(8 * math.pi * eta * r * s[1] - 1.0) < 2.1 * (a / r) ** 2
    # tensor form: a unit force along x at the origin moves a far particle on the x axis twice as
    # fast as one on the y axis (Stokeslet: (I + rr^T)/(8 pi eta r))
    pos = np.array([[0, 0, 0], [1e4, 0, 0], [0, 1e4, 0.0]])
    F = np.array([[1.0, 0, 0], [0, 0, 0], [0, 0, 0]])
    U, _ = rpy.mdot(pos, F, a=a, eta=eta)
    assert U[1, 0] / U[2, 0] == pytest.approx(2.0, rel=1e-7)
    assert U[2, 0] == pytest.approx(1 / (8 * math.pi * eta * 1e4), rel=1e-7)


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("r", [2.0, 2.5, 4.0, 11.0])
def test_p4_two_sphere_sedimentation(r):
    a, eta = 1.0, 1.0
    mu0 = 1 / (6 * math.pi * eta * a)
    pos = np.array([[0, 0, 0], [0, 0, r]], dtype=float)
    Fpar = np.array([[0, 0, 1.0], [0, 0, 1.0]])
    Fperp = np.array([[1.0, 0, 0], [1.0, 0, 0]])
    U, _ = rpy.mdot(pos, Fpar)
    np.testing.assert_allclose(U[:, 2], mu0 * (1 + 3 * a / (2 * r) - a ** 3 / r ** 3), rtol=1e-14)
    U, _ = rpy.mdot(pos, Fperp)
    np.testing.assert_allclose(U[:, 0], mu0 * (1 + 3 * a / (4 * r) + a ** 3 / (2 * r ** 3)), rtol=1e-14)


# ---------------------------------------------------------------- P5
@pytest.mark.parametrize("side", [3.0, 6.0, 20.0])
@pytest.mark.parametrize("angular", [False, True])
def test_p5_dense_symmetric_positive_definite(side, angular):
    rng = np.random.default_rng(int(side) + 10 * angular)
    pos = rng.random((40, 3)) * side
    M = rpy.dense(pos, angular=angular)
    assert np.abs(M - M.T).max() <= 4e-16 * np.abs(M).max()      # symmetric up to rounding order
    lam = np.linalg.eigvalsh(M)
    assert lam.min() > 1e-4, lam.min()


def test_p5_coupling_blocks_are_transposes():
    rng = np.random.default_rng(3)
    N = 12
    pos = rng.random((N, 3)) * 4
    M = rpy.dense(pos, angular=True)
    MuT, MwF = M[:3 * N, 3 * N:], M[3 * N:, :3 * N]
    assert np.abs(MuT - MwF.T).max() <= 4e-16 * np.abs(MuT).max()   # M_uT^{ij} = (M_wF^{ji})^T
    for i in range(N):                          # no self coupling
        assert np.all(MuT[3 * i:3 * i + 3, 3 * i:3 * i + 3] == 0)


# ---------------------------------------------------------------- P6
@pytest.mark.parametrize("r0", [0.7, 1.9, 2.1, 5.0])
def test_p6_divergence_free(r0):
    """sum_l d/dx_l M_uF,kl(x) = 0: finite-difference divergence of the pair tensor (both branches)."""
    a = eta = 1.0
    base = np.array([0.3, -0.5, 0.81])
    base = base / np.linalg.norm(base) * r0
    h = 1e-5

    def tensor(x):
        r = np.linalg.norm(x)
        s = rpy.pair_scalars(r, a, eta)
        e = x / r
        return s[0] * np.eye(3) + s[1] * np.outer(e, e)

    div = np.zeros(3)
    for l in range(3):
        dx = np.zeros(3)
        dx[l] = h
        div += (tensor(base + dx)[:, l] - tensor(base - dx)[:, l]) / (2 * h)
    assert np.all(np.abs(div) < 1e-9), div


# ---------------------------------------------------------------- P7
def _gl(lo, hi, n=48):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (hi - lo) * x + 0.5 * (lo + hi), 0.5 * (hi - lo) * w


_NPHI = 16
_PHI = (np.arange(_NPHI) + 0.5) * 2 * np.pi / _NPHI


def _surface_average(R, a, field):
    """Average of field(x, s) over the sphere |x - R zhat| = a, parametrised by s = |x| (the
    distance from the other sphere's centre, at the origin) so that the kink at s = a is a
    sub-interval boundary: dA / (4 pi a^2) = s ds dphi / (4 pi R a)."""
    bps = [b for b in sorted({abs(R - a), a, R + a}) if abs(R - a) <= b <= R + a]
    tot = np.zeros(3)
    for lo, hi in zip(bps[:-1], bps[1:]):
        for s, w in zip(*_gl(lo, hi)):
            u = (s * s - R * R - a * a) / (2 * R * a)
            st = math.sqrt(max(0.0, 1 - u * u))
            pts = np.stack([a * st * np.cos(_PHI), a * st * np.sin(_PHI), np.full(_NPHI, R + a * u)], -1)
            tot += w * s / (2 * R * a) * field(pts, s).mean(0)
    return tot


def _ball_average(R, a, field):
    """Average of field(x, s) over the ball |x - R zhat| < a, in spherical coordinates about the
    origin: for each s the ball cuts the sphere of radius s in the cap cos(theta) >= u_min(s)."""
    bps = sorted({0.0 if R < a else R - a, abs(R - a), a, R + a})
    tot = np.zeros(3)
    for lo, hi in zip(bps[:-1], bps[1:]):
        if hi - lo < 1e-14:
            continue
        for s, ws in zip(*_gl(lo, hi)):
            umin = min(max((s * s + R * R - a * a) / (2 * s * R), -1.0), 1.0)
            if umin >= 1.0:
                continue
            uu, wu = _gl(umin, 1.0)
            st = np.sqrt(1 - uu ** 2)
            pts = s * np.stack([np.outer(st, np.cos(_PHI)), np.outer(st, np.sin(_PHI)),
                                np.outer(uu, np.ones(_NPHI))], -1)
            tot += ws * s * s * np.einsum("u,upk->k", wu, field(pts, s)) * (2 * np.pi / _NPHI)
    return tot / (4 / 3 * np.pi * a ** 3)


@pytest.mark.parametrize("q", [0.2, 0.8, 1.0, 1.7, 2.0, 2.6, 4.0])
def test_p7_integral_definition_of_all_blocks(q):
    """eq. (8) with delta_F = surface delta of radius a, and eq. (4)
    with delta_T = uniform ball of radius a (the regularisations that DEFINE the RPY tensors; the
    paper leaves them generic, S1).  Particle j sits at the origin, particle i at R zhat.

    tt: a force F spread over sphere j drives the textbook Stokes flow of a translating sphere
        (outside: (1 + a^2/6 lap) Oseen . F, inside: rigid F/(6 pi eta a)); U_i is its average over
        the SURFACE of sphere i.
    rt: W_i = 1/2 <curl v> over the BALL i; the sphere-j surface average of half the curl of a
        Stokeslet, F x rho /(8 pi eta rho^3), is by the shell theorem F x s/(8 pi eta s^3) outside
        sphere j and 0 inside.
    rr: a torque T spread over ball j drives v = T x s /(8 pi eta max(s,a)^3) (ball potential);
        1/2 curl v = T/(8 pi eta a^3) inside, (3 (T.shat) shat - T)/(16 pi eta s^3) outside;
        W_i is its average over the BALL i.
    """
    a, eta = 1.3, 0.7
    R = q * a
    F = np.array([0.3, -1.1, 0.8])
    T = np.array([-0.6, 0.4, 1.2])
    z = np.array([0.0, 0.0, 1.0])            # rhat = (x_i - x_j)/R

    def v_translating_sphere(pts, s):
        if s < a:
            return np.broadcast_to(F / (6 * np.pi * eta * a), pts.shape)
        sh = pts / s
        return ((1 / s + a * a / (3 * s ** 3)) * F + (1 / s - a * a / s ** 3) * (sh @ F)[..., None] * sh) / (8 * np.pi * eta)

    def half_curl_from_force(pts, s):
        if s < a:
            return np.zeros(pts.shape)
        return np.cross(F, pts) / s ** 3 / (8 * np.pi * eta)

    def half_curl_from_torque(pts, s):
        if s < a:
            return np.broadcast_to(T / (8 * np.pi * eta * a ** 3), pts.shape)
        sh = pts / s
        return (3 * (sh @ T)[..., None] * sh - T) / s ** 3 / (16 * np.pi * eta)

    sc = rpy.pair_scalars(R, a, eta)
    pos = np.array([[0, 0, 0], [0, 0, R]])
    zero = np.zeros(3)
    # through the oracle's own summation: source j = particle 0, read target i = particle 1,
    # subtracting nothing: particle 1 carries no force, so U_1 is the pure pair term
    U, W = rpy.mdot(pos, np.array([F, zero]), np.array([zero, zero]), a, eta, angular=True)
    np.testing.assert_allclose(U[1], _surface_average(R, a, v_translating_sphere), rtol=0, atol=1e-12)
    np.testing.assert_allclose(W[1], _ball_average(R, a, half_curl_from_force), rtol=0, atol=1e-12)
    U, W = rpy.mdot(pos, np.array([zero, zero]), np.array([T, zero]), a, eta, angular=True)
    np.testing.assert_allclose(W[1], _ball_average(R, a, half_curl_from_torque), rtol=0, atol=1e-12)
    # and M_uT is the transpose of M_wF: velocity of i from a torque on j
    np.testing.assert_allclose(U[1], sc[4] * np.cross(T, z), rtol=0, atol=1e-15)


# ---------------------------------------------------------------- P8
def test_p8_coupling_handedness():
    consts = {r[0]: float(r[1]) for r in _read_rows("closed_form_constants.txt")}
    zero = [0.0, 0.0, 0.0]
    # T = +z at the origin: a particle at +x (r = 5) moves along +y (rotlet u = T x r /(8 pi eta r^3))
    pos = np.array([[0, 0, 0], [5.0, 0, 0]])
    U, W = rpy.mdot(pos, np.array([zero, zero]), np.array([[0, 0, 1.0], zero]), angular=True)
    np.testing.assert_allclose(U[1], [0, consts["rotlet_r5"], 0], atol=1e-18)
    # F = +x at the origin: a particle at +y spins about +z (omega = curl u / 2 = F x r/(8 pi eta r^3))
    pos = np.array([[0, 0, 0], [0, 5.0, 0]])
    U, W = rpy.mdot(pos, np.array([[1.0, 0, 0], zero]), np.array([zero, zero]), angular=True)
    np.testing.assert_allclose(W[1], [0, 0, consts["rotlet_r5"]], atol=1e-18)


# ---------------------------------------------------------------- P9
def _numpy_double_loop(pos, F, T, a, eta):
    """Independent restatement with dense 3x3 blocks built from outer products / cross matrices
    (a different arrangement from the C loop): u_i += A F_j + B^T-type couplings."""
    N = len(pos)
    U = np.zeros((N, 3))
    W = np.zeros((N, 3))
    for i in range(N):
        for j in range(N):
            d = pos[i] - pos[j]
            r = math.sqrt(d @ d)
            s = rpy.pair_scalars(r, a, eta)
            e = d / r if r > 0 else np.zeros(3)
            P = np.outer(e, e)
            X = np.array([[0, -e[2], e[1]], [e[2], 0, -e[0]], [-e[1], e[0], 0]])   # X v = e x v
            U[i] += (s[0] * np.eye(3) + s[1] * P) @ F[j] - s[4] * X @ T[j]
            W[i] += (s[2] * np.eye(3) + s[3] * P) @ T[j] - s[4] * X @ F[j]
    return U, W


def test_p9_brute_force_and_dense():
    rng = np.random.default_rng(11)
    N, a, eta = 23, 0.9, 1.7
    pos = rng.random((N, 3)) * 5.0
    pos[7] = pos[3]                              # exactly coincident pair (S5)
    F, T = rng.standard_normal((N, 3)), rng.standard_normal((N, 3))
    U, W = rpy.mdot(pos, F, T, a, eta, angular=True)
    U2, W2 = _numpy_double_loop(pos, F, T, a, eta)
    np.testing.assert_allclose(U, U2, rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(W, W2, rtol=1e-13, atol=1e-15)
    M = rpy.dense(pos, a, eta, angular=True)
    y = M @ np.concatenate([F.reshape(-1), T.reshape(-1)])
    np.testing.assert_allclose(np.concatenate([U.reshape(-1), W.reshape(-1)]), y, rtol=1e-13, atol=1e-15)
    Mt = rpy.dense(pos, a, eta, angular=False)
    assert np.array_equal(Mt, M[:3 * N, :3 * N])
    Ut, none = rpy.mdot(pos, F, None, a, eta)
    assert none is None
    np.testing.assert_allclose(Ut.reshape(-1), Mt @ F.reshape(-1), rtol=1e-13, atol=1e-15)
    # forces=None means zero forces
    U0, W0 = rpy.mdot(pos, None, T, a, eta, angular=True)
    np.testing.assert_allclose(np.concatenate([U0.reshape(-1), W0.reshape(-1)]),
                               M[:, 3 * N:] @ T.reshape(-1), rtol=1e-13, atol=1e-15)
    with pytest.raises(ValueError):
        rpy.mdot(pos, F, T, a, eta, angular=False)


def test_p9_row_sampled_equals_full():
    rng = np.random.default_rng(5)
    N = 301
    pos = rng.random((N, 3)) * 12
    F, T = rng.standard_normal((N, 3)), rng.standard_normal((N, 3))
    rows = np.array([0, 17, 300, 5, 5])
    U, W = rpy.mdot(pos, F, T, angular=True)
    Ur, Wr = rpy.mdot_rows(pos, rows, F, T, angular=True)
    assert np.array_equal(Ur, U[rows]) and np.array_equal(Wr, W[rows])
    with pytest.raises(ValueError):
        rpy.mdot_rows(pos, [N], F)


def test_p9_translation_rotation_invariance():
    """Free space: M depends on relative positions only, and rotates as a tensor."""
    rng = np.random.default_rng(8)
    N = 17
    pos = rng.random((N, 3)) * 6
    F, T = rng.standard_normal((N, 3)), rng.standard_normal((N, 3))
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1                           # proper rotation: pseudo-vectors rotate like vectors
    U, W = rpy.mdot(pos, F, T, angular=True)
    U2, W2 = rpy.mdot(pos @ Q.T + np.array([100.0, -3.0, 7.0]), F @ Q.T, T @ Q.T, angular=True)
    np.testing.assert_allclose(U2, U @ Q.T, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(W2, W @ Q.T, rtol=1e-9, atol=1e-12)


# ---------------------------------------------------------------- golden typo guards
def test_golden_pair_scalars():
    for row in _read_rows("survey_pair_scalars.txt"):
        vals = [float(v) for v in row]
        np.testing.assert_allclose(rpy.pair_scalars(vals[0]), vals[1:], rtol=1e-13)


def test_golden_two_particle():
    g = {r[0]: np.array([float(v) for v in r[1:]]).reshape(2, 3) for r in _read_rows("survey_two_particle.txt")}
    U, W = rpy.mdot(g["pos"], g["F"], g["T"], angular=True)
    np.testing.assert_allclose(U, g["U_near"], rtol=1e-12)
    np.testing.assert_allclose(W, g["W_near"], rtol=1e-12)
    U, W = rpy.mdot(2.5 * g["pos"], g["F"], g["T"], angular=True)
    np.testing.assert_allclose(U, g["U_far"], rtol=1e-12)
    np.testing.assert_allclose(W, g["W_far"], rtol=1e-12)
    U, _ = rpy.mdot(2.5 * g["pos"], g["F"])
    np.testing.assert_allclose(U, g["U_far_t"], rtol=1e-12)


@pytest.mark.parametrize("lam,eta", [(0.37, 1.0), (2.5e-6, 1e-3), (1.0e4, 7.0)])
def test_p11_dimensional_scaling(lam, eta):
    """Dimensional analysis of Stokes flow: with every length (positions AND radius) scaled by lam and the
    viscosity by eta, the four blocks of eq. (7) scale as  M_uF ~ 1/(eta lam),  M_uT = M_wF ~ 1/(eta lam^2),
    M_wT ~ 1/(eta lam^3).  A wrong power of a anywhere in the ten scalar formulas (either branch) breaks it."""
    rng = np.random.default_rng(11)
    N = 14
    x = rng.random((N, 3)) * 5.0                      # overlapping and separated pairs at a = 1
    F, T = rng.standard_normal((N, 3)), rng.standard_normal((N, 3))
    zero = np.zeros((N, 3))
    UF, WF = rpy.mdot(x, F, zero, angular=True)        # a = eta = 1
    UT, WT = rpy.mdot(x, zero, T, angular=True)
    UF2, WF2 = rpy.mdot(lam * x, F, zero, a=lam, eta=eta, angular=True)
    UT2, WT2 = rpy.mdot(lam * x, zero, T, a=lam, eta=eta, angular=True)
    np.testing.assert_allclose(UF2, UF / (eta * lam), rtol=1e-12)
    np.testing.assert_allclose(WF2, WF / (eta * lam ** 2), rtol=1e-12)
    np.testing.assert_allclose(UT2, UT / (eta * lam ** 2), rtol=1e-12)
    np.testing.assert_allclose(WT2, WT / (eta * lam ** 3), rtol=1e-12)
