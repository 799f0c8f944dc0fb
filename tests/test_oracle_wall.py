"""Pins of the single-wall (Swan-Brady) oracle, ``oracle/wall.py`` + ``oracle/wall_oracle.c`` (all ``-m "not gpu"``).

PAPER.md prints neither the wall tensors nor the damping matrix, so the oracle's closed forms are pinned
by what the paper's DEFINITION and the mathematics fix, with nothing taken from the oracle itself:

  W0  an independent implementation of the half-space Green's function (Blake's image system), written out below
      in index form, is itself pinned: no slip on the wall, incompressible, a Stokes flow (curl of its Laplacian
      vanishes), reciprocal G(x,y) = G(y,x)^T, and its singular part is the Oseen tensor.  A Stokes flow in the
      half space that vanishes on the wall and at infinity is unique, so these fix it.
  W1  eq. (8): M^w_uF = the double surface average of the image part over the two spheres (quadrature).
  W2  eq. (4) + eq. (3): the coupling and rotation blocks = surface averages of 1/2 curl (complex-step
      derivatives of W0's tensor).
  W3  the Faxen form (1 + a^2/6 lap_x)(1 + a^2/6 lap_y) G_im by finite differences (reading S18's exactness claim).
  W4  one sphere above the wall: the known series of its mobilities in a/h -- translation parallel (Faxen) and
      perpendicular (Lorentz), rotation, translation-rotation coupling (refs. [37], [51] of the paper), to the order
      the RPY level keeps; the rolling direction of the coupling.
  W5  far from the wall the free-space oracle is recovered.
  W6  dense M symmetric positive (semi-)definite with particles overlapping each other and the wall.
  W7  damping (reading S19): continuity at h = a, (h/a)^2 below, zero at and under the wall.
  W8  invariances: shift and rotation in the plane, joint shift of wall and particles, mirror symmetry.
  W9  rows == full == dense @ [F;T]; dimensional scaling.
  W10 thermal drift: the RFD of eq. (11) summed over unit vectors is the central-difference divergence; the divergence
      of one sphere is d mu_perp / dh; a Monte-Carlo mean of RFD samples approaches it.
  W11 wall steric force of eq. (13) with d = a: minus the derivative of the potential.
  W12 the time step of eq. (14) above a wall: one sphere settling (dt mu_perp F), its drift displacement
      (dt kT d mu_perp/dh), Adams-Bashforth weights, noise term, and the free-space step far from the wall.
"""
import math

import numpy as np
import pytest

from oracle import bd, rpy, wall

PI = math.pi


# ---------------------------------------------------------------- W0: Blake's tensor, index form, units 1/(8 pi eta)
def oseen(r):
    r = np.asarray(r)
    n = np.sqrt(np.sum(r * r, axis=-1))
    G = np.zeros(r.shape[:-1] + (3, 3), dtype=r.dtype)
    for i in range(3):
        for j in range(3):
            G[..., i, j] = (i == j) / n + r[..., i] * r[..., j] / n ** 3
    return G


def blake_image(x, y):
    """G_im[i][j](x, y): velocity component i at x per unit force component j at y, minus the Oseen tensor; wall z = 0.
    R = x - y*, y* the mirror image of y, h = y_3, Delta = diag(1, 1, -1):
        G_im_ij = -(d_ij/R + R_i R_j/R^3) + 2 h Delta_jj d/dR_j [ h R_i/R^3 - (d_i3/R + R_i R_3/R^3) ]."""
    x, y = np.asarray(x), np.asarray(y)
    h = y[..., 2]
    R = np.stack([x[..., 0] - y[..., 0], x[..., 1] - y[..., 1], x[..., 2] + y[..., 2]], axis=-1)
    n = np.sqrt(np.sum(R * R, axis=-1))            # analytic in the coordinates: complex-step safe
    G = np.zeros(np.broadcast(x[..., 0], y[..., 0]).shape + (3, 3), dtype=np.result_type(x, y))
    for i in range(3):
        for j in range(3):
            dij, di3, dj3 = float(i == j), float(i == 2), float(j == 2)
            stokeslet = dij / n + R[..., i] * R[..., j] / n ** 3
            d_dipole = h * (dij / n ** 3 - 3 * R[..., i] * R[..., j] / n ** 5)                      # d/dR_j (h R_i / R^3)
            d_rest = (-di3 * R[..., j] / n ** 3                                                       # d/dR_j (d_i3 / R)
                      + (dij * R[..., 2] + R[..., i] * dj3) / n ** 3 - 3 * R[..., i] * R[..., 2] * R[..., j] / n ** 5)
            G[..., i, j] = -stokeslet + 2 * h * (-1.0 if j == 2 else 1.0) * (d_dipole - d_rest)
    return G


def blake(x, y):
    return oseen(np.asarray(x) - np.asarray(y)) + blake_image(x, y)


def test_w0_blake_tensor_is_the_half_space_greens_function():
    rng = np.random.default_rng(0)
    for _ in range(20):
        y = np.array([rng.normal(), rng.normal(), 0.2 + 3 * rng.random()])
        xw = np.array([rng.normal() * 3, rng.normal() * 3, 0.0])
        assert np.abs(blake(xw, y)).max() <= 1e-13 * np.abs(oseen(xw - y)).max()             # no slip
        x = np.array([rng.normal(), rng.normal(), 0.2 + 3 * rng.random()])
        np.testing.assert_allclose(blake(x, y), blake(y, x).T, rtol=1e-12, atol=1e-14)       # reciprocity
        # incompressible: d/dx_i G_im_ij = 0 (complex step)
        eps = 1e-30
        div = np.zeros(3)
        for i in range(3):
            xc = x.astype(complex)
            xc[i] += 1j * eps
            div += blake_image(xc, y)[i, :].imag / eps
        assert np.abs(div).max() <= 1e-12
        # Stokes: eta lap u = grad p  =>  curl_x (lap_x G_im[:, j]) = 0   (Laplacian by central differences of the
        # complex-step gradient)
        s = 1e-3

        def grad(xx):                                # g[k][i][j] = d G_im_ij / d x_k
            g = np.zeros((3, 3, 3))
            for k in range(3):
                xc = xx.astype(complex)
                xc[k] += 1j * eps
                g[k] = blake_image(xc, y).imag / eps
            return g

        lap_grad = np.zeros((3, 3, 3))               # lap of d_k G_ij
        for m in range(3):
            e = np.zeros(3)
            e[m] = s
            lap_grad += (grad(x + e) - 2 * grad(x) + grad(x - e)) / s ** 2
        for j in range(3):
            curl = np.array([lap_grad[1, 2, j] - lap_grad[2, 1, j], lap_grad[2, 0, j] - lap_grad[0, 2, j], lap_grad[0, 1, j] - lap_grad[1, 0, j]])
            assert np.abs(curl).max() <= 1e-4 * (1.0 + np.abs(lap_grad).max())
    # the image part is regular where the Oseen tensor is singular (x -> y)
    y = np.array([0.3, -0.2, 1.1])
    assert np.abs(blake_image(y + 1e-9, y)).max() < 10.0


# ---------------------------------------------------------------- sphere quadrature
def sphere_nodes(n=20):
    """Product rule on the unit sphere: Gauss-Legendre in cos(theta) x uniform in phi; weights sum to 1.  Exact for
    polynomials of degree < 2n; the integrands here are analytic, so it converges geometrically."""
    t, w = np.polynomial.legendre.leggauss(n)
    phi = (np.arange(2 * n) + 0.5) * (PI / n)
    st = np.sqrt(1 - t * t)
    pts = np.stack([np.outer(st, np.cos(phi)), np.outer(st, np.sin(phi)), np.outer(t, np.ones_like(phi))], axis=-1).reshape(-1, 3)
    wts = np.repeat(w / 2, 2 * n) / (2 * n)
    return pts, wts


def averaged(fn, xi, xj, a, n=20):
    """<< fn(x, y) >> over x on the sphere (xi, a) and y on the sphere (xj, a): eq. (8) with surface deltas."""
    pts, wts = sphere_nodes(n)
    X = xi + a * pts
    Y = xj + a * pts
    vals = fn(X[:, None, :], Y[None, :, :])                   # (nx, ny, 3, 3)
    return np.einsum("p,q,pqij->ij", wts, wts, vals)


def half_curl_x(x, y, eps=1e-30):
    """1/2 eps_ikl d/dx_k G_im_lj : angular velocity at x per unit force at y (eq. (4))."""
    x = np.asarray(x)
    g = []
    for k in range(3):
        xc = x.astype(complex).copy()
        xc[..., k] += 1j * eps
        g.append(blake_image(xc, y).imag / eps)               # g[k][..., l, j]
    out = np.zeros_like(g[0])
    out[..., 0, :] = 0.5 * (g[1][..., 2, :] - g[2][..., 1, :])
    out[..., 1, :] = 0.5 * (g[2][..., 0, :] - g[0][..., 2, :])
    out[..., 2, :] = 0.5 * (g[0][..., 1, :] - g[1][..., 0, :])
    return out


def half_curl_y_rows(x, y, eps=1e-30, fn=blake_image):
    """1/2 eps_nml d/dy_m G_kl : velocity component k at x per unit TORQUE component n at y (force density
    1/2 curl(T delta), eq. (3), integrated by parts)."""
    y = np.asarray(y)
    g = []
    for m in range(3):
        yc = y.astype(complex).copy()
        yc[..., m] += 1j * eps
        g.append(fn(x, yc).imag / eps)                        # g[m][..., k, l]
    out = np.zeros_like(g[0])
    out[..., :, 0] = 0.5 * (g[1][..., :, 2] - g[2][..., :, 1])
    out[..., :, 1] = 0.5 * (g[2][..., :, 0] - g[0][..., :, 2])
    out[..., :, 2] = 0.5 * (g[0][..., :, 1] - g[1][..., :, 0])
    return out


def quarter_curl_curl(x, y, s=1e-4):
    """1/4 curl_x curl_y G_im: angular velocity at x per unit torque at y.  Complex step in y, central differences in x."""
    x = np.asarray(x, dtype=float)
    g = []
    for k in range(3):
        e = np.zeros(3)
        e[k] = s
        g.append((half_curl_y_rows(x + e, y) - half_curl_y_rows(x - e, y)) / (2 * s))     # d/dx_k of (u_l per T_n)
    out = np.zeros_like(g[0])
    out[..., 0, :] = 0.5 * (g[1][..., 2, :] - g[2][..., 1, :])
    out[..., 1, :] = 0.5 * (g[2][..., 0, :] - g[0][..., 2, :])
    out[..., 2, :] = 0.5 * (g[0][..., 1, :] - g[1][..., 0, :])
    return out


PAIRS = [  # (xi, xj, a): heights above the wall > a, including the self pair, touching-range and far pairs
    ((0.0, 0.0, 1.5), (0.0, 0.0, 1.5), 1.0),
    ((0.3, -0.4, 1.3), (0.3, -0.4, 2.9), 1.0),
    ((1.7, 0.6, 2.2), (-0.8, 1.1, 1.4), 1.0),
    ((4.0, -3.0, 1.25), (-2.0, 5.0, 6.0), 1.0),
    ((0.2, 0.1, 0.9), (-0.3, 0.5, 0.45), 0.35),
]


@pytest.mark.parametrize("xi,xj,a", PAIRS)
def test_w1_w2_blocks_are_the_surface_averages_of_eq8(xi, xj, a):
    xi, xj = np.array(xi), np.array(xj)
    eta = 0.7
    uF, uT, wF, wT = wall.pair_correction(xi, xj, a, eta)
    c = 1.0 / (8 * PI * eta)
    ref_uF = c * averaged(blake_image, xi, xj, a)
    ref_wF = c * averaged(half_curl_x, xi, xj, a)
    ref_uT = c * averaged(half_curl_y_rows, xi, xj, a)
    scale = np.abs(ref_uF).max()
    np.testing.assert_allclose(uF, ref_uF, rtol=0, atol=2e-9 * scale)
    np.testing.assert_allclose(wF, ref_wF, rtol=0, atol=2e-9 * np.abs(ref_wF).max())
    np.testing.assert_allclose(uT, ref_uT, rtol=0, atol=2e-9 * np.abs(ref_uT).max())
    ref_wT = c * averaged(quarter_curl_curl, xi, xj, a, n=12)
    np.testing.assert_allclose(wT, ref_wT, rtol=0, atol=2e-6 * np.abs(ref_wT).max())
    # the blocks are not degenerate: every one of them is non-zero for a generic pair
    if not np.allclose(xi[:2], xj[:2]):
        assert all(np.abs(B).max() > 0 for B in (uF, uT, wF, wT))


def test_w2b_free_space_coupling_has_the_same_definition():
    """The same quadrature applied to the Oseen tensor reproduces the FREE-space coupling of oracle/rpy (non-overlapping
    pair): the curl conventions used in W2 are those of the free-space pins (P7/P8)."""
    xi, xj, a, eta = np.array([1.0, 0.4, 2.0]), np.array([-1.5, 0.2, 0.3]), 1.0, 1.0
    ref = averaged(lambda x, y: half_curl_y_rows(x, y, fn=lambda p, q: oseen(p - q)), xi, xj, a) / (8 * PI * eta)
    d = xi - xj
    r = np.linalg.norm(d)
    e = d / r
    gc = rpy.pair_scalars(r, a, eta)[4]
    ex = np.array([[0, -e[2], e[1]], [e[2], 0, -e[0]], [-e[1], e[0], 0]])
    np.testing.assert_allclose(ref, -gc * ex, atol=1e-10)


def test_w3_faxen_operators_by_finite_differences():
    xi, xj, a, eta = np.array([0.9, -0.3, 1.8]), np.array([-0.6, 0.7, 1.3]), 1.0, 1.0
    s = 2e-3

    def lap(f, which):
        def g(x, y):
            out = -6 * f(x, y)
            for m in range(3):
                e = np.zeros(3)
                e[m] = s
                out = out + (f(x + e, y) + f(x - e, y) if which == "x" else f(x, y + e) + f(x, y - e))
            return out / s ** 2
        return g

    gy = lambda x, y: blake_image(x, y) + a * a / 6 * lap(blake_image, "y")(x, y)
    full = gy(xi, xj) + a * a / 6 * lap(gy, "x")(xi, xj)
    uF = wall.pair_correction(xi, xj, a, eta)[0]
    np.testing.assert_allclose(uF, full / (8 * PI * eta), rtol=0, atol=1e-4 * np.abs(uF).max())


# ---------------------------------------------------------------- W4: one sphere above a wall
@pytest.mark.parametrize("a,eta", [(1.0, 1.0), (0.656, 1.0e-3)])
@pytest.mark.parametrize("eps", [1.0, 0.8, 0.5, 0.2, 0.05])
def test_w4_single_sphere_series(a, eta, eps):
    """eps = a/h.  mu_par/mu_0 = 1 - 9/16 eps + 1/8 eps^3 - 1/16 eps^5 (Faxen; its eps^4 term is beyond the RPY level),
    mu_perp/mu_0 = 1 - 9/8 eps + 1/2 eps^3 - 1/8 eps^5 (Lorentz),  rotation 1 - 5/16 eps^3 (axis parallel to the wall)
    and 1 - 1/8 eps^3 (axis normal), coupling (3/32) eps^4 / (6 pi eta a^2)."""
    h = a / eps
    M = wall.dense(np.array([[0.3, -1.2, h + 2.5]]), a, eta, wall_z=2.5, angular=True)
    mu_t, mu_r = 1 / (6 * PI * eta * a), 1 / (8 * PI * eta * a ** 3)
    par = 1 - 9 / 16 * eps + eps ** 3 / 8 - eps ** 5 / 16
    perp = 1 - 9 / 8 * eps + eps ** 3 / 2 - eps ** 5 / 8
    want = np.zeros((6, 6))
    want[0, 0] = want[1, 1] = mu_t * par
    want[2, 2] = mu_t * perp
    want[3, 3] = want[4, 4] = mu_r * (1 - 5 / 16 * eps ** 3)
    want[5, 5] = mu_r * (1 - eps ** 3 / 8)
    cpl = 3 / 32 * eps ** 4 / (6 * PI * eta * a * a)
    # rolling: a torque about +y drives the sphere towards +x, a torque about +x towards -y (and reciprocally)
    want[0, 4] = want[4, 0] = cpl
    want[1, 3] = want[3, 1] = -cpl
    np.testing.assert_allclose(M, want, rtol=1e-12, atol=1e-14 * mu_r + 1e-14 * mu_t)


def test_w5_free_space_limit_far_from_the_wall():
    rng = np.random.default_rng(3)
    x = rng.random((12, 3)) * 6.0
    Mf = rpy.dense(x, 1.0, 1.0, angular=True)
    errs = []
    for H in (1e2, 1e3, 1e4):
        xs = x + np.array([0, 0, H])
        errs.append(np.abs(wall.dense(xs, 1.0, 1.0, 0.0, angular=True) - Mf).max())
    assert errs[0] < 2e-3 and errs[1] < errs[0] / 8 and errs[2] < errs[1] / 8          # O(1/H)
    F = rng.standard_normal((12, 3))
    U, _ = wall.mdot(x + np.array([0, 0, 1e9]), F)
    np.testing.assert_allclose(U, rpy.mdot(x, F)[0], rtol=1e-6)


# ---------------------------------------------------------------- W6, W7: SPD and damping
@pytest.mark.parametrize("angular", [False, True])
@pytest.mark.parametrize("seed,side,zlo,zhi", [(0, 4.0, 1.0, 4.0), (1, 3.0, 0.05, 2.0), (2, 6.0, -0.5, 1.5), (3, 2.0, 0.3, 0.9)])
def test_w6_dense_mobility_is_symmetric_positive_definite(angular, seed, side, zlo, zhi):
    rng = np.random.default_rng(seed)
    N = 30
    x = np.column_stack([rng.random(N) * side, rng.random(N) * side, zlo + rng.random(N) * (zhi - zlo)])
    M = wall.dense(x, 1.0, 1.0, 0.0, angular)
    assert np.abs(M - M.T).max() <= 1e-15 * np.abs(M).max() * 10
    lam = np.linalg.eigvalsh(0.5 * (M + M.T))
    if zlo > 0:
        assert lam.min() > 0, lam.min()
    else:                                            # particles at or under the wall have b = 0: zero rows, semi-definite
        assert lam.min() > -1e-13 * lam.max()
        stuck = np.where(x[:, 2] <= 0)[0]
        assert stuck.size > 0
        for i in stuck:
            assert np.all(M[3 * i:3 * i + 3] == 0) and np.all(M[:, 3 * i:3 * i + 3] == 0)
    if angular:                                      # coupling blocks are each other's transposes
        n3 = 3 * N
        np.testing.assert_allclose(M[:n3, n3:], M[n3:, :n3].T, atol=1e-15)


def test_w6b_undamped_kernel_is_not_spd_but_the_damped_one_is():
    """the reason for the damping.  The Faxen closed forms evaluated at the TRUE heights of particles that
    cut the wall are not a surface average any more and lose definiteness; reading S19 evaluates them at raised heights."""
    a = 1.0
    x = np.array([[0.0, 0.0, 0.15], [0.4, 0.0, 0.2]])
    # closed forms at the true heights, assembled by hand from the oracle's own pair blocks
    M = np.zeros((6, 6))
    for i in range(2):
        for j in range(2):
            d = x[i] - x[j]
            r = np.linalg.norm(d)
            s = rpy.pair_scalars(r, a, 1.0)
            e = d / r if r > 0 else np.zeros(3)
            M[3 * i:3 * i + 3, 3 * j:3 * j + 3] = s[0] * np.eye(3) + s[1] * np.outer(e, e) + wall.pair_correction(x[i], x[j], a, 1.0)[0]
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() < 0
    assert np.linalg.eigvalsh(wall.dense(x, a, 1.0)).min() > 0


def test_w7_damping_matrix():
    a, eta = 0.8, 1.3
    at_a = wall.dense(np.array([[0.0, 0.0, a]]), a, eta, 0.0, True)
    for h in (0.999 * a, 0.5 * a, 0.1 * a, 1e-6 * a):
        M = wall.dense(np.array([[0.0, 0.0, h]]), a, eta, 0.0, True)
        np.testing.assert_allclose(M, (h / a) ** 2 * at_a, rtol=1e-13)
    np.testing.assert_allclose(wall.dense(np.array([[0.0, 0.0, a * (1 + 1e-9)]]), a, eta, 0.0, True), at_a, rtol=1e-8)   # continuous at h = a
    assert np.all(wall.dense(np.array([[0.0, 0.0, 0.0]]), a, eta, 0.0, True) == 0)
    assert np.all(wall.dense(np.array([[0.0, 0.0, -0.3]]), a, eta, 0.0, True) == 0)
    xt, b = wall.damping(np.array([[0, 0, 2.0], [0, 0, 0.4], [0, 0, -1.0]]), a, 0.0)
    np.testing.assert_allclose(b, [1.0, 0.5, 0.0])
    np.testing.assert_allclose(xt[:, 2], [2.0, a, a])
    # pair: M~_ij = b_i b_j M_ij(raised heights)
    x = np.array([[0.0, 0.0, 0.3 * a], [1.5, 0.2, 2.0]])
    xr = x.copy()
    xr[0, 2] = a
    B = np.diag(np.repeat([0.3, 1.0], 3))
    np.testing.assert_allclose(wall.dense(x, a, eta), B @ wall.dense(xr, a, eta) @ B, rtol=1e-13)


# ---------------------------------------------------------------- W8, W9
def _case(seed, N=25, angular=True):
    rng = np.random.default_rng(seed)
    x = np.column_stack([rng.random(N) * 5, rng.random(N) * 5, 0.2 + rng.random(N) * 3])
    return x, rng.standard_normal((N, 3)), rng.standard_normal((N, 3)) if angular else None


def test_w8_invariances():
    x, F, T = _case(5)
    U, W = wall.mdot(x, F, T, angular=True)
    # shift in the plane; joint shift of wall and particles along z
    U2, W2 = wall.mdot(x + np.array([3.0, -7.0, 0.0]), F, T, angular=True)
    np.testing.assert_allclose(U2, U, rtol=1e-11, atol=1e-13)
    U3, W3 = wall.mdot(x + np.array([0.0, 0.0, -4.2]), F, T, wall_z=-4.2, angular=True)
    np.testing.assert_allclose(U3, U, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(W3, W, rtol=1e-11, atol=1e-13)
    # rotation about the wall normal
    th = 0.7
    Q = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1]])
    U4, W4 = wall.mdot(x @ Q.T, F @ Q.T, T @ Q.T, angular=True)
    np.testing.assert_allclose(U4, U @ Q.T, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(W4, W @ Q.T, rtol=1e-11, atol=1e-13)
    # mirror x -> -x: polar vectors flip their x component, axial vectors (T, omega) flip y and z
    P, A = np.diag([-1.0, 1.0, 1.0]), np.diag([1.0, -1.0, -1.0])
    U5, W5 = wall.mdot(x @ P, F @ P, T @ A, angular=True)
    np.testing.assert_allclose(U5, U @ P, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(W5, W @ A, rtol=1e-11, atol=1e-13)
    # a mirror through the wall is NOT a symmetry
    assert np.abs(wall.mdot(x, F)[0] - rpy.mdot(x, F)[0]).max() > 1e-3


def test_w9_rows_full_dense_and_scaling():
    x, F, T = _case(6, N=40)
    for angular in (False, True):
        Tt = T if angular else None
        U, W = wall.mdot(x, F, Tt, a=0.9, eta=1.7, wall_z=0.1, angular=angular)
        M = wall.dense(x, 0.9, 1.7, 0.1, angular)
        v = np.concatenate([F.reshape(-1), T.reshape(-1)]) if angular else F.reshape(-1)
        out = M @ v
        np.testing.assert_allclose(U.reshape(-1), out[:120], rtol=1e-12, atol=1e-14)
        if angular:
            np.testing.assert_allclose(W.reshape(-1), out[120:], rtol=1e-12, atol=1e-14)
        rows = np.array([39, 0, 7, 7, 21])
        Ur, Wr = wall.mdot_rows(x, rows, F, Tt, 0.9, 1.7, 0.1, angular)
        np.testing.assert_array_equal(Ur, U[rows])
        if angular:
            np.testing.assert_array_equal(Wr, W[rows])
        np.testing.assert_allclose(wall.apply_vec(x, v, 0.9, 1.7, 0.1, angular), out, rtol=1e-12, atol=1e-14)
    with pytest.raises(ValueError):
        wall.mdot_rows(x, [40], F)
    with pytest.raises(ValueError):
        wall.mdot(x, F, T, angular=False)
    # forces only / torques only
    U0, W0 = wall.mdot(x, None, T, angular=True)
    U1, W1 = wall.mdot(x, np.zeros_like(F), T, angular=True)
    np.testing.assert_array_equal(U0, U1)
    # dimensional analysis: lengths x L, viscosity x c  =>  tt / (c L), tr / (c L^2), rr / (c L^3)
    L, c = 3.0, 0.25
    Ma = wall.dense(x, 0.9, 1.7, 0.1, True)
    Mb = wall.dense(x * L, 0.9 * L, 1.7 * c, 0.1 * L, True)
    n3 = 120
    np.testing.assert_allclose(Mb[:n3, :n3], Ma[:n3, :n3] / (c * L), rtol=1e-11, atol=1e-16)
    np.testing.assert_allclose(Mb[:n3, n3:], Ma[:n3, n3:] / (c * L ** 2), rtol=1e-11, atol=1e-16)
    np.testing.assert_allclose(Mb[n3:, n3:], Ma[n3:, n3:] / (c * L ** 3), rtol=1e-11, atol=1e-16)


def test_w9b_square_roots():
    x, _, _ = _case(8, N=30)
    rng = np.random.default_rng(9)
    for angular in (False, True):
        z = rng.standard_normal((6 if angular else 3) * 30)
        y = wall.dense_sqrt_mdot_w(x, z, angular=angular)
        yy = wall.dense_sqrt_mdot_w(x, y, angular=angular)
        np.testing.assert_allclose(yy, wall.apply_vec(x, z, angular=angular), rtol=1e-9, atol=1e-12)
        yl, k, conv = wall.lanczos_sqrt_mdot_w(x, z, 1e-4, angular=angular)
        assert conv and np.linalg.norm(yl - y) <= 2e-4 * np.linalg.norm(y)


# ---------------------------------------------------------------- W10: thermal drift
def test_w10_thermal_drift():
    a, eta = 1.0, 1.0
    # one sphere: (d/dX).M = d mu_perp/dh zhat, mu_perp = mu_0 (1 - 9/8 e + 1/2 e^3 - 1/8 e^5), e = a/h
    for h in (1.2, 2.0, 5.0):
        div = wall.divergence_fd(np.array([[0.0, 0.0, h]]), a, eta)
        e = a / h
        want = (1 / (6 * PI * eta * a)) * (9 / 8 * e - 3 / 2 * e ** 3 + 5 / 8 * e ** 5) / h
        np.testing.assert_allclose(div, [0, 0, want], rtol=1e-6, atol=1e-9)
    # under the damping the mobility grows like h^2: divergence 2 h / a^2 mu_perp(a)
    div = wall.divergence_fd(np.array([[0.0, 0.0, 0.4]]), a, eta)
    mu_perp_a = wall.dense(np.array([[0.0, 0.0, a]]), a, eta)[2, 2]
    np.testing.assert_allclose(div, [0, 0, 2 * 0.4 * mu_perp_a], rtol=1e-6, atol=1e-9)
    # several particles: the RFD of eq. (11) summed over the unit vectors IS the central-difference divergence
    x = np.array([[0.0, 0.0, 1.3], [1.9, 0.3, 1.1], [0.5, 2.2, 2.4], [2.5, 2.0, 0.7]])
    delta = 2e-5
    for angular in (False, True):
        div = wall.divergence_fd(x, a, eta, angular=angular, step=delta / 2)
        acc_l, acc_a = np.zeros((4, 3)), np.zeros((4, 3))
        for c in range(12):
            W = np.zeros(12)
            W[c] = 1.0
            lin, ang = wall.thermal_drift_rfd(x, W, delta, a, eta, angular=angular)
            acc_l += lin
            if angular:
                acc_a += ang
        got = np.concatenate([acc_l.reshape(-1), acc_a.reshape(-1)]) if angular else acc_l.reshape(-1)
        np.testing.assert_allclose(got, div, rtol=1e-9, atol=1e-12)
        assert np.abs(div[:12]).max() > 1e-3                      # non-zero near a wall
    # free space: the same construction gives zero
    Wz = np.zeros(12)
    tot = np.zeros((4, 3))
    for c in range(12):
        Wz[:] = 0
        Wz[c] = 1.0
        tot += bd.thermal_drift_rfd(x, Wz, 1e-4)[0]
    assert np.abs(tot).max() < 1e-9
    # Monte-Carlo mean of Gaussian samples approaches the divergence (standard error ~ 1/sqrt(n))
    rng = np.random.default_rng(0)
    n = 4000
    mean = np.zeros((4, 3))
    for _ in range(n):
        mean += wall.thermal_drift_rfd(x, rng.standard_normal(12), 1e-4, a, eta)[0]
    mean /= n
    div = wall.divergence_fd(x, a, eta).reshape(4, 3)
    assert np.abs(mean - div).max() < 6 * 0.12 / math.sqrt(n) + 1e-4, np.abs(mean - div).max()


def test_w11_wall_steric_force_is_minus_the_gradient_of_eq13():
    a, U0, b, wz = 0.7, 4.0, 0.07, -1.0
    x = np.array([[0.0, 0.0, wz + 0.2], [1.0, 2.0, wz + 0.7 - 1e-9], [1.0, 2.0, wz + 0.7 + 1e-9], [3.0, 1.0, wz + 1.0], [0.0, 5.0, wz + 4.0]])
    F = wall.wall_steric_forces(x, U0, b, a, wz)
    assert np.all(F[:, :2] == 0)
    s = 1e-6
    for i in (0, 3, 4):
        r = x[i, 2] - wz
        dU = (bd.steric_potential(r + s, U0, b, a) - bd.steric_potential(r - s, U0, b, a)) / (2 * s)
        assert F[i, 2] == pytest.approx(-dU, rel=1e-6)
    assert F[1, 2] == pytest.approx(F[2, 2], rel=1e-6) == pytest.approx(U0 / b, rel=1e-6)     # C^1 potential: continuous force at r = d
    assert F[4, 2] < 1e-18 * U0 / b * 1e3 or F[4, 2] < 1e-15


def test_w12_bd_step_above_a_wall():
    a, eta, dt, kT = 1.0, 1.0, 1e-2, 0.3
    h = 1.8
    e = a / h
    mu_perp = (1 - 9 / 8 * e + e ** 3 / 2 - e ** 5 / 8) / (6 * PI * eta * a)
    dmu = (9 / 8 * e - 3 / 2 * e ** 3 + 5 / 8 * e ** 5) / h / (6 * PI * eta * a)
    x0 = np.array([[0.0, 0.0, h]])
    # settling under a force: forward Euler on the first step
    x1, v0, _ = wall.bd_step(x0, None, dt, 0.0, ext_forces=np.array([[0.0, 0.0, -2.0]]))
    np.testing.assert_allclose(x1, [[0, 0, h - dt * 2.0 * mu_perp]], rtol=1e-13)
    np.testing.assert_allclose(v0, [[0, 0, -2.0 * mu_perp]], rtol=1e-13)
    # the drift alone (rfd_noise = e_z makes the sample the central difference of mu_perp)
    x1d, vd, _ = wall.bd_step(x0, None, dt, kT, rfd_noise=np.array([0.0, 0.0, 1.0]), delta=1e-4)
    np.testing.assert_allclose(x1d[0, 2] - h, dt * kT * dmu, rtol=1e-6)
    assert x1d[0, 2] > h                                            # pushes away from the wall
    assert np.all(wall.bd_step(x0, None, dt, 0.0, rfd_noise=np.array([0.0, 0.0, 1.0]))[0] == x0)   # kT = 0: no drift
    # second step: 3/2 v^1 - 1/2 v^0 (eq. (14)), v including the drift
    x2, v1, _ = wall.bd_step(x1d, vd, dt, kT, ext_forces=np.array([[0.3, 0.0, -1.0]]), rfd_noise=np.array([0.0, 0.0, 1.0]), delta=1e-4)
    _, v1_alone, _ = wall.bd_step(x1d, None, dt, kT, ext_forces=np.array([[0.3, 0.0, -1.0]]), rfd_noise=np.array([0.0, 0.0, 1.0]), delta=1e-4)
    np.testing.assert_allclose(v1, v1_alone, rtol=1e-14)
    np.testing.assert_allclose(x2, x1d + dt * (1.5 * v1 - 0.5 * vd), rtol=1e-14)
    # noise term: sqrt(2 kT dt) M^{1/2} W with the dense root
    rng = np.random.default_rng(1)
    x = np.column_stack([rng.random(20) * 6, rng.random(20) * 6, 0.4 + rng.random(20) * 2])
    W = rng.standard_normal(60)
    xn, _, _ = wall.bd_step(x, None, dt, kT, noise=W)
    np.testing.assert_allclose((xn - x).reshape(-1), math.sqrt(2 * kT * dt) * wall.dense_sqrt_mdot_w(x, W), rtol=1e-12, atol=1e-15)
    xl, _, info = wall.bd_step(x, None, dt, kT, noise=W, sqrt_mode="lanczos", tol=1e-5)
    assert info["iterations"] > 3 and np.linalg.norm(xl - xn) <= 5e-5 * np.linalg.norm(xn - x)
    # steric forces: particle-particle at the true positions plus particle-wall
    F = rng.standard_normal((20, 3))
    xs, vs, _ = wall.bd_step(x, None, dt, 0.0, U0=4.0, b=0.1, ext_forces=F)
    Ftot = bd.steric_forces(x, 4.0, 0.1, 2 * a) + wall.wall_steric_forces(x, 4.0, 0.1, a) + F
    np.testing.assert_allclose(vs, wall.mdot(x, Ftot)[0], rtol=1e-13)
    # far from the wall: the free-space step of oracle/bd
    xf = x + np.array([0, 0, 1e7])
    a1, _, _ = wall.bd_step(xf, None, dt, kT, U0=4.0, b=0.1, ext_forces=F, noise=W)
    b1, _, _ = bd.bd_step(xf, None, dt, kT, U0=4.0, b=0.1, ext_forces=F, noise=W)
    np.testing.assert_allclose(a1 - xf, b1 - xf, rtol=1e-4, atol=1e-9)
