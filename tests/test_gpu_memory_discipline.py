"""Memory and race discipline of every kernel variant, checked with the library's own means (SURVEY.md sec. 5 asks for
compute-sanitizer memcheck / racecheck / initcheck; the tool is closed on this GPU pool -- profiles/r2_sanitizer.md quotes
the refusal -- so the same questions are put directly):

  out-of-bounds writes    every caller buffer (inputs AND outputs) lives inside a larger allocation whose guard bands are
                          filled with a NaN sentinel pattern; after the call the guards are bit-for-bit untouched;
  out-of-bounds reads     the inputs' neighbours are NaN: a kernel that read one element past an array would poison its
                          results, which are compared with the CPU oracle;
  uninitialised reads     the handle's internal scratch (packed vectors, partial sums, Lanczos basis) is poisoned by
                          first running the same call with NaN inputs on the same handle (the scratch then holds
                          NaN), then the real call, whose results must be clean;
  races                   each variant is run 8 times; a data race shows as run-to-run differences, so the outputs
                          must be bit-identical (all reductions are fixed-order by design).
"""
import numpy as np
import pytest

from oracle import bd, rpy, wall
from paper_2510_02135_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}
GUARD = 4096          # elements on each side


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


class Guarded:
    """n elements in the middle of an allocation of n + 2 GUARD, the rest NaN."""

    def __init__(self, torch, n, dtype, init=None):
        self.torch, self.n = torch, n
        self.buf = torch.full((n + 2 * GUARD,), float("nan"), dtype=dtype, device="cuda")
        self.view = self.buf[GUARD:GUARD + n]
        if init is not None:
            self.view.copy_(torch.from_numpy(np.ascontiguousarray(init).reshape(-1)).cuda())

    def guards_intact(self):
        g = self.torch.cat([self.buf[:GUARD], self.buf[GUARD + self.n:]])
        return bool(self.torch.isnan(g).all())


SHAPES = {"cluster": (333, 1), "small": (333, 0), "large": (9000, 0)}


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("angular,nrhs", [(False, 1), (False, 2), (False, 4), (True, 1), (True, 2)])
@pytest.mark.parametrize("with_wall", [False, True])
@pytest.mark.parametrize("shape", ["cluster", "small", "large"])
def test_apply_touches_only_its_buffers_and_is_deterministic(lm, torch, prec, angular, nrhs, with_wall, shape):
    N, mode = SHAPES[shape]
    side = 1.6 * N ** (1.0 / 3.0)
    if with_wall:
        c = workloads.wall_slab_case(N, side * 1.5, -0.2, 4.0, 11 + nrhs, prec, angular, wall_z=0.5)
    else:
        c = workloads.random_case(N, side, 11 + nrhs, prec, angular)
    rng = np.random.default_rng(nrhs)
    dt = workloads.np_dtype(prec)
    F = np.stack([c["forces"]] + [rng.standard_normal((N, 3)).astype(dt) for _ in range(nrhs - 1)])
    T = np.stack([c["torques"]] + [rng.standard_normal((N, 3)).astype(dt) for _ in range(nrhs - 1)]) if angular else None
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    tdt = s.torch_dtype
    if with_wall:
        s.set_wall(True, c["wall_z"])
    s.set_option(lm.LM_OPT_SMALL_KERNEL, mode)
    gpos = Guarded(torch, 3 * N, tdt, c["pos"])
    gF = Guarded(torch, nrhs * 3 * N, tdt, F)
    gT = Guarded(torch, nrhs * 3 * N, tdt, T) if angular else None
    gU = Guarded(torch, nrhs * 3 * N, tdt)
    gW = Guarded(torch, nrhs * 3 * N, tdt) if angular else None
    s.set_positions(gpos.view)
    # poison the handle's scratch: the same call with NaN right-hand sides first
    nanF = torch.full_like(gF.view, float("nan"))
    s.mdot_batch(nrhs, nanF, nanF if angular else None, gU.view, gW.view if angular else None)
    runs = []
    for _ in range(8):
        gU.view.fill_(float("nan"))
        if angular:
            gW.view.fill_(float("nan"))
        s.mdot_batch(nrhs, gF.view, gT.view if angular else None, gU.view, gW.view if angular else None)
        torch.cuda.synchronize()
        runs.append((gU.view.cpu().numpy().copy(), gW.view.cpu().numpy().copy() if angular else None))
    for g in (gpos, gF, gT, gU, gW):
        assert g is None or g.guards_intact()
    for U, W in runs[1:]:
        np.testing.assert_array_equal(U, runs[0][0])
        if angular:
            np.testing.assert_array_equal(W, runs[0][1])
    U = runs[0][0].reshape(nrhs, N, 3)
    W = runs[0][1].reshape(nrhs, N, 3) if angular else None
    q = nrhs - 1                                                  # the last right-hand side ends at the guard band
    if with_wall:
        Uo, Wo = wall.mdot(c["pos"], F[q], None if T is None else T[q], wall_z=c["wall_z"], angular=angular)
    else:
        Uo, Wo = rpy.mdot(c["pos"], F[q], None if T is None else T[q], angular=angular)
    assert rel(U[q], Uo) <= TOL[prec]
    if angular:
        assert rel(W[q], Wo) <= TOL[prec]
    s.close()


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f32", True)])
@pytest.mark.parametrize("N,graph,small", [(300, 1, 1), (300, 0, 1), (300, 1, 0), (9000, 0, 0)])
def test_lanczos_scratch_and_determinism(lm, torch, prec, angular, N, graph, small):
    """The Lanczos workspace (basis, w, packed vector, partials, Gram partials) after a NaN run; 6 repeats bit-identical."""
    c = workloads.random_case(N, 2.0 * N ** (1.0 / 3.0), 19, prec, angular, with_noise=True)
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    tdt = s.torch_dtype
    s.set_option(lm.LM_OPT_GRAPH_REPLAY, graph)
    s.set_option(lm.LM_OPT_SMALL_KERNEL, small)
    dof = (6 if angular else 3) * N
    gpos, gz = Guarded(torch, 3 * N, tdt, c["pos"]), Guarded(torch, dof, tdt, c["noise"])
    gy, gya = Guarded(torch, 3 * N, tdt), (Guarded(torch, 3 * N, tdt) if angular else None)
    s.set_max_iter(6)
    # NaN positions: the first apply writes NaN into the basis, w, the packed vector and the partials, and the call
    # must fail cleanly; NaN noise must be refused as well
    s.set_positions(torch.full_like(gpos.view, float("nan")))
    for noise in (gz.view, torch.full_like(gz.view, float("nan"))):
        with pytest.raises(lm.LmError) as e:
            s.sqrt_mdot_w(noise, 1e-3, gy.view, gya.view if angular else None)
        assert e.value.code == lm.LM_E_INVALID            # an input error, not a CUDA runtime error
    s.set_positions(gpos.view)
    runs = []
    for _ in range(6):
        it = s.sqrt_mdot_w(gz.view, 1e-30, gy.view, gya.view if angular else None, allow_noconv=True)
        torch.cuda.synchronize()
        runs.append(np.concatenate([gy.view.cpu().numpy()] + ([gya.view.cpu().numpy()] if angular else [])))
        assert it == 6
    for g in (gpos, gz, gy, gya):
        assert g is None or g.guards_intact()
    for r in runs[1:]:
        np.testing.assert_array_equal(r, runs[0])
    yo, ko, conv = rpy.lanczos_sqrt_mdot_w(c["pos"], c["noise"], 1e-30, angular=angular, max_iter=6)
    assert rel(runs[0], yo) <= (1e-10 if prec == "f64" else 3e-5)
    s.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("N", [257, 5000])
def test_steric_and_bd_step_guards(lm, torch, prec, N):
    c = workloads.random_case(N, 1.6 * N ** (1.0 / 3.0), 5, prec, False, with_noise=True)
    s = lm.Solver(prec, N)
    tdt = s.torch_dtype
    gpos, gext, gout, gz = Guarded(torch, 3 * N, tdt, c["pos"]), Guarded(torch, 3 * N, tdt, c["forces"]), Guarded(torch, 3 * N, tdt), Guarded(torch, 3 * N, tdt, c["noise"])
    s.set_positions(gpos.view)
    outs = []
    for _ in range(4):
        s.steric_forces(4.0, 0.1, gext.view, gout.view)
        torch.cuda.synchronize()
        outs.append(gout.view.cpu().numpy().copy())
    for o in outs[1:]:
        np.testing.assert_array_equal(o, outs[0])
    Fo = bd.steric_forces(c["pos"], 4.0, 0.1, 2.0) + c["forces"].astype(np.float64)
    assert rel(outs[0], Fo) <= (1e-11 if prec == "f64" else 2e-5)
    s.set_max_iter(300)
    s.bd_step(gpos.view, gext.view, None, gz.view, 1e-3, 1.0, 4.0, 0.1, 1e-3)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(gpos.view).all())
    for g in (gpos, gext, gout, gz):
        assert g.guards_intact()
    s.close()
