"""GPU tests of the row-sharded apply.  Only ONE GPU is available to the
tests, so (i) the row-range kernel path is exercised rank by rank, one after the other, with lm_mdot_rows
(no kernel ever waits for another), each block against the oracle's rows; and (ii) the NCCL path runs with
a world of one rank: communicator, all-gather buffers, in-place all-gather and copy-out all execute, and
every entry point must give exactly what the undistributed handle gives.  Needs a B200 (``-m gpu``)."""
import os

import numpy as np
import pytest

from oracle import rpy
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


@pytest.mark.parametrize("prec,angular", [("f64", False), ("f64", True), ("f32", False), ("f32", True)])
@pytest.mark.parametrize("N,G", [(1000, 3), (37, 8), (5000, 2), (2049, 4)])
def test_row_blocks_one_rank_after_the_other(lm, torch, prec, angular, N, G):
    c = workloads.random_case(N, 2.2 * N ** (1 / 3), 61, prec, angular)
    s = lm.Solver(prec, N, 1.0, 1.0, angular)
    s.set_positions(dev(torch, c["pos"]))
    F, T = dev(torch, c["forces"]), dev(torch, c["torques"])
    sentinel = -12345.0
    U = torch.full((3 * N,), sentinel, dtype=s.torch_dtype, device="cuda")
    W = torch.full((3 * N,), sentinel, dtype=s.torch_dtype, device="cuda") if angular else None
    Uo, Wo = rpy.mdot(c["pos"], c["forces"], c["torques"], angular=angular)
    for r in range(G):
        b, e = lm.lm_dist_row_block(N, G, r)
        s.mdot_rows(b, e - b, F, T, U, W)
        torch.cuda.synchronize()
        got = U.cpu().numpy().reshape(N, 3)
        if e > b:
            assert rel(got[b:e], Uo[b:e]) <= TOL[prec] * 4        # a block's norm is smaller than the whole's
        assert np.all(got[e:] == sentinel)                         # rows of later ranks: untouched
        if angular and e > b:
            assert rel(W.cpu().numpy().reshape(N, 3)[b:e], Wo[b:e]) <= TOL[prec] * 4
    assert rel(U.cpu().numpy(), Uo) <= TOL[prec]                   # the union is the full product
    U2 = torch.empty_like(U)
    s.mdot(F, T, U2, torch.empty_like(U) if angular else None)     # the handle is back to all rows
    torch.cuda.synchronize()
    assert rel(U2.cpu().numpy(), Uo) <= TOL[prec]
    with pytest.raises(lm.LmError) as ei:
        s.mdot_rows(N - 1, 2, F, T, U, W)
    assert ei.value.code == lm.LM_E_INVALID
    s.close()


def test_nccl_world_of_one_equals_the_undistributed_handle(lm, torch):
    import torch.distributed as dist
    from paper_2510_02135_b200 import multi
    port = 33500 + os.getpid() % 2000
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        for prec, angular, in_place, acc64 in (("f32", False, 1, 0), ("f64", True, 1, 0), ("f32", True, 0, 0), ("f64", False, 0, 0), ("f32", False, 1, 1)):
            N = 3000
            c = workloads.random_case(N, 30.0, 62, prec, angular, with_noise=True)
            ref, sh = lm.Solver(prec, N, 1.0, 1.0, angular), lm.Solver(prec, N, 1.0, 1.0, angular)
            # a sharded handle always takes the general path (its outputs go through the all-gather buffers); the
            # reference is held to the same kernels so that the comparison can be bit for bit
            ref.set_option(lm.LM_OPT_SMALL_KERNEL, 0)
            for s_ in (ref, sh):
                s_.set_option(lm.LM_OPT_ACCUMULATE_F64, acc64)           # mixed precision: fp64 partials through the same all-gather path
            sh.set_option(lm.LM_OPT_GATHER_IN_PLACE, in_place)   # all-gather into the caller's arrays / through the handle's buffers
            assert multi.init_sharded(sh) == (0, N)
            with pytest.raises(lm.LmError):
                sh.dist_init(1, 0, lm.lm_dist_unique_id())        # only once per handle
            outs = []
            for s in (ref, sh):
                s.set_positions(dev(torch, c["pos"]))
                mk = lambda n=1: torch.empty(n * 3 * N, dtype=s.torch_dtype, device="cuda")
                U, W = mk(), (mk() if angular else None)
                s.mdot(dev(torch, c["forces"]), dev(torch, c["torques"]), U, W)
                nb = 2
                Fb = torch.cat([dev(torch, c["forces"]).reshape(-1)] * nb)
                Tb = torch.cat([dev(torch, c["torques"]).reshape(-1)] * nb) if angular else None
                Ub, Wb = mk(nb), (mk(nb) if angular else None)
                s.mdot_batch(nb, Fb, Tb, Ub, Wb)
                y, ya = mk(), (mk() if angular else None)
                it = s.sqrt_mdot_w(dev(torch, c["noise"]), 1e-3, y, ya)
                X = dev(torch, c["pos"]).reshape(-1).clone()
                s.bd_step(X, dev(torch, c["forces"]).reshape(-1), None, dev(torch, c["noise"]), 1e-3, 1.0, 4.0, 0.1, 1e-3)
                torch.cuda.synchronize()
                outs.append([t.cpu().numpy() for t in (U, Ub, y, X)] + [it])
            for a, b in zip(outs[0][:-1], outs[1][:-1]):
                np.testing.assert_array_equal(a, b)               # same kernels, same grid: bit-identical
            assert outs[0][-1] == outs[1][-1]
            Uo, _ = rpy.mdot(c["pos"], c["forces"], c["torques"], angular=angular)
            assert rel(outs[1][0], Uo) <= TOL[prec]
            ref.close()
            sh.close()
    finally:
        dist.destroy_process_group()
