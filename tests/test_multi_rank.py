"""N>1 path ("replicas only") on CPU: world_size-2 gloo process group."""
import os
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2510_02135_b200 import multi, workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each rank: its own replica of config 1 at reduced N, its own (fake) device time
    cfg = workloads.CONFIGS[1]
    data = workloads.generate(1, N=64, seed=multi.replica_seed(cfg.seed, rank))
    ms, pairs = 10.0 + 5.0 * rank, float(data["N"]) ** 2
    ms_max, pairs_sum = multi.aggregate_over_ranks(ms, pairs)
    dist.barrier()
    out.put((rank, ms_max, pairs_sum, float(data["pos"][0, 0])))
    dist.destroy_process_group()


def test_replicas_aggregate_max_time_and_sum_units():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ms_max, pairs_sum, _ in res:
        assert ms_max == 15.0 and pairs_sum == 2 * 64.0 ** 2
    assert res[0][3] != res[1][3]          # replicas draw different inputs


def test_single_process_passthrough_and_seeds():
    sys.path.insert(0, ROOT)
    from paper_2510_02135_b200 import multi
    assert multi.aggregate_over_ranks(3.5, 7.0) == (3.5, 7.0)
    assert multi.replica_seed(2, 0) == 2 and multi.replica_seed(2, 3) == 3002


# ---------------------------------------------------------------- row-sharded applies: host logic (no GPU)
def test_row_blocks_tile_the_rows():
    sys.path.insert(0, ROOT)
    import paper_2510_02135_b200 as lm
    for N in (1, 2, 7, 64, 1000, 1024, 131072, 1048576 + 3):
        for G in (1, 2, 3, 4, 8, 16):
            B = -(-N // G)
            prev_end = 0
            for r in range(G):
                b, e = lm.lm_dist_row_block(N, G, r)
                assert b == prev_end and b <= e <= N and e - b <= B     # contiguous, in order, at most B rows
                assert b == min(N, r * B)                                # rank r's all-gather segment starts at 3 B r
                prev_end = e
            assert prev_end == N                                         # every row exactly once
    with pytest.raises(lm.LmError):
        lm.lm_dist_row_block(10, 2, 2)
    with pytest.raises(lm.LmError):
        lm.lm_dist_row_block(0, 2, 0)


def _block_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import paper_2510_02135_b200 as lm
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N = 1001
    b, e = lm.lm_dist_row_block(N, world, rank)
    mine = torch.tensor([b, e], dtype=torch.int64)
    allb = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allb, mine)
    # what the library's in-place all-gather does, on the host: rank r fills rows [b, e) of a 3 B G buffer
    B = -(-N // world)
    seg = torch.full((3 * B,), -1.0, dtype=torch.float64)
    seg[: 3 * (e - b)] = torch.arange(3 * b, 3 * e, dtype=torch.float64)
    parts = [torch.zeros(3 * B, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(parts, seg)
    full = torch.cat(parts)[: 3 * N]
    out.put((rank, [t.tolist() for t in allb], bool(torch.equal(full, torch.arange(3 * N, dtype=torch.float64)))))
    dist.destroy_process_group()


def test_row_blocks_across_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_block_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, blocks, ok in res:
        assert blocks == [[0, 501], [501, 1001]] and ok


def _stop_worker(rank, world, port, out):
    """Both ranks replay the host side of a row-sharded Lanczos run (csrc/lanczos_host.h through tests/hooks): the
    stopping test on their own copies of alpha_k, beta_k and the Gram columns, then agree_on_stops with a gloo
    broadcast from rank 0 as the transport.  Rank 1's scalars are deliberately perturbed, so its own verdict comes
    at another step; every iteration ends with a collective (the stand-in for the next apply's all-gather), which
    would hang if the ranks disagreed on whether there IS a next iteration."""
    sys.path.insert(0, ROOT)
    import ctypes
    import numpy as np
    import torch
    import torch.distributed as dist
    from oracle import rpy
    from tests import hooks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L = hooks.lib()
    dp = ctypes.POINTER(ctypes.c_double)
    rng = np.random.default_rng(11)
    N, tol = 150, 1e-3
    pos = rng.random((N, 3)) * 9.0
    M = rpy.dense(pos)
    z = rng.standard_normal(3 * N)
    wobble = np.random.default_rng(5)                       # rank 1 sees slightly different scalars
    V = [z / np.linalg.norm(z)]
    st = L.hook_stopper_new(0, tol, 1e-14, 100)
    col = lambda m: np.ascontiguousarray([V[j] @ V[m] for j in range(m + 1)])
    L.hook_stopper_gram_column(st, 0, col(0).ctypes.data_as(dp))

    def exchange(words):                                    # the protocol of lanczos_host.h agree_on_stops
        t = torch.tensor([int(words[0])], dtype=torch.int64)
        dist.broadcast(t, src=0)                            # rank 0's stop bits
        f = torch.tensor([int(words[1])], dtype=torch.int64)
        dist.all_reduce(f, op=dist.ReduceOp.MAX)            # anybody's failure flag
        words[0], words[1] = int(t.item()), int(f.item())

    cb = hooks.EXCHANGE_FN(exchange)
    beta_prev, k_local, k_agreed = 0.0, None, None
    for k in range(1, 101):
        w = M @ V[k - 1] - (beta_prev * V[k - 2] if k > 1 else 0.0)
        alpha = w @ V[k - 1]
        w = w - alpha * V[k - 1]
        beta = np.linalg.norm(w)
        V.append(w / beta)
        eps = 0.0 if rank == 0 else 3e-2 * wobble.standard_normal()
        verdict = L.hook_stopper_feed(st, k, float(alpha * (1 + eps)), float(beta * (1 - eps)))
        if verdict == 1 and k_local is None:
            k_local = k
        word = L.hook_agree_on_stops(1 if verdict == 1 else 0, cb, 1)
        if word & 1:
            k_agreed = k
            break
        L.hook_stopper_advance(st)
        L.hook_stopper_gram_column(st, k, col(k).ctypes.data_as(dp))
        beta_prev = beta
        dist.all_reduce(torch.zeros(1))                     # the next iteration's collective: both ranks must post it
    L.hook_stopper_free(st)
    out.put((rank, k_local, k_agreed))
    dist.destroy_process_group()


def test_lanczos_stop_is_rank_zeros_verdict_even_when_the_ranks_scalars_differ():
    """VERDICT r1 item 6 / ADVICE: ranks must not part ways on the stopping decision (a rank that goes on posts an
    all-gather the others never match).  Two gloo ranks, rank 1 with perturbed scalars: both leave the loop at rank
    0's step, although rank 1's own test says otherwise."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 35500 + os.getpid() % 2000
    procs = [ctx.Process(target=_stop_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict((r, (kl, ka)) for r, kl, ka in (out.get(timeout=180) for _ in procs))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert res[0][0] == res[0][1] == res[1][1]              # rank 0's verdict is everybody's
    assert res[1][0] != res[0][0]                           # ... and rank 1's own verdict really was another one


def _fail_worker(rank, world, port, out):
    """Iteration 1: nobody stops, nobody fails.  Iteration 2: rank 1 (NOT rank 0) reports a failure (bit 31) while rank 0 wants to
    go on.  Every rank must come out of agree_on_stops with bit 31 set -- otherwise rank 0 would post the next all-gather
    and wait for ever for rank 1, which has returned."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from tests import hooks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L = hooks.lib()

    def exchange(words):
        t = torch.tensor([int(words[0])], dtype=torch.int64)
        dist.broadcast(t, src=0)
        f = torch.tensor([int(words[1])], dtype=torch.int64)
        dist.all_reduce(f, op=dist.ReduceOp.MAX)
        words[0], words[1] = int(t.item()), int(f.item())

    cb = hooks.EXCHANGE_FN(exchange)
    seen = []
    local_words = [[0x0, 0x0], [0x2, 0x80000001]]           # [iteration][rank]: rank 0 stops vector 1 in iteration 2, rank 1 fails
    for it in range(2):
        word = L.hook_agree_on_stops(local_words[it][rank], cb, 1)
        seen.append(int(word))
        if word & 0x80000000:
            break
        dist.all_reduce(torch.zeros(1))                     # the next apply's collective
    out.put((rank, seen))
    dist.destroy_process_group()


def test_a_failure_on_a_rank_other_than_zero_stops_every_rank():
    """only rank 0's word used to be broadcast, so a failure seen on another rank made that rank return while the
    others enqueued the next collective (deadlock).  The failure flag is now max-reduced over the ranks; the stop bits
    stay rank 0's."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 37500 + os.getpid() % 2000
    procs = [ctx.Process(target=_fail_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    # iteration 1: rank 0's stop bits (none) everywhere; iteration 2: rank 0's stop bits (0x2) + the failure flag, on BOTH ranks
    assert res[0] == res[1] == [0x0, 0x80000002]

