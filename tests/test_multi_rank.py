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
