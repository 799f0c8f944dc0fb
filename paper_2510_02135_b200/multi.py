"""Multi-GPU plumbing: "replicas only".

The path does not shard in this build (north_star: one GPU, no collectives): N ranks run N
independent replicas of the workload.  The only cross-rank traffic is the timing aggregation
below, on whatever backend the process group uses (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

REPLICA_SEED_STRIDE = 1000


def replica_seed(seed: int, rank: int) -> int:
    """Seed of rank `rank`'s replica: rank 0 keeps the config's own seed."""
    return int(seed) + REPLICA_SEED_STRIDE * int(rank)


def aggregate_over_ranks(ms: float, units: float, device=None):
    """(max over ranks of the device time `ms`, sum over ranks of the processed `units`).

    Without an initialised process group (single process) returns the inputs unchanged."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(units)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
