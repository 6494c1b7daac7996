"""Multi-GPU use of the path: independent replicas.

The solve of one network runs on one GPU (BASELINE.json north_star).  With N GPUs every rank solves its OWN
network -- another realisation of the same recipe -- and no data-path collective exists.  What the ranks do
share is host-side bookkeeping only: which realisation a rank takes, and the aggregation of timings and
counts for the one JSON line rank 0 prints.  These helpers hold that logic so that it can be tested on CPU
with the gloo backend (tests/test_replicas.py); bench.py uses them with NCCL.
"""
from __future__ import annotations

import os


def env_rank_world() -> tuple:
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the realisation rank `rank` solves: rank 0 takes the config's own seed."""
    return int(base_seed) + int(rank)


def assign(n_problems: int, rank: int, world: int) -> list:
    """Indices of the problems rank `rank` owns when `n_problems` independent solves (realisations,
    or the x / z directions of CFG5) are dealt round-robin to `world` ranks."""
    return list(range(int(rank), int(n_problems), int(world)))


def reduce_max(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the timed region: the job is as slow as its slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value: float, device=None) -> float:
    """SUM over ranks of a per-rank count (iterations, node updates, launches): whole-job aggregates."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_list(value, device=None) -> list:
    """Every rank's python object, in rank order, on every rank (small host-side records only)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [value]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, value)
    return out
