"""Multi-GPU plumbing: replicas only.

The path of this build does not shard (north_star: "everything runs on one GPU"; the paper never
shards), so N GPUs run N independent replicas of the same workload -- the
analogue of the paper's vmap over PRNG keys -- with no collective on the data
path.  The only exchanges are the barrier and the max-over-ranks of the measured time that
bench.py needs; they go through torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> tuple[int, int]:
    """(rank, world_size); (0, 1) when torch.distributed is not initialised."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def replica_index(rank: int) -> int:
    """Rank r simulates replica r: an independent sample (seed + 1000 r) of the same config."""
    return int(rank)


def max_over_ranks(value: float, device=None) -> float:
    """Max of a host scalar over all ranks (the slowest rank's time is the job's time)."""
    _, n = world()
    if n == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def whole_job_rate(units_per_rank: float, seconds_max: float) -> float:
    """Aggregate throughput of a weak-scaling replica job: every rank processed
    `units_per_rank` units in at most `seconds_max`."""
    _, n = world()
    return n * units_per_rank / seconds_max
