"""Multi-GPU plumbing of the hot path: one process per GPU, no data-path collective.

A single fit does not shard in this build ("replicas only"); the batched / survey mode shards as independent
problems.  This module holds the host logic both cases need -- which problems a rank owns, the per-rank seed of
a replica, and the max-over-ranks reduction of a device-measured time -- so that it can be covered with
world_size-2 `gloo` tests on a CPU box.  It contains none of the method's arithmetic.
"""
from __future__ import annotations

from typing import List

import torch
import torch.distributed as dist


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s independent replica of a workload (rank 0 keeps the config's own seed)."""
    return base_seed + 7919 * rank


def shard_problems(n_problems: int, rank: int, world: int) -> List[int]:
    """Contiguous block partition of `n_problems` independent problems over `world` ranks;
    the first n_problems % world ranks get one more.  Every problem is owned by exactly one rank."""
    if world < 1 or not (0 <= rank < world) or n_problems < 0:
        raise ValueError("bad shard request")
    per, extra = divmod(n_problems, world)
    lo = rank * per + min(rank, extra)
    return list(range(lo, lo + per + (1 if rank < extra else 0)))


def max_over_ranks(value: float, device: torch.device | str = "cpu") -> float:
    """MAX all-reduce of a per-rank scalar (a device-measured time); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: float, seconds_this_rank: float, device: torch.device | str = "cpu") -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's time (weak scaling)."""
    world = dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1
    return world * units_per_rank / max_over_ranks(seconds_this_rank, device)
