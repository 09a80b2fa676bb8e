"""Multi-GPU plumbing: the path shards by independent units -- camera poses or whole frames -- with
every rank holding the full scene; the data path needs no collective.  torch.distributed is used only to launch one
process per GPU, to barrier around timed regions and to take the max of device timings over ranks."""
from __future__ import annotations

from typing import List, Sequence

import torch
import torch.distributed as dist


def shard_units(n_units: int, rank: int, world: int) -> List[int]:
    """Units (poses / frames) rank `rank` renders: round-robin, every unit exactly once over the ranks."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world")
    return list(range(rank, n_units, world))


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank device timing (ms); identity when not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_per_rank: Sequence[int], ms_max: float) -> float:
    """Whole-job units per second from the units every rank processed and the max-over-ranks time."""
    return sum(units_per_rank) / (ms_max * 1e-3)
