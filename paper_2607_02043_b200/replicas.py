"""Replica bookkeeping for N > 1 (the path shards by request with no data-path collective, so
`bench.py --gpus N` runs N independent replicas).  Only timing scalars cross ranks."""
from __future__ import annotations

import torch
import torch.distributed as dist


def replica_seed_shift(rank: int) -> int:
    """Rank r draws its batch from seed + r: same shapes, independent data."""
    return int(rank)


def max_over_ranks(value: float, device: torch.device | str = "cpu") -> float:
    """Max of a per-rank scalar (time is reported as the slowest rank's)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_us_per_step(local_ms: float, steps: int, world: int, device: torch.device | str = "cpu") -> float:
    """µs per mixed step of the whole job: every iteration advances `world` replicas by one step each, and the
    iteration takes as long as the slowest rank."""
    return max_over_ranks(local_ms, device) * 1e3 / (steps * world)
