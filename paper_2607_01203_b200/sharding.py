"""Multi-GPU plumbing: every (trajectory, timestep) tile is independent in forward and VJP
(gradients are with respect to per-tile inputs), so ranks take contiguous slices of the batch and
there is NO collective on the data path; only the benchmark's timing / unit counts
are reduced across ranks."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(total: int, rank: int, world: int):
    """Contiguous [begin, end) slice of `total` units for `rank`; sizes differ by at most 1."""
    base, rem = divmod(total, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def _reduce(value: float, op, device=None) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(value: float, device=None) -> float:
    return _reduce(value, dist.ReduceOp.MAX, device)


def sum_over_ranks(value: float, device=None) -> float:
    return _reduce(value, dist.ReduceOp.SUM, device)
