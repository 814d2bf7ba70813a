"""Host-side multi-GPU plumbing: walkers shard across ranks with no data-path collective
(the local-energy evaluations are independent).  The only exchanges are the
max-over-ranks of the device timings and, for a global energy estimate, the 3-number
reduction (sum E, sum E^2, count) of eq. 3."""
from __future__ import annotations

import math

import torch
import torch.distributed as dist


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous walker range [w0, w1) of `rank`; sizes differ by at most one."""
    base, rem = divmod(n_total, world)
    w0 = rank * base + min(rank, rem)
    return w0, w0 + base + (1 if rank < rem else 0)


def max_over_ranks(values, device="cpu"):
    """Element-wise max of a list of floats over all ranks (timings: the slowest rank counts)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def global_energy(sum_e: float, sum_e2: float, count: int, device="cpu"):
    """Mean and standard error of E_L over all ranks from per-rank (sum, sum of squares, count)."""
    t = torch.tensor([sum_e, sum_e2, float(count)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    s, s2, n = (float(x) for x in t.cpu())
    mean = s / n
    var = max(s2 / n - mean * mean, 0.0) * n / max(n - 1.0, 1.0)
    return mean, math.sqrt(var / n)
