"""Batch sharding across ranks: samples are independent, so a multi-GPU
run gives every rank its own slice of the batch and its own KV pool; the only exchange is the
reduction of three scalars for F_q = <E + T log q> (Eq. 5) and its spread."""
from __future__ import annotations

import math

import torch
import torch.distributed as dist


def shard_bounds(total: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of `total` samples for `rank` (sizes differ by <= 1)."""
    base, rem = divmod(total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def local_moments(E: torch.Tensor, logq: torch.Tensor, temperature: float) -> torch.Tensor:
    """(sum L, sum L^2, count) of L = E + T log q over this rank's samples, fp64."""
    L = E.double() + temperature * logq.double()
    return torch.stack([L.sum(), (L * L).sum(), torch.tensor(float(L.numel()), dtype=torch.float64, device=L.device)])


def merge_free_energy(moments: torch.Tensor) -> tuple[float, float]:
    """All-reduce the three moments over the default process group (if any) -> (mean, population std)."""
    m = moments.clone()
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(m, op=dist.ReduceOp.SUM)
    s, s2, n = (float(x) for x in m.tolist())
    mean = s / n
    return mean, math.sqrt(max(s2 / n - mean * mean, 0.0))


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing rule of bench.py: a multi-rank time is the max over ranks."""
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
