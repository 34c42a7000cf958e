"""Batch sharding across ranks: samples are independent, so a multi-GPU
run gives every rank its own slice of the batch and its own KV pool; the only exchange is the merge
of the per-rank outputs of fv_free_energy (count, mean, sum of squared deviations of L = E + T log q,
Eq. 5) into the whole batch's F_q and its spread.  Nothing here evaluates the method:
the per-sample values are reduced by the library's kernel on each rank."""
from __future__ import annotations

import math

import torch
import torch.distributed as dist


def shard_bounds(total: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of `total` samples for `rank` (sizes differ by <= 1)."""
    base, rem = divmod(total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def merge_free_energy(stats: torch.Tensor) -> tuple[float, float]:
    """`stats` = this rank's (mean, std, count, M2) as fv_free_energy returns them (fp64, any device).
    All-gather over the default process group (if any) and combine the ranks in rank order with the
    pairwise update of Chan et al. -> (mean, population std) of the whole batch."""
    mine = stats.detach().to(torch.float64).reshape(4)
    parts = [mine]
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        parts = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
        dist.all_gather(parts, mine)
    n, mean, m2 = 0.0, 0.0, 0.0
    for p in parts:
        mean_b, _, n_b, m2_b = (float(x) for x in p.tolist())
        if n_b == 0.0:
            continue
        delta = mean_b - mean
        tot = n + n_b
        mean += delta * n_b / tot
        m2 += m2_b + delta * delta * n * n_b / tot
        n = tot
    return mean, math.sqrt(max(m2 / n, 0.0))


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing rule of bench.py: a multi-rank time is the max over ranks."""
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
