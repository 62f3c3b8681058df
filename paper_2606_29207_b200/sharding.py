"""Multi-GPU plumbing of the benchmark: the path shards over independent requests.

One process per GPU; rank k runs an independent batch of the same recipe (seed + k), so there is NO data-path
collective: `torch.distributed` carries only the barrier and the reduction of the per-rank measurements below
(NCCL on GPUs, gloo in the CPU tests).  Nothing here touches the method's arithmetic.
"""
from __future__ import annotations

from typing import Optional, Tuple


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s batch: independent requests per rank (weak scaling)."""
    return base_seed + rank


def aggregate(ms: float, n_bytes: float, launches: int, dist=None, device=None) -> Tuple[float, float, int]:
    """Whole-job numbers from per-rank ones: time = MAX over ranks (every rank timed the same K steps on its own
    device clock), bytes and kernel launches = SUM over ranks.  `dist` is torch.distributed (initialised) or None."""
    if dist is None:
        return float(ms), float(n_bytes), int(launches)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tb = torch.tensor([float(n_bytes), float(launches)], dtype=torch.float64, device=device)
    dist.all_reduce(tb, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tb[0].item()), int(round(tb[1].item()))


def throughput_gbs(total_bytes: float, ms: float) -> float:
    """Whole-job GB/s = bytes all ranks processed / the slowest rank's time."""
    return total_bytes / (ms * 1e-3) / 1e9
