"""Host-side logic of the multi-GPU path: the hot path shards BY CCD (PAPER.md:324 -- "each GPU
processes a queue of approximately ~30 CCD images sequentially"), with no data-path collective.
The only exchanges are a barrier and a max-over-ranks of the device time."""
from __future__ import annotations

from typing import List


def shard_ccds(n_ccd: int, rank: int, world: int) -> List[int]:
    """Static round-robin partition of CCD indices 0..n_ccd-1 over `world` ranks."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return list(range(rank, n_ccd, world))


def max_over_ranks(ms: float, device=None) -> float:
    """MAX all-reduce of a per-rank device time (no-op without an initialised process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, world: int, ms: float) -> float:
    """Whole-job units/s when every rank processed `units_per_rank` units in `ms` (max over ranks)."""
    return world * units_per_rank / (ms * 1e-3)
