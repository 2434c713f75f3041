"""Host-side logic of the N>1 path: the apply shards by vector columns with no data-path collective
(Eq. 16: columns are independent).  Only the timing is reduced over ranks."""
from __future__ import annotations

from typing import Tuple


def column_block(rank: int, world: int, nvec_per_rank: int) -> Tuple[int, int]:
    """Weak scaling: rank r owns global columns [r*nvec_per_rank, (r+1)*nvec_per_rank)."""
    if not (0 <= rank < world) or nvec_per_rank < 1:
        raise ValueError("bad rank/world/nvec")
    return rank * nvec_per_rank, (rank + 1) * nvec_per_rank


def split_columns(nvec_total: int, world: int, rank: int) -> Tuple[int, int]:
    """Strong scaling helper: contiguous, balanced column ranges covering [0, nvec_total)."""
    base, rem = divmod(nvec_total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def generator_offset(rank: int, ndof: int, nvec_per_rank: int) -> int:
    """Counter offset so that every rank fills a distinct, reproducible block of the input stream."""
    return rank * ndof * nvec_per_rank


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a per-rank time (the contract's 'max over ranks')."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    return units_per_rank * world / seconds_max
