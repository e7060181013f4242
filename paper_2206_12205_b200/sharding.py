"""Host-side sharding for N > 1 GPUs.

The path has no exchange step: every (series, segment, template) triple is independent, so
ranks take disjoint sets of series and never communicate on the data path.  torch.distributed
is used for exactly two things: a barrier around the timed region and the max-over-ranks of
the elapsed time (and, for a survey, gathering the per-series peak counts)."""
from __future__ import annotations

from typing import List


def series_for_rank(n_series: int, rank: int, world: int) -> List[int]:
    """Cyclic partition of series indices 0..n_series-1: rank r takes r, r+world, ...
    (cyclic keeps the 10 % signal-carrying series of config 4 spread evenly)."""
    if not (0 <= rank < world) or n_series < 0:
        raise ValueError("bad rank/world/n_series")
    return list(range(rank, n_series, world))


def sub_batches(indices: List[int], max_resident: int) -> List[List[int]]:
    """Split a rank's series into sub-batches whose planes fit in HBM together
    (config 4: 256 x 97 x 2^21 x 4 B = 208 GB does not fit at once)."""
    if max_resident < 1:
        raise ValueError("max_resident must be >= 1")
    return [indices[i:i + max_resident] for i in range(0, len(indices), max_resident)]


def max_resident_series(K: int, M: int, plane_elem_bytes: int, hbm_bytes: int, reserve: float = 0.15) -> int:
    """How many [K][M] planes fit in `hbm_bytes` leaving `reserve` of it free."""
    per = K * M * plane_elem_bytes + M * 16
    return max(1, int(hbm_bytes * (1.0 - reserve)) // per)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a host float (elapsed time); identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
