"""Beam sharding over ranks (beams are independent through dedispersion and search).

One process per GPU; rank r owns the global beams r*nbeam .. r*nbeam + nbeam - 1 (weak scaling: every rank brings its own
beams); there is no data-path collective.  The only exchange is the timing reduction (max over ranks) and, for a report,
the candidate counts -- scalars, outside the hot path.
"""
from __future__ import annotations

from typing import List


def beams_of_rank(rank: int, world: int, nbeam_per_rank: int) -> List[int]:
    """Global beam indices (= generator seeds offsets) of this rank's local beams 0..nbeam_per_rank-1."""
    if not (0 <= rank < world) or nbeam_per_rank < 1:
        raise ValueError("bad rank/world/nbeam")
    return [rank * nbeam_per_rank + b for b in range(nbeam_per_rank)]


def max_over_ranks(value: float, device=None) -> float:
    """Max of a host scalar over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: int, device=None) -> int:
    """Sum of a host integer over all ranks (candidate totals for the report)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return int(value)
    t = torch.tensor([int(value)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.item())
