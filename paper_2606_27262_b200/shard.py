"""Beam sharding over ranks (beams are independent through dedispersion and search).

One process per GPU; rank r owns the global beams r*nbeam .. r*nbeam + nbeam - 1 (weak scaling: every rank brings its own
beams); there is no data-path collective.  The only exchange is the timing reduction (max over ranks) and, for a report,
the candidate counts -- scalars, outside the hot path -- and, when one list of the whole job is wanted, the merge of the
ranks' candidate lists on rank 0 (variable length: counts first, then one padded gather).
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


def merge_candidates(local, rank: int, world: int, nbeam_per_rank: int, device=None):
    """The whole job's candidate list on rank 0 (None elsewhere): every rank's records (numpy structured array as
    api.Plan.candidates_read returns it: beam, trial, t, width, snr) with the beam field renumbered from local to global
    (beams_of_rank), concatenated in rank order.  SURVEY.md 8(e): the only exchange after the search; not on the hot path."""
    import numpy as np
    import torch
    import torch.distributed as dist
    rec = np.array(local, copy=True)
    if rec.size:
        rec["beam"] += rank * nbeam_per_rank
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return rec
    nbytes = rec.dtype.itemsize
    counts = torch.zeros(world, dtype=torch.int64, device=device)
    counts[rank] = rec.size
    dist.all_reduce(counts, op=dist.ReduceOp.SUM)
    nmax = int(counts.max().item())
    buf = torch.zeros(max(1, nmax) * nbytes, dtype=torch.uint8, device=device)
    if rec.size:
        buf[: rec.size * nbytes] = torch.from_numpy(rec.view(np.uint8).reshape(-1).copy()).to(buf.device)
    gathered = [torch.empty_like(buf) for _ in range(world)] if rank == 0 else None
    dist.gather(buf, gathered, dst=0)
    if rank != 0:
        return None
    parts = [gathered[r][: int(counts[r].item()) * nbytes].cpu().numpy().view(rec.dtype) for r in range(world)]
    return np.concatenate(parts)
