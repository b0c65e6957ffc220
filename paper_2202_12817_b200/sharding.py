"""Multi-GPU shape of the path: spectra (DM trials) are independent
("scaling in the number of power spectra is linear"), so the batch dimension is
split across ranks, each rank owns a plan for its rows, and there is NO data-path collective.
Only timing (max over ranks) and the tiny candidate lists cross ranks."""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist


def shard_rows(n_spectra: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [lo, hi) rows of rank `rank`; sizes differ by at most one row."""
    base, rem = divmod(n_spectra, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing convention of bench.py: the slowest rank defines the step time."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_candidates(local: torch.Tensor, row_offset: int) -> List[Tuple[int, int, int]]:
    """local: int64 [k, 3] rows (local spectrum, bin, best_h) on the CPU.  Returns the global list,
    sorted, identical on every rank (a small all_gather of variable-length lists)."""
    loc = local.clone()
    if loc.numel():
        loc[:, 0] += row_offset
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        parts = [loc]
    else:
        objs = [None] * dist.get_world_size()
        dist.all_gather_object(objs, loc)
        parts = objs
    allc = torch.cat([p.reshape(-1, 3) for p in parts], dim=0)
    return sorted((int(a), int(b), int(c)) for a, b, c in allc.tolist())
