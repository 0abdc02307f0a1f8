"""Multi-GPU plumbing: how the path shards.

Rows (b,d) of ``selective_scan_fwd`` and sequences of ``affine_scan`` never interact, so
the path shards over independent units with NO data-path collective: each rank takes a
contiguous slice of the batch (B, C are then not replicated) and runs the single-GPU
library on it.  The only cross-rank step is the timing reduction (max over ranks) in
bench.py.  Nothing here touches the arithmetic.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) slice of ``n_units`` for ``rank`` (first ranks get +1)."""
    if world <= 0 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (device time in ms) over all ranks; identity if not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
