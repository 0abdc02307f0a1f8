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


# ----------------------------------------------------------------------------- L-sharding
def shard_range_aligned(n_units: int, rank: int, world: int, align: int):
    """Like shard_range, but every boundary is a multiple of ``align`` (the 128-bit vector width
    along L), so each slice keeps the vector-load kernels; the last rank takes the ragged tail."""
    blocks = -(-n_units // align)
    lo, hi = shard_range(blocks, rank, world)
    return min(lo * align, n_units), min(hi * align, n_units)


def selective_scan_fwd_l_sharded(x, delta, A, B, C, D, h0, y, h_last, group=None, ops=None):
    """The multi-GPU L-sharded forward selective scan.

    Every rank holds the L-slice [t_r, t_{r+1}) of x, delta, B, C (and writes the same slice of y);
    A, D, h0 are replicated.  The path has ONE exchange step, a NCCL all-gather of the slices'
    transition pairs (rows*N*2 floats per rank):
        1. (P_r, U_r) = selective_scan_slice_aggregate(slice)             [kernels]
        2. all_gather over the ranks                                       [NCCL]
        3. h_in = (P_{r-1},U_{r-1}) (+) ... (+) (P_0,U_0) applied to h0    [kernel]
        4. selective_scan_fwd(slice, h0 = h_in) -> y slice, state after the slice
    Rank 0 needs no carry (its h_in is h0) and nobody consumes the last rank's aggregate, so rank 0
    skips step 3 and the last rank skips step 1 (it contributes zeros to the all-gather): with R
    ranks the extra scan costs R-1 of R slices, and a single rank runs the plain forward only.
    The last rank's state is the global h_last; it is broadcast so every rank returns it.

    ``delta`` is the step size that enters the recurrence, i.e. AFTER any softplus / bias: the
    prologue, gate and resets of selective_scan_fwd_ext are not threaded through the slice
    aggregate, so the extended forward cannot be L-sharded with this driver.
    Unmeasured on more than one GPU: parity is proven with ranks emulated on one B200 and with
    gloo on CPU; no NCCL timing exists.

    ``ops`` injects the three compute steps (tests on CPU pass the oracle); by default they are
    the library's CUDA entry points.  Only plumbing happens here.
    """
    if ops is None:
        from . import binding as ops
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    batch, d_inner, _ = x.shape
    N = A.shape[1]
    f32 = dict(dtype=torch.float32, device=x.device)
    h_in = h0
    if world > 1:
        PU = torch.zeros((2, batch, d_inner, N), **f32)       # one message per rank
        if rank < world - 1:
            ops.selective_scan_slice_aggregate(x, delta, A, B, C, PU[0], PU[1])
        gathered = [torch.empty_like(PU) for _ in range(world)]
        dist.all_gather(gathered, PU, group=group)
        if rank > 0:
            # ranks 0..rank (the fold reads ranks < rank only; the C call wants rank < rows)
            PU_all = torch.stack(gathered[:rank + 1])         # [rank+1, 2, batch, d_inner, N]
            h_in = torch.empty((batch, d_inner, N), **f32)
            ops.compose_carry(PU_all[:, 0].contiguous(), PU_all[:, 1].contiguous(), h0, h_in, rank)
    state = torch.empty((batch, d_inner, N), **f32)
    ops.selective_scan_fwd(x, delta, A, B, C, D, h_in, y, state)
    if world > 1:
        dist.broadcast(state, src=dist.get_global_rank(group, world - 1) if group else world - 1,
                       group=group)
    if h_last is not None:
        h_last.copy_(state)
    return y, h_last
