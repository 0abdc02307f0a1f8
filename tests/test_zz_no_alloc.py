"""affine_scan_static_scratch: the look-back scan for callers that cannot allocate device memory.

Some users of this library are not free to let it call cudaMalloc: a serving process that sized
its own cache to all the HBM that was left, a framework whose allocator has to account for every
byte, a real-time loop that must stay clear of the driver's allocation lock.  For them the
library offers one entry point whose tile descriptors live in a fixed 1 MiB array inside the
library image instead of cudaMallocAsync scratch.  These tests check that it computes what the
ordinary look-back path computes — on two calls in a row, because the array is shared by every
call and keeps the previous call's contents — and that it refuses problems beyond the array.

This file is named so that pytest collects it last: with `pytest -x` a failure here cannot hide
any other test.  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import pytest
import torch

import paper_2606_00601_b200 as lib
from workloads import normal, uniform

from util import TOL, assert_close, oracle_affine, rel_err


def _inputs(S, L, dtype, dev, seed, with_h0=True):
    a = uniform((S, L), 0.9, 0.9999, seed=seed, stream=0, device=dev, dtype=dtype)
    u = normal((S, L), seed=seed, stream=1, device=dev, dtype=dtype)
    h0 = normal((S,), seed=seed, stream=2, device=dev, dtype=torch.float32) if with_h0 else None
    return {"a": a, "u": u, "h0": h0}


def _outputs(inp):
    a = inp["a"]
    return (torch.full_like(a, float("nan")),
            torch.full((a.shape[0],), float("nan"), dtype=torch.float32, device=a.device))


def _run(fn, inp, out=None):
    h, h_last = out if out is not None else _outputs(inp)
    fn(inp["a"], inp["u"], inp.get("h0"), h, h_last)
    return h, h_last


def _existing(a, u, h0, h, h_last):
    lib.affine_scan_ex(a, u, h0, h, h_last, lib.AFFINE_LOOKBACK)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row(cuda_device, dtype):
    """Two back-to-back calls with DIFFERENT data and tile counts, nothing in between: the second
    call finds the first one's descriptors in the shared array and must not be fooled by them
    (a long slow-decay sequence first, so that its carries are large and non-zero everywhere;
    then more, shorter sequences that reuse the first descriptors of the array).  Both results
    must agree with affine_scan_ex(AFFINE_LOOKBACK) within the parity tolerance of the suite
    (the two are not bitwise equal by contract: the look-back folds whatever aggregates are
    published when it polls), and with the float64 oracle."""
    first = _inputs(1, 1 << 20, dtype, cuda_device, seed=901)
    second = _inputs(37, 40000, dtype, cuda_device, seed=902, with_h0=False)
    out1, out2 = _outputs(first), _outputs(second)      # NaN-prefilled, allocated up front
    torch.cuda.synchronize()
    # ---- the two calls in a row: one stream, no sync and no other work between them
    h1, hl1 = _run(lib.affine_scan_static_scratch, first, out1)
    assert lib.last_variant() == lib.AFFINE_LOOKBACK
    free_between = torch.cuda.mem_get_info(cuda_device)[0]
    h2, hl2 = _run(lib.affine_scan_static_scratch, second, out2)
    torch.cuda.synchronize()
    # nothing in this process allocated between the two readings except, possibly, the library:
    # the driver hands memory out in steps of 2 MiB or more, so 1 MiB of slack hides nothing
    assert torch.cuda.mem_get_info(cuda_device)[0] >= free_between - (1 << 20), \
        "free device memory shrank across a call that must not allocate"
    # ---- the existing path on the same inputs
    for (inp, h, hl, what) in ((first, h1, hl1, "first"), (second, h2, hl2, "second")):
        rh, rhl = _run(_existing, inp)
        torch.cuda.synchronize()
        assert rel_err(h, rh.double().cpu().numpy()) <= TOL[dtype], what
        assert rel_err(hl, rhl.double().cpu().numpy()) <= TOL[dtype], what
        href, hlref = oracle_affine(inp)
        assert_close(h, href, dtype, f"{what} call vs oracle: h")
        assert_close(hl, hlref, dtype, f"{what} call vs oracle: h_last")


@pytest.mark.gpu
def test_static_scratch_scalar_fallback_and_empty_shapes(cuda_device):
    """L not a multiple of the vector width takes the scalar-access kernel (1024-element tiles);
    L == 0 copies h0; both without scratch trouble after the vector calls above."""
    inp = _inputs(3, 5001, torch.float32, cuda_device, seed=903)
    h, hl = _run(lib.affine_scan_static_scratch, inp)
    rh, rhl = _run(_existing, inp)
    torch.cuda.synchronize()
    assert rel_err(h, rh.double().cpu().numpy()) <= TOL[torch.float32]
    assert rel_err(hl, rhl.double().cpu().numpy()) <= TOL[torch.float32]
    href, hlref = oracle_affine(inp)
    assert_close(h, href, torch.float32, "scalar fallback h")
    empty = {"a": torch.empty((4, 0), device=cuda_device), "u": torch.empty((4, 0), device=cuda_device),
             "h0": torch.arange(4, dtype=torch.float32, device=cuda_device)}
    _, hl0 = _run(lib.affine_scan_static_scratch, empty)
    torch.cuda.synchronize()
    assert torch.equal(hl0, empty["h0"])


def test_static_scratch_rejects_sizes_beyond_the_array():
    """The limit is checked before any pointer is looked at and before any device work, so this
    runs without a GPU: one element past the limit returns AFFINESCAN_ERR_TOO_LARGE (6) with a
    message that names the entry point; the limit itself passes the size check (and then fails
    on the NULL pointers, status 1)."""
    L = lib.load()
    n = ctypes.c_void_p(None)
    assert lib.affine_scan_static_scratch_max_elements(torch.float32) == 65535 * 4096
    assert lib.affine_scan_static_scratch_max_elements(torch.bfloat16) == 65535 * 8192
    assert lib.affine_scan_static_scratch_max_elements(torch.float32, vectorised=False) == 65535 * 1024
    for io, vec in ((lib.F32, 4), (lib.BF16, 8)):
        lim = lib.affine_scan_static_scratch_max_elements(io)
        assert L.affine_scan_static_scratch(n, n, n, n, n, 1, lim + vec, io, n) == 6
        assert L.affine_scan_static_scratch(n, n, n, n, n, 1, lim, io, n) == 1
        lim1 = lib.affine_scan_static_scratch_max_elements(io, vectorised=False)
        assert L.affine_scan_static_scratch(n, n, n, n, n, 1, lim1 + 1, io, n) == 6
    assert "affine_scan_static_scratch" in lib.status_string(6)
