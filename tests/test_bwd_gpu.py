"""GPU parity of selective_scan_bwd against the float64 oracle's backward pass
(itself pinned by finite differences of the forward oracle, tests/test_oracle_pins_ext.py).

Tolerance: every gradient is produced in fp32 from the already-rounded io-dtype inputs, so the
io dtype does not enter; what does is the fp32 accumulation over L (dA: L*batch terms, dB/dC:
d_inner terms, the adjoint recurrence itself) and the 2-ulp ex2: max|err|/(1+|ref|) <= 2e-4,
twice BASELINE.json's fp32 bound for the forward (the backward recomputes the forward and then
runs a second recurrence on top of it).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_00601_b200 as lib
from workloads import config, make_selective_inputs, normal, to_f64_numpy

from util import rel_err, rel_err_device

pytestmark = pytest.mark.gpu

TOL_BWD = 2e-4
NAMES = ["dx", "ddelta", "dA", "dB", "dC", "dD", "dh0"]


def _inputs(batch, d_inner, L, dtype, dev, seed, with_h0=True, with_D=True):
    c = config(2, batch=batch, d_inner=d_inner, L=L, dtype=dtype, seed=seed)
    inp = make_selective_inputs(c, device=dev, with_h0=with_h0)
    if not with_D:
        inp["D"] = None
    inp["dy"] = normal(inp["x"].shape, seed=seed, stream=40, device=dev, dtype=dtype)
    inp["dh_last"] = normal((batch, d_inner, 16), seed=seed, stream=41, device=dev,
                            dtype=torch.float32)
    return inp


def gpu_bwd(inp, with_dh_last=True, workspace="torch"):
    x = inp["x"]
    batch, d_inner, L = x.shape
    dev = x.device
    nan = float("nan")
    out = {"dx": torch.full(x.shape, nan, device=dev), "ddelta": torch.full(x.shape, nan, device=dev),
           "dA": torch.full((d_inner, 16), nan, device=dev), "dB": torch.full((batch, 16, L), nan, device=dev),
           "dC": torch.full((batch, 16, L), nan, device=dev), "dD": torch.full((d_inner,), nan, device=dev),
           "dh0": torch.full((batch, d_inner, 16), nan, device=dev)}
    lib.selective_scan_bwd(x, inp["delta"], inp["A"], inp["B"], inp["C"], inp["D"], inp["h0"],
                           inp["dy"], inp["dh_last"] if with_dh_last else None, out["dx"],
                           out["ddelta"], out["dA"], out["dB"], out["dC"], out["dD"], out["dh0"],
                           workspace=workspace)
    torch.cuda.synchronize()
    return out


def oracle_bwd(inp, with_dh_last=True):
    f = to_f64_numpy
    return oracle.selective_scan_bwd(f(inp["x"]), f(inp["delta"]), f(inp["A"]), f(inp["B"]),
                                     f(inp["C"]), f(inp["D"]), f(inp["h0"]), f(inp["dy"]),
                                     f(inp["dh_last"]) if with_dh_last else None)


def check(inp, what, with_dh_last=True):
    out = gpu_bwd(inp, with_dh_last)
    ref = oracle_bwd(inp, with_dh_last)
    for k in NAMES:
        err = rel_err_device(out[k], ref[k])
        assert err <= TOL_BWD, f"{what} {k}: max|err|/(1+|ref|) = {err:.3e} > {TOL_BWD:.0e}"


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_backward_small_and_ragged_tiles(cuda_device, dtype):
    seed = 1000
    for (batch, d_inner, L) in [(1, 32, 8), (2, 32, 16), (1, 64, 24), (3, 32, 40), (2, 96, 264),
                                (1, 32, 1000), (2, 64, 2048)]:
        seed += 1
        inp = _inputs(batch, d_inner, L, dtype, cuda_device, seed, with_h0=(seed % 2 == 0),
                      with_D=(seed % 3 != 0))
        check(inp, f"bwd {dtype} {batch}x{d_inner}x{L}", with_dh_last=(seed % 2 == 1))


def test_backward_config2_shape_and_reproducibility(cuda_device):
    """BASELINE.json configs[1] shape (batch 2, d_inner 768, N 16, L 2048, fp32): every gradient
    element against the oracle; two runs are bitwise equal (fixed-order sums, no atomics)."""
    inp = _inputs(2, 768, 2048, torch.float32, cuda_device, 7, with_h0=False)
    check(inp, "bwd cfg2")
    a, b = gpu_bwd(inp), gpu_bwd(inp)
    for k in NAMES:
        assert torch.equal(a[k], b[k]), k


def test_backward_matches_autograd_of_a_torch_restatement(cuda_device):
    """Second, independent check: torch.autograd through a float64 restatement of the forward
    (plain torch ops on the GPU, test harness only) on a tiny shape."""
    dev = cuda_device
    inp = _inputs(1, 32, 64, torch.float32, dev, 9)
    leaves = {k: inp[k].double().requires_grad_(True) for k in ("x", "delta", "A", "B", "C", "D", "h0")}
    h = leaves["h0"]
    ys = []
    for t in range(64):
        a = torch.exp(leaves["delta"][:, :, t, None] * leaves["A"][None])
        u = leaves["delta"][:, :, t, None] * leaves["B"][:, None, :, t] * leaves["x"][:, :, t, None]
        h = a * h + u
        ys.append((h * leaves["C"][:, None, :, t]).sum(-1) + leaves["D"][None] * leaves["x"][:, :, t])
    y = torch.stack(ys, dim=-1)
    loss = (y * inp["dy"].double()).sum() + (h * inp["dh_last"].double()).sum()
    loss.backward()
    out = gpu_bwd(inp)
    for k, leaf in zip(NAMES, ("x", "delta", "A", "B", "C", "D", "h0")):
        assert rel_err(out[k], leaves[leaf].grad.cpu().numpy()) <= TOL_BWD, k


def test_backward_optional_outputs_empty_and_unsupported(cuda_device):
    dev = cuda_device
    inp = _inputs(1, 32, 64, torch.float32, dev, 11)
    full = gpu_bwd(inp)
    dx = torch.empty_like(full["dx"])
    lib.selective_scan_bwd(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"], inp["D"], inp["h0"],
                           inp["dy"], inp["dh_last"], dx, None, None, None, None, None, None)
    torch.cuda.synchronize()
    assert torch.equal(dx, full["dx"])
    # L == 0: only h_last = h0 depends on the inputs
    e = torch.empty((1, 32, 0), device=dev)
    bc = torch.empty((1, 16, 0), device=dev)
    dA = torch.full((32, 16), float("nan"), device=dev)
    dh0 = torch.full((1, 32, 16), float("nan"), device=dev)
    lib.selective_scan_bwd(e, e, inp["A"], bc, bc, None, None, e, inp["dh_last"], None, None, dA,
                           None, None, None, dh0)
    torch.cuda.synchronize()
    assert torch.equal(dh0, inp["dh_last"]) and torch.equal(dA, torch.zeros_like(dA))
    # shapes outside the tuned layout are refused, not mis-computed
    bad = _inputs(1, 33, 64, torch.float32, dev, 12)
    with pytest.raises(lib.AffineScanError) as ei:
        gpu_bwd(bad)
    assert ei.value.status == 4
    bad = _inputs(1, 32, 60, torch.float32, dev, 12)
    with pytest.raises(lib.AffineScanError):
        gpu_bwd(bad)


def test_backward_workspace_from_the_caller_from_torch_or_from_the_library(cuda_device):
    """The ~16 B per (b,d,t) of scratch may come from (i) torch's allocator through the binding
    (default), (ii) a buffer the caller passes to selective_scan_bwd_ws, (iii) a per-call
    cudaMallocAsync inside the library: the three give bitwise the same gradients, a dirty
    workspace changes nothing (every word is written before it is read), and a workspace that is
    too small is refused before any device work."""
    inp = _inputs(2, 64, 512, torch.bfloat16, cuda_device, 21)
    need = lib.selective_scan_bwd_workspace_bytes(2, 64, 16, 512)
    groups = 2 * 64 // 16
    assert need == 4 * (groups * (512 // 8) * 16 * 16 + groups * 512 * 32 + 2 * 64 * 16 + 2 * 64)
    assert lib.selective_scan_bwd_workspace_bytes(2, 65, 16, 512) == 0      # unsupported shape
    ref = gpu_bwd(inp, workspace="torch")
    check(inp, "bwd workspace=torch")
    ws = torch.full((need + 64,), 0xFF, dtype=torch.uint8, device=cuda_device)  # NaN bit patterns
    for mode in (ws, None):
        out = gpu_bwd(inp, workspace=mode)
        for k in NAMES:
            assert torch.equal(out[k], ref[k]), k
    with pytest.raises(lib.AffineScanError) as ei:
        gpu_bwd(inp, workspace=ws[:need - 16])
    assert ei.value.status == 6
