"""Shared helpers for the parity tests: run the CUDA path through the binding, run the
oracle on the very same bytes, and compare with BASELINE.json's tolerances."""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_2606_00601_b200 as lib
from workloads import to_f64_numpy

# BASELINE.json north_star: max|err| <= tol * (1 + |ref|)
TOL = {torch.float32: 1e-4, torch.bfloat16: 2e-2}


def rel_err(gpu, ref) -> float:
    """max_i |gpu_i - ref_i| / (1 + |ref_i|); NaN/Inf in gpu => inf."""
    g = to_f64_numpy(gpu) if isinstance(gpu, torch.Tensor) else np.asarray(gpu, dtype=np.float64)
    r = np.asarray(ref, dtype=np.float64)
    assert g.shape == r.shape, (g.shape, r.shape)
    if g.size == 0:
        return 0.0
    if not np.all(np.isfinite(g)):
        return float("inf")
    return float(np.max(np.abs(g - r) / (1.0 + np.abs(r))))


def assert_close(gpu, ref, dtype, what=""):
    err = rel_err(gpu, ref)
    assert err <= TOL[dtype], f"{what}: max|err|/(1+|ref|) = {err:.3e} > {TOL[dtype]:.0e}"
    return err


# ------------------------------------------------------------------------- affine_scan
def gpu_affine(inp, variant=lib.VARIANT_AUTO, want_h_last=True, stream=None):
    a, u, h0 = inp["a"], inp["u"], inp.get("h0")
    h = torch.full_like(a, float("nan"))
    h_last = torch.full((a.shape[0],), float("nan"), dtype=torch.float32, device=a.device) \
        if want_h_last else None
    lib.affine_scan_ex(a, u, h0, h, h_last, variant, stream)
    torch.cuda.synchronize()
    return h, h_last


def oracle_affine(inp):
    return oracle.affine_scan(to_f64_numpy(inp["a"]), to_f64_numpy(inp["u"]),
                              to_f64_numpy(inp.get("h0")))


def check_affine(inp, variant=lib.VARIANT_AUTO, what=""):
    h, h_last = gpu_affine(inp, variant)
    href, hlref = oracle_affine(inp)
    dt = inp["a"].dtype
    e1 = assert_close(h, href, dt, f"{what} h")
    # h_last is fp32 even for bf16 io: it must match the un-rounded final state
    e2 = assert_close(h_last, hlref, dt, f"{what} h_last")
    return e1, e2


# ------------------------------------------------------------------ selective_scan_fwd
def gpu_selective(inp, variant=lib.VARIANT_AUTO, want_h_last=True, stream=None):
    x = inp["x"]
    batch, d_inner, _ = x.shape
    N = inp["A"].shape[1]
    y = torch.full_like(x, float("nan"))
    h_last = torch.full((batch, d_inner, N), float("nan"), dtype=torch.float32, device=x.device) \
        if want_h_last else None
    lib.selective_scan_fwd_ex(x, inp["delta"], inp["A"], inp["B"], inp["C"], inp.get("D"),
                              inp.get("h0"), y, h_last, variant, stream)
    torch.cuda.synchronize()
    return y, h_last


def oracle_selective(inp):
    return oracle.selective_scan_fwd(*(to_f64_numpy(inp.get(k)) for k in
                                       ("x", "delta", "A", "B", "C", "D", "h0")))


def oracle_selective_rows(inp, rows):
    """Oracle on a sample of (b, d) rows: returns (y [len(rows), L], h_last [len(rows), N])."""
    ys, hs = [], []
    for (b, d) in rows:
        sub = {
            "x": inp["x"][b:b + 1, d:d + 1], "delta": inp["delta"][b:b + 1, d:d + 1],
            "A": inp["A"][d:d + 1], "B": inp["B"][b:b + 1], "C": inp["C"][b:b + 1],
            "D": None if inp.get("D") is None else inp["D"][d:d + 1],
            "h0": None if inp.get("h0") is None else inp["h0"][b:b + 1, d:d + 1],
        }
        y, hl = oracle_selective(sub)
        ys.append(y[0, 0])
        hs.append(hl[0, 0])
    return np.stack(ys), np.stack(hs)


def check_selective(inp, variant=lib.VARIANT_AUTO, what=""):
    y, h_last = gpu_selective(inp, variant)
    yref, hlref = oracle_selective(inp)
    dt = inp["x"].dtype
    e1 = assert_close(y, yref, dt, f"{what} y")
    e2 = assert_close(h_last, hlref, dt, f"{what} h_last")
    return e1, e2


def lane_row_ok(inp) -> bool:
    x = inp["x"]
    vec = 4 if x.dtype == torch.float32 else 8
    return inp["A"].shape[1] == 16 and x.shape[1] % 32 == 0 and x.shape[2] % vec == 0
