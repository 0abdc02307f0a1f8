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


# ------------------------------------------------- full-size, every-element comparisons
def host_threads() -> int:
    """Host threads the TEST HARNESS spreads oracle calls over (oracle.c stays the plain
    one-thread loop; ctypes releases the GIL during each call)."""
    import os
    return max(1, min(32, os.cpu_count() or 1))


def oracle_selective_all_rows(inp, rows_per_task=64):
    """The oracle over EVERY (b, d) row of a selective workload, the row range cut into slices
    that run on several host threads.  Returns (y [batch, d_inner, L], h_last [batch, d_inner, N])
    in float64."""
    from concurrent.futures import ThreadPoolExecutor
    x = inp["x"]
    batch, d_inner, L = x.shape
    N = inp["A"].shape[1]
    host = {k: (None if v is None else v.detach().cpu()) for k, v in inp.items()}
    A64 = host["A"].double().numpy()
    D64 = None if host.get("D") is None else host["D"].double().numpy()
    yref = np.empty((batch, d_inner, L), dtype=np.float64)
    hlref = np.empty((batch, d_inner, N), dtype=np.float64)

    def task(b, d0, d1, B64, C64):
        y, hl = oracle.selective_scan_fwd(
            host["x"][b:b + 1, d0:d1].double().numpy(), host["delta"][b:b + 1, d0:d1].double().numpy(),
            A64[d0:d1], B64, C64, None if D64 is None else D64[d0:d1],
            None if host.get("h0") is None else host["h0"][b:b + 1, d0:d1].double().numpy())
        yref[b, d0:d1] = y[0]
        hlref[b, d0:d1] = hl[0]

    with ThreadPoolExecutor(host_threads()) as pool:
        futs = []
        for b in range(batch):
            B64 = host["B"][b:b + 1].double().numpy()
            C64 = host["C"][b:b + 1].double().numpy()
            for d0 in range(0, d_inner, rows_per_task):
                futs.append(pool.submit(task, b, d0, min(d_inner, d0 + rows_per_task), B64, C64))
        for f in futs:
            f.result()
    return yref, hlref


def rel_err_device(gpu: torch.Tensor, ref: np.ndarray, chunk_elems: int = 1 << 25) -> float:
    """max |gpu - ref| / (1 + |ref|) over EVERY element, evaluated in float64 on the device the
    result lives on (the reference slab is uploaded; nothing is sampled).  NaN/Inf => inf."""
    assert tuple(gpu.shape) == tuple(ref.shape), (gpu.shape, ref.shape)
    g = gpu.reshape(-1)
    r = np.ascontiguousarray(ref).reshape(-1)
    worst = 0.0
    for s0 in range(0, g.numel(), chunk_elems):
        s1 = min(g.numel(), s0 + chunk_elems)
        gd = g[s0:s1].double()
        rd = torch.from_numpy(r[s0:s1]).to(g.device)
        if not bool(torch.isfinite(gd).all()):
            return float("inf")
        worst = max(worst, float(((gd - rd).abs() / (1.0 + rd.abs())).max().item()))
    return worst


def assert_close_all(gpu, ref, dtype, what=""):
    err = rel_err_device(gpu, ref)
    assert err <= TOL[dtype], f"{what}: max|err|/(1+|ref|) = {err:.3e} > {TOL[dtype]:.0e} (all elements)"
    return err


def lane_row_ok(inp) -> bool:
    x = inp["x"]
    vec = 4 if x.dtype == torch.float32 else 8
    return inp["A"].shape[1] == 16 and x.shape[1] % 32 == 0 and x.shape[2] % vec == 0
