"""ctypes binding of libaffinescan (include/affinescan.h) — argument marshalling only.

Every function has the name and argument order of its C entry point.  Tensors are
torch tensors (PyTorch is used for device memory and streams only); every step of
the computation runs in the library's CUDA kernels.  There is NO fallback: if the
shared library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
import re

import torch

from . import build as _build

F32 = 0
BF16 = 1

VARIANT_AUTO = 0
AFFINE_LOOKBACK = 1
AFFINE_CTA_LOOP = 2
AFFINE_BLELLOCH = 3
AFFINE_WARP_SEQ = 4
SELECTIVE_WARP_ROW = 11
SELECTIVE_LANE_ROW = 12
SELECTIVE_WARP_ROW_TMA = 13
SELECTIVE_CHUNKED = 14

A_GENERAL = 0
A_SCALAR_PER_ROW = 1
A_POWERS = 2

VARIANT_NAMES = {
    0: "auto", 1: "affine_lookback", 2: "affine_cta_loop", 3: "affine_blelloch",
    4: "affine_warp_seq",
    11: "selective_warp_row", 12: "selective_lane_row",
    13: "selective_warp_row_tma", 14: "selective_chunked",
}

_vp = ctypes.c_void_p
_i64 = ctypes.c_int64
_int = ctypes.c_int

_SIGNATURES = {
    "affine_scan": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _i64, _int, _vp]),
    "affine_scan_ex": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _i64, _int, _int, _vp]),
    "affine_scan_host": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _i64, _int, _vp]),
    "affine_scan_static_scratch": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _i64, _int, _vp]),
    "affine_scan_static_scratch_max_elements": (_i64, [_int, _int]),
    "selective_scan_fwd": (_int, [_vp] * 9 + [_int, _int, _int, _i64, _int, _vp]),
    "selective_scan_fwd_ex": (_int, [_vp] * 9 + [_int, _int, _int, _i64, _int, _int, _vp]),
    "selective_scan_fwd_host": (_int, [_vp] * 9 + [_int, _int, _int, _i64, _int, _vp]),
    "selective_scan_fwd_ext": (_int, [_vp] * 12 + [_int, _int, _int, _i64, _int, _int, _int, _int, _vp]),
    "selective_scan_fwd_ext_host": (_int, [_vp] * 12 + [_int, _int, _int, _i64, _int, _int, _int, _vp]),
    "selective_scan_fwd_gated": (_int, [_vp] * 11 + [_int, _int, _int, _i64, _int, _vp]),
    "affinescan_reset_mask_from_cu_seqlens": (_int, [_vp, _int, _vp, _i64, _vp]),
    "selective_scan_slice_aggregate": (_int, [_vp] * 7 + [_int, _int, _int, _i64, _int, _vp]),
    "affinescan_compose_carry": (_int, [_vp] * 4 + [_int, _int, _i64, _vp]),
    "selective_scan_bwd": (_int, [_vp] * 16 + [_int, _int, _int, _i64, _int, _vp]),
    "selective_scan_bwd_ws": (_int, [_vp] * 16 + [_int, _int, _int, _i64, _int, _vp, _i64, _vp]),
    "selective_scan_bwd_workspace_bytes": (_i64, [_int, _int, _int, _i64]),
    "affinescan_status_string": (ctypes.c_char_p, [_int]),
    "affinescan_last_cuda_error": (_int, []),
    "affinescan_last_variant": (_int, []),
    "affinescan_launch_count": (_i64, []),
    "affinescan_version": (_int, []),
    "affinescan_cached_scratch_buffers": (_int, []),
    "affinescan_release_cache": (_int, []),
    "affinescan_set_option": (_int, [_int, _int]),
}

OPT_LANE_ROW_G = 1
OPT_LANE_ROW_POLY16 = 2
OPT_DETERMINISTIC = 3


class AffineScanError(RuntimeError):
    def __init__(self, fn: str, status: int, detail: str, cuda_error: int):
        self.status = status
        self.cuda_error = cuda_error
        extra = f" (cudaError {cuda_error})" if status == 5 else ""
        super().__init__(f"{fn} failed: status {status}: {detail}{extra}")


_lib = None


def library_path() -> str:
    return _build.LIB_PATH


def declared_symbols(header_path: str | None = None):
    """Names of every AFFINESCAN_API function declared in include/affinescan.h."""
    if header_path is None:
        header_path = os.path.join(_build.ROOT, "include", "affinescan.h")
    with open(header_path) as f:
        text = f.read()
    return re.findall(r"AFFINESCAN_API\s+[\w\s\*]+?\b(\w+)\s*\(", text)


def load():
    """dlopen libaffinescan.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise FileNotFoundError(
                f"{path} not found: build it with `python -m paper_2606_00601_b200.build` "
                "(or __graft_entry__.build()); there is no CPU fallback")
        lib = ctypes.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(fn: str, status: int):
    if status != 0:
        lib = load()
        raise AffineScanError(fn, status, lib.affinescan_status_string(status).decode(),
                              lib.affinescan_last_cuda_error())


def _io_dtype(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise TypeError(f"io dtype must be float32 or bfloat16, got {t.dtype}")


def _ptr(t, *, dtype=None, shape=None, device=None, name="tensor"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor):
        raise TypeError(f"{name}: expected a torch.Tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name}: expected {dtype}, got {t.dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    if not t.is_contiguous():
        raise ValueError(f"{name}: must be contiguous (dense row-major)")
    if device is not None and t.device.type != device:
        raise ValueError(f"{name}: expected a {device} tensor, got {t.device}")
    return t.data_ptr() if t.numel() else (t.data_ptr() or None)


def _stream_ptr(stream, ref: torch.Tensor):
    if stream is None:
        if ref.is_cuda:
            return torch.cuda.current_stream(ref.device).cuda_stream
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


# ------------------------------------------------------------------------ affine_scan
def _affine_args(a, u, h0, h, h_last, device):
    if a.dim() != 2:
        raise ValueError("a must be [num_seq, L]")
    S, L = a.shape
    io = _io_dtype(a)
    return (
        _ptr(a, shape=(S, L), device=device, name="a"),
        _ptr(u, dtype=a.dtype, shape=(S, L), device=device, name="u"),
        _ptr(h0, dtype=torch.float32, shape=(S,), device=device, name="h0"),
        _ptr(h, dtype=a.dtype, shape=(S, L), device=device, name="h"),
        _ptr(h_last, dtype=torch.float32, shape=(S,), device=device, name="h_last"),
        S, L, io,
    )


def affine_scan(a, u, h0, h, h_last, stream=None):
    """h[s,t] = a[s,t]*h[s,t-1] + u[s,t]; device tensors; async on ``stream``."""
    args = _affine_args(a, u, h0, h, h_last, "cuda")
    with torch.cuda.device(a.device):
        _check("affine_scan", load().affine_scan(*args, _stream_ptr(stream, a)))


def affine_scan_ex(a, u, h0, h, h_last, variant, stream=None):
    args = _affine_args(a, u, h0, h, h_last, "cuda")
    with torch.cuda.device(a.device):
        _check("affine_scan_ex", load().affine_scan_ex(*args, int(variant), _stream_ptr(stream, a)))


def affine_scan_static_scratch(a, u, h0, h, h_last, stream=None):
    """affine_scan for callers that may not allocate device memory (a server that gave all of
    HBM to its own cache, an allocator that must own every byte, a loop that cannot afford the
    driver's allocation lock): the look-back descriptors sit in a fixed 1 MiB array inside the
    library instead of cudaMallocAsync scratch.  Same result as
    ``affine_scan_ex(..., AFFINE_LOOKBACK)``.  Raises ``AffineScanError`` with status 6 when
    ``num_seq * L`` exceeds ``affine_scan_static_scratch_max_elements``.  Every call on a GPU
    shares that one array: calls that may overlap on the GPU race, so keep them on one stream.
    Make the first call on each device outside stream capture (it looks up the array's address).
    """
    args = _affine_args(a, u, h0, h, h_last, "cuda")
    with torch.cuda.device(a.device):
        _check("affine_scan_static_scratch",
               load().affine_scan_static_scratch(*args, _stream_ptr(stream, a)))


def affine_scan_static_scratch_max_elements(io_dtype, vectorised=True) -> int:
    """Largest ``num_seq * L`` affine_scan_static_scratch accepts (``io_dtype``: a torch dtype or
    F32 / BF16; ``vectorised=False``: the limit of the scalar-access fallback)."""
    if isinstance(io_dtype, torch.dtype):
        io_dtype = {torch.float32: F32, torch.bfloat16: BF16}[io_dtype]
    return int(load().affine_scan_static_scratch_max_elements(int(io_dtype), int(bool(vectorised))))


def affine_scan_host(a, u, h0, h, h_last, stream=None):
    """Same with HOST tensors (pinned or pageable); synchronises before returning."""
    args = _affine_args(a, u, h0, h, h_last, "cpu")
    _check("affine_scan_host", load().affine_scan_host(*args, _stream_ptr(stream, a)))


# ----------------------------------------------------------------- selective_scan_fwd
def _selective_args(x, delta, A, B, C, D, h0, y, h_last, device):
    if x.dim() != 3:
        raise ValueError("x must be [batch, d_inner, L]")
    if A.dim() != 2:
        raise ValueError("A must be [d_inner, N]")
    batch, d_inner, L = x.shape
    N = A.shape[1]
    io = _io_dtype(x)
    f32 = torch.float32
    return (
        _ptr(x, shape=(batch, d_inner, L), device=device, name="x"),
        _ptr(delta, dtype=x.dtype, shape=(batch, d_inner, L), device=device, name="delta"),
        _ptr(A, dtype=f32, shape=(d_inner, N), device=device, name="A"),
        _ptr(B, dtype=x.dtype, shape=(batch, N, L), device=device, name="B"),
        _ptr(C, dtype=x.dtype, shape=(batch, N, L), device=device, name="C"),
        _ptr(D, dtype=f32, shape=(d_inner,), device=device, name="D"),
        _ptr(h0, dtype=f32, shape=(batch, d_inner, N), device=device, name="h0"),
        _ptr(y, dtype=x.dtype, shape=(batch, d_inner, L), device=device, name="y"),
        _ptr(h_last, dtype=f32, shape=(batch, d_inner, N), device=device, name="h_last"),
        batch, d_inner, N, L, io,
    )


def selective_scan_fwd(x, delta, A, B, C, D, h0, y, h_last, stream=None):
    """Fused Mamba-style forward selective scan; device tensors; async on ``stream``."""
    args = _selective_args(x, delta, A, B, C, D, h0, y, h_last, "cuda")
    with torch.cuda.device(x.device):
        _check("selective_scan_fwd", load().selective_scan_fwd(*args, _stream_ptr(stream, x)))


def selective_scan_fwd_ex(x, delta, A, B, C, D, h0, y, h_last, variant, stream=None):
    args = _selective_args(x, delta, A, B, C, D, h0, y, h_last, "cuda")
    with torch.cuda.device(x.device):
        _check("selective_scan_fwd_ex",
               load().selective_scan_fwd_ex(*args, int(variant), _stream_ptr(stream, x)))


def selective_scan_fwd_host(x, delta, A, B, C, D, h0, y, h_last, stream=None):
    """Same with HOST tensors (pinned or pageable); synchronises before returning."""
    args = _selective_args(x, delta, A, B, C, D, h0, y, h_last, "cpu")
    _check("selective_scan_fwd_host",
           load().selective_scan_fwd_host(*args, _stream_ptr(stream, x)))


def _ext_args(x, delta, A, B, C, D, z, delta_bias, reset, h0, y, h_last, device):
    base = _selective_args(x, delta, A, B, C, D, h0, y, h_last, device)
    batch, d_inner, L = x.shape
    (px, pdelta, pA, pB, pC, pD, ph0, py, phl, batch, d_inner, N, L, io) = base
    return (px, pdelta, pA, pB, pC, pD,
            _ptr(z, dtype=x.dtype, shape=(batch, d_inner, L), device=device, name="z"),
            _ptr(delta_bias, dtype=torch.float32, shape=(d_inner,), device=device, name="delta_bias"),
            _ptr(reset, dtype=torch.uint8, shape=(batch, L), device=device, name="reset"),
            ph0, py, phl, batch, d_inner, N, L, io)


def selective_scan_fwd_ext(x, delta, A, B, C, D, z, delta_bias, reset, h0, y, h_last,
                           delta_softplus=False, a_structure=A_GENERAL, variant=VARIANT_AUTO,
                           stream=None):
    """selective_scan_fwd with the fused softplus/bias prologue, silu(z) gate and resets."""
    args = _ext_args(x, delta, A, B, C, D, z, delta_bias, reset, h0, y, h_last, "cuda")
    with torch.cuda.device(x.device):
        _check("selective_scan_fwd_ext",
               load().selective_scan_fwd_ext(*args, int(bool(delta_softplus)), int(a_structure),
                                             int(variant), _stream_ptr(stream, x)))


def selective_scan_fwd_ext_host(x, delta, A, B, C, D, z, delta_bias, reset, h0, y, h_last,
                                delta_softplus=False, a_structure=A_GENERAL, stream=None):
    args = _ext_args(x, delta, A, B, C, D, z, delta_bias, reset, h0, y, h_last, "cpu")
    _check("selective_scan_fwd_ext_host",
           load().selective_scan_fwd_ext_host(*args, int(bool(delta_softplus)), int(a_structure),
                                              _stream_ptr(stream, x)))


def selective_scan_fwd_gated(x, delta_raw, delta_bias, A, B, C, D, z, h0, y, h_last, stream=None):
    """Delta = softplus(delta_raw + delta_bias[d]) prologue and y * silu(z) epilogue, fused."""
    (px, pdelta, pA, pB, pC, pD, pz, pbias, _, ph0, py, phl, batch, d_inner, N, L, io) = _ext_args(
        x, delta_raw, A, B, C, D, z, delta_bias, None, h0, y, h_last, "cuda")
    with torch.cuda.device(x.device):
        _check("selective_scan_fwd_gated",
               load().selective_scan_fwd_gated(px, pdelta, pbias, pA, pB, pC, pD, pz, ph0, py, phl,
                                               batch, d_inner, N, L, io, _stream_ptr(stream, x)))


def selective_scan_bwd_workspace_bytes(batch, d_inner, N, L) -> int:
    return int(load().selective_scan_bwd_workspace_bytes(int(batch), int(d_inner), int(N), int(L)))


def selective_scan_bwd(x, delta, A, B, C, D, h0, dy, dh_last, dx, ddelta, dA, dB, dC, dD, dh0,
                       stream=None, workspace="torch"):
    """Gradients of <dy, y> + <dh_last, h_last> of selective_scan_fwd; outputs fp32, may be None.

    ``workspace``: "torch" (default) takes the ~16 B per (b,d,t) of scratch from torch's caching
    allocator for this call, so torch sees, reuses and can reclaim it; a uint8 device tensor of at
    least ``selective_scan_bwd_workspace_bytes`` is used as is; None lets the library take it
    from cudaMallocAsync per call (the plain C entry point)."""
    batch, d_inner, L = x.shape
    N = A.shape[1]
    f32 = torch.float32
    bdl, bnl, bdn = (batch, d_inner, L), (batch, N, L), (batch, d_inner, N)
    args = (
        _ptr(x, shape=bdl, device="cuda", name="x"),
        _ptr(delta, dtype=x.dtype, shape=bdl, device="cuda", name="delta"),
        _ptr(A, dtype=f32, shape=(d_inner, N), device="cuda", name="A"),
        _ptr(B, dtype=x.dtype, shape=bnl, device="cuda", name="B"),
        _ptr(C, dtype=x.dtype, shape=bnl, device="cuda", name="C"),
        _ptr(D, dtype=f32, shape=(d_inner,), device="cuda", name="D"),
        _ptr(h0, dtype=f32, shape=bdn, device="cuda", name="h0"),
        _ptr(dy, dtype=x.dtype, shape=bdl, device="cuda", name="dy"),
        _ptr(dh_last, dtype=f32, shape=bdn, device="cuda", name="dh_last"),
        _ptr(dx, dtype=f32, shape=bdl, device="cuda", name="dx"),
        _ptr(ddelta, dtype=f32, shape=bdl, device="cuda", name="ddelta"),
        _ptr(dA, dtype=f32, shape=(d_inner, N), device="cuda", name="dA"),
        _ptr(dB, dtype=f32, shape=bnl, device="cuda", name="dB"),
        _ptr(dC, dtype=f32, shape=bnl, device="cuda", name="dC"),
        _ptr(dD, dtype=f32, shape=(d_inner,), device="cuda", name="dD"),
        _ptr(dh0, dtype=f32, shape=bdn, device="cuda", name="dh0"),
    )
    with torch.cuda.device(x.device):
        sp = _stream_ptr(stream, x)
        if isinstance(workspace, str):
            if workspace != "torch":
                raise ValueError("workspace must be 'torch', a uint8 device tensor or None")
            nbytes = selective_scan_bwd_workspace_bytes(batch, d_inner, N, L)
            # a raw stream handle cannot be recorded on a torch tensor: the library allocates then
            torch_stream = stream if isinstance(stream, torch.cuda.Stream) else \
                (torch.cuda.current_stream(x.device) if stream is None else None)
            workspace = None
            if nbytes > 0 and torch_stream is not None:
                workspace = torch.empty(nbytes, dtype=torch.uint8, device=x.device)
                workspace.record_stream(torch_stream)
        if workspace is None:
            _check("selective_scan_bwd",
                   load().selective_scan_bwd(*args, batch, d_inner, N, L, _io_dtype(x), sp))
        else:
            _check("selective_scan_bwd_ws",
                   load().selective_scan_bwd_ws(
                       *args, batch, d_inner, N, L, _io_dtype(x),
                       _ptr(workspace, dtype=torch.uint8, device="cuda", name="workspace"),
                       workspace.numel(), sp))


def selective_scan_slice_aggregate(x, delta, A, B, C, P, U, stream=None):
    """(P, U) of this rank's L-slice per (row, state): step 1 of the L-sharded scan."""
    batch, d_inner, L = x.shape
    N = A.shape[1]
    f32 = torch.float32
    args = (
        _ptr(x, shape=(batch, d_inner, L), device="cuda", name="x"),
        _ptr(delta, dtype=x.dtype, shape=(batch, d_inner, L), device="cuda", name="delta"),
        _ptr(A, dtype=f32, shape=(d_inner, N), device="cuda", name="A"),
        _ptr(B, dtype=x.dtype, shape=(batch, N, L), device="cuda", name="B"),
        _ptr(C, dtype=x.dtype, shape=(batch, N, L), device="cuda", name="C"),
        _ptr(P, dtype=f32, shape=(batch, d_inner, N), device="cuda", name="P"),
        _ptr(U, dtype=f32, shape=(batch, d_inner, N), device="cuda", name="U"),
    )
    with torch.cuda.device(x.device):
        _check("selective_scan_slice_aggregate",
               load().selective_scan_slice_aggregate(*args, batch, d_inner, N, L, _io_dtype(x),
                                                     _stream_ptr(stream, x)))


def compose_carry(P_all, U_all, h0, h_in, rank, stream=None):
    """h_in = fold of the aggregates of ranks < rank applied to h0: step 3 of the L-sharded scan."""
    world = int(P_all.shape[0])
    n = int(h_in.numel())
    f32 = torch.float32
    with torch.cuda.device(h_in.device):
        _check("affinescan_compose_carry",
               load().affinescan_compose_carry(
                   _ptr(P_all.reshape(world, n), dtype=f32, device="cuda", name="P_all"),
                   _ptr(U_all.reshape(world, n), dtype=f32, device="cuda", name="U_all"),
                   _ptr(None if h0 is None else h0.reshape(n), dtype=f32, device="cuda", name="h0"),
                   _ptr(h_in.reshape(n), dtype=f32, device="cuda", name="h_in"),
                   int(rank), world, n, _stream_ptr(stream, h_in)))


def reset_mask_from_cu_seqlens(cu_seqlens, reset_row, stream=None):
    """reset_row[t] = 1 at every t in cu_seqlens (int32, device), 0 elsewhere; reset_row: [L] uint8."""
    if cu_seqlens.dtype != torch.int32 or reset_row.dtype != torch.uint8:
        raise TypeError("cu_seqlens must be int32 and reset_row uint8")
    with torch.cuda.device(reset_row.device):
        _check("affinescan_reset_mask_from_cu_seqlens",
               load().affinescan_reset_mask_from_cu_seqlens(
                   _ptr(cu_seqlens, device="cuda", name="cu_seqlens"), int(cu_seqlens.numel()),
                   _ptr(reset_row, device="cuda", name="reset_row"), int(reset_row.numel()),
                   _stream_ptr(stream, reset_row)))


# ------------------------------------------------------------------------ introspection
def status_string(status: int) -> str:
    return load().affinescan_status_string(int(status)).decode()


def last_cuda_error() -> int:
    return load().affinescan_last_cuda_error()


def last_variant() -> int:
    return load().affinescan_last_variant()


def launch_count() -> int:
    return load().affinescan_launch_count()


def version() -> int:
    return load().affinescan_version()


def cached_scratch_buffers(device=None) -> int:
    """Look-back scratch buffers the library caches on ``device`` (default: current)."""
    with torch.cuda.device(device):
        return load().affinescan_cached_scratch_buffers()


def release_cache() -> None:
    _check("affinescan_release_cache", load().affinescan_release_cache())


def set_option(key: int, value: int) -> None:
    """Process-wide tuning knob (ablations / sweeps); -1 restores the default."""
    _check("affinescan_set_option", load().affinescan_set_option(int(key), int(value)))
