"""numpy/ctypes front end of ``oracle.c`` — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The arithmetic lives in ``oracle.c`` (plain C, float64, sequential loops written
from PAPER.md Eq.(1)-(7) and BASELINE.json's north_star).  This file only builds
that C file with gcc, widens the caller's arrays to float64 (exact for fp32 and
bf16 storage) and marshals pointers.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_i64 = ctypes.c_int64


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so (gcc, no FMA contraction, no fast-math)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(
                ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared",
                 "-fPIC", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_affine_scan.argtypes = [_dp, _dp, _dp, _dp, _dp, _i64, _i64]
        lib.oracle_affine_scan.restype = None
        lib.oracle_selective_scan_fwd.argtypes = [_dp] * 9 + [_i64] * 4
        lib.oracle_selective_scan_fwd.restype = None
        lib.oracle_selective_scan_fwd_ext.argtypes = [_dp] * 12 + [_i64] * 5
        lib.oracle_selective_scan_fwd_ext.restype = None
        lib.oracle_selective_scan_bwd.argtypes = [_dp] * 16 + [_i64] * 4
        lib.oracle_selective_scan_bwd.restype = None
        lib.oracle_compose.argtypes = [ctypes.c_double] * 4 + [_dp, _dp]
        lib.oracle_compose.restype = None
        lib.oracle_fold_pairs.argtypes = [_dp, _dp, _i64, _dp, _dp]
        lib.oracle_fold_pairs.restype = None
        lib.oracle_blelloch_scan.argtypes = [_dp, _dp, ctypes.c_double, _dp, _i64]
        lib.oracle_blelloch_scan.restype = None
        _lib = lib
    return _lib


def _f64(arr, shape=None):
    """Widen to a C-contiguous float64 array (exact for fp32/bf16-valued input)."""
    if arr is None:
        return None
    out = np.ascontiguousarray(np.asarray(arr, dtype=np.float64))
    if shape is not None and tuple(out.shape) != tuple(shape):
        raise ValueError(f"oracle: expected shape {tuple(shape)}, got {tuple(out.shape)}")
    return out


def _ptr(arr):
    return None if arr is None else arr.ctypes.data_as(_dp)


def affine_scan(a, u, h0=None):
    """h[s,t] = a[s,t]*h[s,t-1] + u[s,t], h[s,-1] = h0[s] (Eq.(1)-(3), (5)).

    a, u: [S, L]; h0: [S] or None.  Returns (h [S, L], h_last [S]) in float64.
    """
    a = _f64(a)
    if a.ndim != 2:
        raise ValueError("oracle.affine_scan: a must be [S, L]")
    S, L = a.shape
    u = _f64(u, (S, L))
    h0 = _f64(h0, (S,))
    h = np.empty((S, L), dtype=np.float64)
    h_last = np.empty((S,), dtype=np.float64)
    _load().oracle_affine_scan(_ptr(a), _ptr(u), _ptr(h0), _ptr(h), _ptr(h_last), S, L)
    return h, h_last


def selective_scan_fwd(x, delta, A, B, C, D=None, h0=None):
    """Mamba-style forward selective scan (BASELINE.json north_star; Eq.(3)-(4)).

    x, delta: [batch, d_inner, L]; A: [d_inner, N]; B, C: [batch, N, L];
    D: [d_inner] or None; h0: [batch, d_inner, N] or None.
    Returns (y [batch, d_inner, L], h_last [batch, d_inner, N]) in float64.
    """
    x = _f64(x)
    if x.ndim != 3:
        raise ValueError("oracle.selective_scan_fwd: x must be [batch, d_inner, L]")
    batch, d_inner, L = x.shape
    delta = _f64(delta, (batch, d_inner, L))
    A = _f64(A)
    if A.ndim != 2 or A.shape[0] != d_inner:
        raise ValueError("oracle.selective_scan_fwd: A must be [d_inner, N]")
    N = A.shape[1]
    B = _f64(B, (batch, N, L))
    C = _f64(C, (batch, N, L))
    D = _f64(D, (d_inner,))
    h0 = _f64(h0, (batch, d_inner, N))
    y = np.empty((batch, d_inner, L), dtype=np.float64)
    h_last = np.empty((batch, d_inner, N), dtype=np.float64)
    _load().oracle_selective_scan_fwd(_ptr(x), _ptr(delta), _ptr(A), _ptr(B), _ptr(C), _ptr(D),
                                      _ptr(h0), _ptr(y), _ptr(h_last), batch, d_inner, N, L)
    return y, h_last


def selective_scan_fwd_ext(x, delta, A, B, C, D=None, z=None, delta_bias=None, reset=None,
                           h0=None, delta_softplus=False):
    """Forward selective scan with the fused steps either side of the recurrence (PAPER.md
    §6.7, §9): Delta = softplus(delta + delta_bias[d]) if ``delta_softplus`` (else delta +
    bias), state reset to 0 where ``reset[b, t] != 0``, and y <- y * silu(z).

    z: [batch, d_inner, L] or None; delta_bias: [d_inner] or None; reset: [batch, L] or None.
    Returns (y, h_last) in float64.
    """
    x = _f64(x)
    if x.ndim != 3:
        raise ValueError("oracle.selective_scan_fwd_ext: x must be [batch, d_inner, L]")
    batch, d_inner, L = x.shape
    delta = _f64(delta, (batch, d_inner, L))
    A = _f64(A)
    if A.ndim != 2 or A.shape[0] != d_inner:
        raise ValueError("oracle.selective_scan_fwd_ext: A must be [d_inner, N]")
    N = A.shape[1]
    B = _f64(B, (batch, N, L))
    C = _f64(C, (batch, N, L))
    D = _f64(D, (d_inner,))
    z = _f64(z, (batch, d_inner, L))
    delta_bias = _f64(delta_bias, (d_inner,))
    reset = _f64(reset, (batch, L))
    h0 = _f64(h0, (batch, d_inner, N))
    y = np.empty((batch, d_inner, L), dtype=np.float64)
    h_last = np.empty((batch, d_inner, N), dtype=np.float64)
    _load().oracle_selective_scan_fwd_ext(_ptr(x), _ptr(delta), _ptr(A), _ptr(B), _ptr(C),
                                          _ptr(D), _ptr(z), _ptr(delta_bias), _ptr(reset),
                                          _ptr(h0), _ptr(y), _ptr(h_last), batch, d_inner, N, L,
                                          1 if delta_softplus else 0)
    return y, h_last


def selective_scan_bwd(x, delta, A, B, C, D, h0, dy, dh_last=None):
    """Gradients of loss = <dy, y> + <dh_last, h_last> of ``selective_scan_fwd`` with respect
    to every input.  Returns dict(dx, ddelta, dA, dB, dC, dD, dh0) in float64."""
    x = _f64(x)
    batch, d_inner, L = x.shape
    delta = _f64(delta, (batch, d_inner, L))
    A = _f64(A)
    N = A.shape[1]
    B = _f64(B, (batch, N, L))
    C = _f64(C, (batch, N, L))
    D = _f64(D, (d_inner,))
    h0 = _f64(h0, (batch, d_inner, N))
    dy = _f64(dy, (batch, d_inner, L))
    dh_last = _f64(dh_last, (batch, d_inner, N))
    out = {
        "dx": np.empty((batch, d_inner, L)), "ddelta": np.empty((batch, d_inner, L)),
        "dA": np.empty((d_inner, N)), "dB": np.empty((batch, N, L)),
        "dC": np.empty((batch, N, L)), "dD": np.empty((d_inner,)),
        "dh0": np.empty((batch, d_inner, N)),
    }
    _load().oracle_selective_scan_bwd(_ptr(x), _ptr(delta), _ptr(A), _ptr(B), _ptr(C), _ptr(D),
                                      _ptr(h0), _ptr(dy), _ptr(dh_last), _ptr(out["dx"]),
                                      _ptr(out["ddelta"]), _ptr(out["dA"]), _ptr(out["dB"]),
                                      _ptr(out["dC"]), _ptr(out["dD"]), _ptr(out["dh0"]),
                                      batch, d_inner, N, L)
    return out


def compose(later, earlier):
    """(A2,U2) (+) (A1,U1) = (A2*A1, A2*U1 + U2) — PAPER.md Eq.(7); left = later."""
    A = ctypes.c_double()
    U = ctypes.c_double()
    _load().oracle_compose(float(later[0]), float(later[1]), float(earlier[0]), float(earlier[1]),
                           ctypes.byref(A), ctypes.byref(U))
    return A.value, U.value


def fold_pairs(a, u):
    """Total composition e_{L-1} (+) ... (+) e_0 of the pairs (a_t, u_t); (1, 0) if empty."""
    a = _f64(a)
    u = _f64(u, a.shape)
    A = ctypes.c_double()
    U = ctypes.c_double()
    _load().oracle_fold_pairs(_ptr(a), _ptr(u), a.shape[0], ctypes.byref(A), ctypes.byref(U))
    return A.value, U.value


def blelloch_scan(a, u, h0=0.0):
    """CPU model of the paper's Blelloch schedule (§3.3, §4) for one sequence."""
    a = _f64(a)
    u = _f64(u, a.shape)
    h = np.empty_like(a)
    _load().oracle_blelloch_scan(_ptr(a), _ptr(u), float(h0), _ptr(h), a.shape[0])
    return h
