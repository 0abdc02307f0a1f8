"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path
(tests, bench.py).  It contains none of the method's arithmetic: no recurrence,
no composition, no exp(Δ·A) — only random draws and the input recipe that
BASELINE.json's ``configs`` state (softplus for Δ and −exp(U) for A are part of
that recipe, i.e. of how the *inputs* are distributed).

The generator is counter-based (splitmix64 of ``seed, stream, index``), so a value
depends only on (seed, stream, flat index) — never on chunking or device — up to
the last-ulp differences of log/cos/exp between CPU and GPU libm.  Tests therefore
never regenerate an input on the other side: the bytes handed to the oracle are
copied from the very tensor handed to the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import torch

_MASK64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_CHUNK = 1 << 24


def _s64(v: int) -> int:
    """Two's-complement reinterpretation of an unsigned 64-bit constant."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical right shift of int64 lanes."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _splitmix64(z: torch.Tensor) -> torch.Tensor:
    z = z + _s64(_GOLDEN)
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def _key(seed: int, stream: int) -> int:
    return _s64((seed * 0xD1342543DE82EF95 + (stream + 1) * _GOLDEN) & _MASK64)


def _bits(seed: int, stream: int, start: int, count: int, device) -> torch.Tensor:
    idx = torch.arange(start, start + count, dtype=torch.int64, device=device)
    return _splitmix64(_splitmix64(idx ^ _key(seed, stream)))


def _unit(bits: torch.Tensor) -> torch.Tensor:
    """53-bit uniform in (0, 1]: never 0, so log() is finite."""
    return (_lsr(bits, 11).to(torch.float64) + 1.0) * (2.0 ** -53)


def _fill(kind, shape, seed, stream, device, dtype, p0=0.0, p1=1.0):
    n = 1
    for s in shape:
        n *= int(s)
    out = torch.empty(n, dtype=dtype, device=device)
    for start in range(0, n, _CHUNK):
        cnt = min(_CHUNK, n - start)
        if kind == "uniform":
            v = p0 + (p1 - p0) * _unit(_bits(seed, stream, start, cnt, device))
        else:  # normal: Box–Muller from two independent counters
            u1 = _unit(_bits(seed, 2 * stream + 1_000_003, start, cnt, device))
            u2 = _unit(_bits(seed, 2 * stream + 1_000_004, start, cnt, device))
            v = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
            v = p0 + p1 * v
        out[start:start + cnt] = v.to(dtype)
    return out.reshape(tuple(int(s) for s in shape))


def uniform(shape, lo, hi, *, seed, stream, device="cpu", dtype=torch.float64):
    """U(lo, hi) drawn in float64, rounded once (RNE) to ``dtype``."""
    return _fill("uniform", shape, seed, stream, device, dtype, float(lo), float(hi))


def normal(shape, mean=0.0, std=1.0, *, seed, stream, device="cpu", dtype=torch.float64):
    """N(mean, std²) drawn in float64 (Box–Muller), rounded once (RNE) to ``dtype``."""
    return _fill("normal", shape, seed, stream, device, dtype, float(mean), float(std))


# --------------------------------------------------------------------------- configs
BASE_SEED = 20260602


@dataclass(frozen=True)
class AffineConfig:
    """An ``affine_scan`` workload: ``num_seq`` independent sequences of length ``L``."""
    name: str
    num_seq: int
    L: int
    a_lo: float
    a_hi: float
    u_recipe: str            # "b*x" (b~U(0,1), x~N(0,1)) or "normal"
    h0_recipe: str           # "none" or "normal"
    seed: int
    dtype: torch.dtype = torch.float32
    kind: str = field(default="affine", init=False)

    @property
    def elements(self) -> int:
        return self.num_seq * self.L


@dataclass(frozen=True)
class SelectiveConfig:
    """A ``selective_scan_fwd`` workload (Mamba shapes)."""
    name: str
    batch: int
    d_inner: int
    N: int
    L: int
    delta_shift: float       # Δ = softplus(N(0,1) + delta_shift)
    seed: int
    dtype: torch.dtype = torch.float32
    kind: str = field(default="selective", init=False)

    @property
    def elements(self) -> int:
        return self.batch * self.d_inner * self.L


def config(k: int, **over):
    """BASELINE.json ``configs`` in file order, k = 1..5 (cfg5 takes ``L=``)."""
    seed = BASE_SEED + 1000 * k + int(over.pop("seed_offset", 0))
    if k == 1:
        c = AffineConfig("cfg1_affine_16x1024_f32", 16, 1024, 0.5, 0.99, "b*x", "none", seed)
    elif k == 2:
        c = SelectiveConfig("cfg2_selective_b2_d768_n16_l2048_f32", 2, 768, 16, 2048, -2.0, seed)
    elif k == 3:
        c = SelectiveConfig("cfg3_selective_b8_d4096_n16_l2048_bf16", 8, 4096, 16, 2048, -2.0,
                            seed, torch.bfloat16)
    elif k == 4:
        c = SelectiveConfig("cfg4_selective_b1_d1536_n16_l65536_f32", 1, 1536, 16, 65536, -4.0,
                            seed)
    elif k == 5:
        L = int(over.pop("L", 1 << 20))
        total = int(over.pop("total", 1 << 30))
        if total % L:
            raise ValueError("cfg5: total must be a multiple of L")
        c = AffineConfig(f"cfg5_affine_sweep_L{L}_f32", total // L, L, 0.9, 0.9999, "normal",
                         "normal", seed)
    else:
        raise ValueError(f"unknown config {k}")
    if over:
        c = replace(c, **over)
    return c


def make_affine_inputs(c: AffineConfig, device="cpu"):
    """Returns dict(a, u, h0): a, u [num_seq, L] in c.dtype; h0 [num_seq] fp32 or None."""
    shape = (c.num_seq, c.L)
    a = uniform(shape, c.a_lo, c.a_hi, seed=c.seed, stream=0, device=device, dtype=c.dtype)
    if c.u_recipe == "b*x":
        b = uniform(shape, 0.0, 1.0, seed=c.seed, stream=1, device=device)
        x = normal(shape, seed=c.seed, stream=2, device=device)
        u = (b * x).to(c.dtype)           # input recipe (BJ configs[0]): u_t = b_t·x_t
    else:
        u = normal(shape, seed=c.seed, stream=2, device=device, dtype=c.dtype)
    h0 = None
    if c.h0_recipe == "normal":
        h0 = normal((c.num_seq,), seed=c.seed, stream=3, device=device, dtype=torch.float32)
    return {"a": a, "u": u, "h0": h0}


def make_selective_inputs(c: SelectiveConfig, device="cpu", with_h0=False):
    """Returns dict(x, delta, A, B, C, D, h0) with BASELINE.json's distributions."""
    bdl = (c.batch, c.d_inner, c.L)
    bnl = (c.batch, c.N, c.L)
    x = normal(bdl, seed=c.seed, stream=10, device=device, dtype=c.dtype)
    z = normal(bdl, mean=c.delta_shift, seed=c.seed, stream=11, device=device)
    delta = torch.nn.functional.softplus(z).to(c.dtype)          # Δ = softplus(N(0,1) + shift)
    A = (-torch.exp(uniform((c.d_inner, c.N), -1.0, 1.0, seed=c.seed, stream=12,
                            device=device))).to(torch.float32)     # A = −exp(U(−1,1))
    B = normal(bnl, seed=c.seed, stream=13, device=device, dtype=c.dtype)
    C = normal(bnl, seed=c.seed, stream=14, device=device, dtype=c.dtype)
    D = normal((c.d_inner,), seed=c.seed, stream=15, device=device, dtype=torch.float32)
    h0 = None
    if with_h0:
        h0 = normal((c.batch, c.d_inner, c.N), seed=c.seed, stream=16, device=device,
                    dtype=torch.float32)
    return {"x": x, "delta": delta, "A": A, "B": B, "C": C, "D": D, "h0": h0}


def to_f64_numpy(t):
    """Exact widening of an fp32/bf16/fp64 tensor (any device) to a float64 numpy array."""
    if t is None:
        return None
    return t.detach().to("cpu").to(torch.float64).numpy()
