"""GPU parity tests: the CUDA path (through the C-ABI, via the ctypes binding) against the
float64 CPU oracle, element by element, on the same seeded inputs.

Tolerances are BASELINE.json's: max|err| <= 1e-4*(1+|ref|) for fp32 io and
2e-2*(1+|ref|) for bf16 io with fp32 state.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_00601_b200 as lib
from workloads import (config, make_affine_inputs, make_selective_inputs, normal, to_f64_numpy,
                       uniform)

from util import (TOL, assert_close, assert_close_all, check_affine, check_selective, gpu_affine,
                  gpu_selective, host_threads, lane_row_ok, oracle_affine, oracle_selective,
                  oracle_selective_all_rows, oracle_selective_rows, rel_err, rel_err_device)

pytestmark = pytest.mark.gpu

AFFINE_VARIANTS = [lib.AFFINE_LOOKBACK, lib.AFFINE_CTA_LOOP, lib.AFFINE_BLELLOCH,
                   lib.AFFINE_WARP_SEQ]
DTYPES = [torch.float32, torch.bfloat16]
SELECTIVE_VARIANTS = [lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW, lib.SELECTIVE_WARP_ROW_TMA]
FEW_ROWS_VARIANTS = [lib.SELECTIVE_WARP_ROW_TMA]      # what AUTO may pick for few rows x long L


def _affine_inputs(S, L, dtype, dev, seed, with_h0=True, a_lo=0.5, a_hi=0.99):
    a = uniform((S, L), a_lo, a_hi, seed=seed, stream=0, device=dev, dtype=dtype)
    u = normal((S, L), seed=seed, stream=1, device=dev, dtype=dtype)
    h0 = normal((S,), seed=seed, stream=2, device=dev, dtype=torch.float32) if with_h0 else None
    return {"a": a, "u": u, "h0": h0}


def _selective_inputs(batch, d_inner, N, L, dtype, dev, seed, with_D=True, with_h0=False,
                      delta_shift=-2.0):
    c = config(2, batch=batch, d_inner=d_inner, N=N, L=L, dtype=dtype, delta_shift=delta_shift,
               seed=seed)
    inp = make_selective_inputs(c, device=dev, with_h0=with_h0)
    if not with_D:
        inp["D"] = None
    return inp


# =============================================================== affine_scan: T1 shapes
@pytest.mark.parametrize("variant", AFFINE_VARIANTS)
@pytest.mark.parametrize("dtype", DTYPES)
def test_affine_small_and_ragged_shapes(cuda_device, variant, dtype):
    """Tiny, odd and ragged shapes spanning several tiles, vector and scalar paths."""
    Ls = [1, 2, 3, 4, 5, 8, 31, 32, 33, 127, 128, 255, 256, 257, 511, 512, 1023, 1024, 1025,
          2047, 2048, 2049, 4095, 4096, 4100, 8191, 8200, 12296]
    seed = 100
    for L in Ls:
        for S in (1, 3, 33):
            if S * L > 300_000:
                continue
            seed += 1
            inp = _affine_inputs(S, L, dtype, cuda_device, seed, with_h0=(seed % 2 == 0))
            check_affine(inp, variant, f"S={S} L={L} {dtype} v={variant}")


@pytest.mark.parametrize("variant", AFFINE_VARIANTS)
def test_affine_long_sequences_cross_many_tiles(cuda_device, variant):
    for (S, L) in [(2, 65536 + 4), (1, 262144), (5, 40000)]:
        inp = _affine_inputs(S, L, torch.float32, cuda_device, 7 + L, a_lo=0.9, a_hi=0.9999)
        check_affine(inp, variant, f"S={S} L={L}")


@pytest.mark.parametrize("variant", AFFINE_VARIANTS)
def test_affine_prefix_sum_exact_through_the_whole_carry_chain(cuda_device, variant):
    """a≡1 (BJ closed form): P never reaches 0, so every tile's carry really depends on all
    its predecessors; u in {0,1} keeps every partial sum an exact fp32 integer."""
    S, L = 2, 1 << 20
    u = (uniform((S, L), 0, 1, seed=5, stream=0, device=cuda_device) > 0.5).to(torch.float32)
    inp = {"a": torch.ones_like(u), "u": u,
           "h0": torch.tensor([3.0, -7.0], device=cuda_device)}
    h, h_last = gpu_affine(inp, variant)
    ref = inp["h0"].double()[:, None] + torch.cumsum(u.double(), dim=1)
    assert torch.equal(h.double(), ref)
    assert torch.equal(h_last.double(), ref[:, -1])
    href, _ = oracle_affine({"a": inp["a"][:, :4096], "u": u[:, :4096], "h0": inp["h0"]})
    assert np.array_equal(to_f64_numpy(h[:, :4096]), href)


@pytest.mark.parametrize("dtype", DTYPES)
def test_affine_lookback_sequences_that_divide_the_tile(cuda_device, dtype):
    """Short sequences whose length divides the look-back tile take its aligned path (every tile
    starts at a head; head / tail flags computed once per thread).  a≡1, u in {0,1}: every prefix
    is an exact small integer in the fp32 state, so h (rounded once to the io dtype) and h_last must
    match bitwise, h0 included."""
    for L in (8, 64, 512, 2048):
        S = 3 * 8192 // L * 5 + 7                       # many tiles and a ragged last one
        u = (uniform((S, L), 0, 1, seed=L, stream=0, device=cuda_device) > 0.5).to(dtype)
        h0 = (uniform((S,), 0, 1, seed=L, stream=1, device=cuda_device) * 8).floor().to(torch.float32)
        inp = {"a": torch.ones_like(u), "u": u, "h0": h0}
        h, h_last = gpu_affine(inp, lib.AFFINE_LOOKBACK)
        ref = h0.double()[:, None] + torch.cumsum(u.double(), dim=1)   # exact in the fp32 state
        assert torch.equal(h.double(), ref.to(dtype).double()), f"L={L} {dtype}"  # one RNE to io
        assert torch.equal(h_last.double(), ref[:, -1]), f"L={L} {dtype} h_last"


def test_affine_running_product_and_geometric(cuda_device):
    """u≡0 gives h0*prod(a) (a=0.5: exact powers of two until underflow); constant a,u gives
    the geometric series (BJ closed forms), here against the closed form itself."""
    L = 100
    inp = {"a": torch.full((1, L), 0.5, device=cuda_device), "u": torch.zeros((1, L), device=cuda_device),
           "h0": torch.tensor([3.0], device=cuda_device)}
    for v in AFFINE_VARIANTS:
        h, _ = gpu_affine(inp, v)
        assert np.array_equal(to_f64_numpy(h[0]), np.ldexp(3.0, -np.arange(1, L + 1)))
    L = 5000
    a0, u0, h00 = 0.999, 0.01, -1.0
    inp = {"a": torch.full((1, L), a0, device=cuda_device), "u": torch.full((1, L), u0, device=cuda_device),
           "h0": torch.tensor([h00], device=cuda_device)}
    a0f, u0f = float(np.float32(a0)), float(np.float32(u0))
    t1 = np.arange(1, L + 1, dtype=np.float64)
    ref = a0f ** t1 * h00 + u0f * (1 - a0f ** t1) / (1 - a0f)
    for v in AFFINE_VARIANTS:
        h, _ = gpu_affine(inp, v)
        assert_close(h[0], ref, torch.float32, f"geometric v={v}")


def test_affine_optional_outputs_and_empty(cuda_device):
    inp = _affine_inputs(4, 1000, torch.float32, cuda_device, 11, with_h0=False)
    h1, _ = gpu_affine(inp, want_h_last=False)
    h2, hl = gpu_affine(inp)
    assert torch.equal(h1, h2) and torch.equal(hl, h2[:, -1])
    # L == 0: h_last <- h0 (or 0); num_seq == 0: no-op
    h0 = torch.tensor([1.5, -2.5], device=cuda_device)
    e = torch.empty((2, 0), device=cuda_device)
    hl = torch.full((2,), float("nan"), device=cuda_device)
    lib.affine_scan(e, e, h0, torch.empty_like(e), hl)
    torch.cuda.synchronize()
    assert torch.equal(hl, h0)
    lib.affine_scan(e, e, None, torch.empty_like(e), hl)
    torch.cuda.synchronize()
    assert torch.equal(hl, torch.zeros_like(hl))
    z = torch.empty((0, 8), device=cuda_device)
    lib.affine_scan(z, z, None, torch.empty_like(z), None)


def test_affine_misaligned_pointers_take_the_scalar_path(cuda_device):
    """Views offset by one element break 16-byte alignment: not an error (header)."""
    S, L = 3, 1000
    for dtype in DTYPES:
        base = _affine_inputs(1, S * L + 1, dtype, cuda_device, 31, with_h0=False)
        a = base["a"].reshape(-1)[1:].reshape(S, L)
        u = base["u"].reshape(-1)[1:].reshape(S, L)
        assert a.data_ptr() % 16 != 0 and a.is_contiguous()
        inp = {"a": a, "u": u, "h0": None}
        for v in AFFINE_VARIANTS:
            hbuf = torch.empty(S * L + 1, dtype=dtype, device=cuda_device)
            h = hbuf[1:].reshape(S, L)
            hl = torch.empty(S, device=cuda_device)
            lib.affine_scan_ex(a, u, None, h, hl, v)
            torch.cuda.synchronize()
            href, hlref = oracle_affine(inp)
            assert_close(h, href, dtype, f"misaligned v={v}")
            assert_close(hl, hlref, dtype, f"misaligned h_last v={v}")


def test_affine_variants_agree_and_are_deterministic(cuda_device):
    inp = _affine_inputs(7, 50_000, torch.float32, cuda_device, 77)
    outs = []
    for v in AFFINE_VARIANTS:
        h1, hl1 = gpu_affine(inp, v)
        h2, hl2 = gpu_affine(inp, v)
        assert torch.equal(h1, h2) and torch.equal(hl1, hl2), f"variant {v} not reproducible"
        outs.append(h1)
    for o in outs[1:]:
        assert rel_err(o, to_f64_numpy(outs[0])) <= 2 * TOL[torch.float32]


def test_affine_lookback_slow_decay_carries_cross_many_tiles(cuda_device):
    """a close to 1: tile products do not underflow, so the look-back really composes AGGREGATE
    descriptors of many predecessors.  Which of them are already INCLUSIVE when a tile polls
    depends on timing, so the fp32 bracketing (and the last bits) may differ between runs: the
    look-back schedule is reproducible up to floating-point association only (include/
    affinescan.h), while both runs stay within the oracle tolerance."""
    S, L = 2, 3_000_000
    a = uniform((S, L), 0.999, 1.0, seed=91, stream=1, device=cuda_device, dtype=torch.float32)
    u = normal((S, L), seed=91, stream=2, device=cuda_device, dtype=torch.float32) * 1e-2
    inp = {"a": a, "u": u, "h0": None}
    href, hlref = oracle_affine(inp)
    h1, hl1 = gpu_affine(inp, lib.AFFINE_LOOKBACK)
    h2, hl2 = gpu_affine(inp, lib.AFFINE_LOOKBACK)
    for h, hl in ((h1, hl1), (h2, hl2)):
        assert_close(h, href, torch.float32, "slow-decay look-back")
        assert_close(hl, hlref, torch.float32, "slow-decay look-back h_last")
    hc, hlc = gpu_affine(inp, lib.AFFINE_CTA_LOOP)
    hc2, _ = gpu_affine(inp, lib.AFFINE_CTA_LOOP)
    assert torch.equal(hc, hc2)                       # fixed combine order: bitwise reproducible
    assert_close(hc, href, torch.float32, "slow-decay cta_loop")


def test_affine_split_invariance_chains_h_last_into_h0(cuda_device):
    """Eq.5 / P:93: one call over L equals two chained calls through h_last -> h0."""
    inp = _affine_inputs(4, 9000, torch.float32, cuda_device, 5)
    h, hl = gpu_affine(inp)
    m = 4096 + 8
    ha, hla = gpu_affine({"a": inp["a"][:, :m].contiguous(), "u": inp["u"][:, :m].contiguous(),
                          "h0": inp["h0"]})
    hb, hlb = gpu_affine({"a": inp["a"][:, m:].contiguous(), "u": inp["u"][:, m:].contiguous(),
                          "h0": hla})
    ref = to_f64_numpy(h)
    assert rel_err(torch.cat([ha, hb], dim=1), ref) <= 1e-5
    assert rel_err(hlb, to_f64_numpy(hl)) <= 1e-5


def test_affine_weighted_prefix_recurrence(cuda_device):
    """P:272 Eq.(10): h_t = alpha_t h_{t-1} + beta_t is affine_scan(a=alpha, u=beta)."""
    S, L = 3, 3000
    alpha = uniform((S, L), 0.2, 1.0, seed=9, stream=0, device=cuda_device, dtype=torch.float32)
    beta = normal((S, L), seed=9, stream=1, device=cuda_device, dtype=torch.float32)
    check_affine({"a": alpha, "u": beta, "h0": None}, what="weighted prefix")


def test_affine_host_api_matches_device_api(cuda_device):
    inp = _affine_inputs(5, 3000, torch.float32, cuda_device, 13)
    h, hl = gpu_affine(inp)
    a, u, h0 = inp["a"].cpu().pin_memory(), inp["u"].cpu().pin_memory(), inp["h0"].cpu()
    hh = torch.empty_like(a).pin_memory()
    hhl = torch.empty(5)
    lib.affine_scan_host(a, u, h0, hh, hhl)
    assert torch.equal(hh, h.cpu()) and torch.equal(hhl, hl.cpu())


def test_affine_host_api_pipelines_over_several_chunks(cuda_device):
    """> 16 MB per tensor: the host call splits the sequences into chunks that overlap H2D,
    kernel and D2H; with and without h0 / h_last; a repeated call reuses the staging buffers."""
    inp = _affine_inputs(45, 200000, torch.float32, cuda_device, 14, a_lo=0.9, a_hi=0.9999)
    h, hl = gpu_affine(inp)
    a, u, h0 = inp["a"].cpu().pin_memory(), inp["u"].cpu().pin_memory(), inp["h0"].cpu()
    for use_h0, want_hl in ((True, True), (False, False), (True, True)):
        hh = torch.full_like(a, float("nan")).pin_memory()
        hhl = torch.full((45,), float("nan")) if want_hl else None
        lib.affine_scan_host(a, u, h0 if use_h0 else None, hh, hhl)
        if use_h0:
            assert rel_err(hh, to_f64_numpy(h)) <= 1e-5
            assert rel_err(hhl, to_f64_numpy(hl)) <= 1e-5
        else:
            href, _ = oracle.affine_scan(to_f64_numpy(a[:3]), to_f64_numpy(u[:3]), None)
            assert_close(hh[:3], href, torch.float32, "host affine without h0")


# ================================================================ selective: T1 shapes
@pytest.mark.parametrize("dtype", DTYPES)
def test_selective_warp_row_small_and_ragged_shapes(cuda_device, dtype):
    seed = 200
    for (batch, d_inner, N, L) in [
        (1, 1, 16, 1), (1, 1, 16, 2), (2, 3, 16, 7), (1, 5, 16, 8), (2, 2, 16, 31), (1, 2, 16, 33),
        (1, 3, 16, 255), (2, 4, 16, 256), (1, 2, 16, 257), (1, 2, 16, 511), (1, 3, 16, 512),
        (1, 2, 16, 513), (2, 33, 16, 1024), (1, 31, 16, 1032), (1, 2, 16, 2047), (1, 2, 16, 2056),
        (1, 3, 1, 300), (1, 3, 4, 300), (2, 2, 33, 264), (1, 2, 64, 520), (1, 2, 17, 100),
    ]:
        seed += 1
        inp = _selective_inputs(batch, d_inner, N, L, dtype, cuda_device, seed,
                                with_D=(seed % 3 != 0), with_h0=(seed % 2 == 0))
        check_selective(inp, lib.SELECTIVE_WARP_ROW, f"warp_row {batch}x{d_inner}x{N}x{L} {dtype}")


@pytest.mark.parametrize("dtype", DTYPES)
def test_selective_warp_row_tma_small_and_ragged_shapes(cuda_device, dtype):
    """CTA-shared TMA-staged B/C tiles: one tile, ragged tails, several tiles, rows that do not
    fill the last CTA, several batches."""
    seed = 400
    vec = 4 if dtype == torch.float32 else 8
    for (batch, d_inner, L) in [
        (1, 1, vec), (1, 3, 2 * vec), (2, 5, 256), (1, 7, 512 - vec), (1, 2, 512), (2, 3, 512 + vec),
        (1, 13, 1024), (3, 37, 1536 - vec), (1, 160, 2048), (2, 150, 1000), (1, 1, 4096 + 3 * vec),
    ]:
        seed += 1
        inp = _selective_inputs(batch, d_inner, 16, L, dtype, cuda_device, seed,
                                with_D=(seed % 3 != 0), with_h0=(seed % 2 == 0))
        check_selective(inp, lib.SELECTIVE_WARP_ROW_TMA,
                        f"warp_row_tma {batch}x{d_inner}x{L} {dtype}")


@pytest.fixture
def lane_row_options():
    """Restores the lane_row tuning knobs to their defaults after a test that sets them."""
    yield
    lib.set_option(lib.OPT_LANE_ROW_G, -1)
    lib.set_option(lib.OPT_LANE_ROW_POLY16, -1)


@pytest.mark.parametrize("poly16", [0, 4])
@pytest.mark.parametrize("G", [1, 2])
@pytest.mark.parametrize("dtype", DTYPES)
def test_selective_lane_row_small_and_ragged_shapes(cuda_device, lane_row_options, dtype, G, poly16):
    """Every (lanes per row, share of exps on the fma-pipe polynomial) instantiation."""
    lib.set_option(lib.OPT_LANE_ROW_G, G)
    lib.set_option(lib.OPT_LANE_ROW_POLY16, poly16)
    seed = 300
    vec = 4 if dtype == torch.float32 else 8
    for (batch, d_inner, L) in [
        (1, 32, vec), (1, 32, 2 * vec), (2, 32, 64 - vec), (1, 64, 64), (2, 32, 64 + vec),
        (1, 96, 128), (1, 32, 192 - vec), (3, 160, 200), (1, 128, 1024), (2, 256, 520),
    ]:
        seed += 1
        inp = _selective_inputs(batch, d_inner, 16, L, dtype, cuda_device, seed,
                                with_D=(seed % 3 != 0), with_h0=(seed % 2 == 0))
        assert lane_row_ok(inp)
        check_selective(inp, lib.SELECTIVE_LANE_ROW,
                        f"lane_row G{G} poly{poly16} {batch}x{d_inner}x{L} {dtype}")


@pytest.mark.parametrize("dtype", DTYPES)
def test_selective_lane_row_polynomial_exp_slow_and_fast_decay(cuda_device, lane_row_options, dtype):
    """The fma-pipe 2^x must keep 1 - a accurate when a is close to 1 (tiny delta*|A|: long
    memory) and must flush cleanly when delta*|A| is huge (a underflows): DESIGN.md §7."""
    lib.set_option(lib.OPT_LANE_ROW_POLY16, 4)
    for G in (1, 2, 3):      # (only G = 1 evaluates part of the 2^x by the polynomial)
        lib.set_option(lib.OPT_LANE_ROW_G, G)
        for shift, a_scale in ((-7.0, 1.0), (-4.0, 0.05), (3.0, 40.0), (5.0, 400.0)):
            inp = _selective_inputs(1, 64 if G < 3 else 256, 16, 1024, dtype, cuda_device, 77,
                                    with_h0=True, delta_shift=shift)
            inp["A"] = (inp["A"] * a_scale).contiguous()
            check_selective(inp, lib.SELECTIVE_LANE_ROW,
                            f"lane_row G{G} poly4 shift{shift} Ax{a_scale} {dtype}")


def test_selective_forced_lane_row_rejects_unsupported_shapes(cuda_device):
    inp = _selective_inputs(1, 33, 16, 64, torch.float32, cuda_device, 1)
    with pytest.raises(lib.AffineScanError) as ei:
        gpu_selective(inp, lib.SELECTIVE_LANE_ROW)
    assert ei.value.status == 4
    inp = _selective_inputs(1, 32, 8, 64, torch.float32, cuda_device, 1)
    with pytest.raises(lib.AffineScanError):
        gpu_selective(inp, lib.SELECTIVE_LANE_ROW)
    with pytest.raises(lib.AffineScanError):
        gpu_selective(inp, lib.AFFINE_LOOKBACK)      # not a selective variant
    gpu_selective(inp, lib.VARIANT_AUTO)             # AUTO falls back to warp_row
    assert lib.last_variant() == lib.SELECTIVE_WARP_ROW


def test_selective_variants_agree_and_are_deterministic(cuda_device):
    inp = _selective_inputs(2, 64, 16, 1536, torch.float32, cuda_device, 21, with_h0=True)
    y1, hl1 = gpu_selective(inp, lib.SELECTIVE_WARP_ROW)
    y1b, hl1b = gpu_selective(inp, lib.SELECTIVE_WARP_ROW)
    y2, hl2 = gpu_selective(inp, lib.SELECTIVE_LANE_ROW)
    y2b, hl2b = gpu_selective(inp, lib.SELECTIVE_LANE_ROW)
    assert torch.equal(y1, y1b) and torch.equal(hl1, hl1b)
    assert torch.equal(y2, y2b) and torch.equal(hl2, hl2b)
    assert rel_err(y2, to_f64_numpy(y1)) <= 2 * TOL[torch.float32]
    assert rel_err(hl2, to_f64_numpy(hl1)) <= 2 * TOL[torch.float32]


@pytest.mark.parametrize("variant", [lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW,
                                     lib.SELECTIVE_WARP_ROW_TMA])
def test_selective_split_invariance(cuda_device, variant):
    inp = _selective_inputs(1, 32, 16, 2048, torch.float32, cuda_device, 8, with_h0=True)
    y, hl = gpu_selective(inp, variant)
    m = 1000
    first = {k: (v[..., :m].contiguous() if k in ("x", "delta", "B", "C") else v)
             for k, v in inp.items()}
    y1, hl1 = gpu_selective(first, variant)
    second = {k: (v[..., m:].contiguous() if k in ("x", "delta", "B", "C") else v)
              for k, v in inp.items()}
    second["h0"] = hl1
    y2, hl2 = gpu_selective(second, variant)
    assert rel_err(torch.cat([y1, y2], dim=2), to_f64_numpy(y)) <= 1e-5
    assert rel_err(hl2, to_f64_numpy(hl)) <= 1e-5


@pytest.mark.parametrize("variant", [lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW,
                                     lib.SELECTIVE_WARP_ROW_TMA])
def test_selective_degenerate_cases(cuda_device, variant):
    """delta≡0 holds the state (y = C·h0 + D·x); N=1-like reduction with one-hot C."""
    dev = cuda_device
    inp = _selective_inputs(1, 32, 16, 256, torch.float32, dev, 4, with_h0=True)
    inp["delta"] = torch.zeros_like(inp["delta"])
    y, hl = gpu_selective(inp, variant)
    ref = torch.einsum("bnl,bdn->bdl", inp["C"].double(), inp["h0"].double()) \
        + inp["D"].double()[None, :, None] * inp["x"].double()
    assert rel_err(y, ref.cpu().numpy()) <= 1e-5
    assert torch.equal(hl, inp["h0"])
    # one-hot C picks state n: y equals the affine scan of (exp(ΔA_n), ΔB_n x), via the oracle
    inp = _selective_inputs(1, 32, 16, 256, torch.float32, dev, 5, with_D=False)
    n = 5
    C = torch.zeros_like(inp["C"])
    C[:, n, :] = 1.0
    inp["C"] = C
    y, _ = gpu_selective(inp, variant)
    a = np.exp(to_f64_numpy(inp["delta"])[0] * to_f64_numpy(inp["A"])[:, n:n + 1])
    u = to_f64_numpy(inp["delta"])[0] * to_f64_numpy(inp["B"])[0, n][None, :] * to_f64_numpy(inp["x"])[0]
    href, _ = oracle.affine_scan(a, u, None)
    assert_close(y[0], href, torch.float32, "one-hot C")


def test_selective_optional_outputs_and_empty(cuda_device):
    inp = _selective_inputs(1, 32, 16, 128, torch.float32, cuda_device, 6)
    for v in (lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW):
        y1, _ = gpu_selective(inp, v, want_h_last=False)
        y2, _ = gpu_selective(inp, v)
        assert torch.equal(y1, y2)
    # L == 0
    e = torch.empty((1, 32, 0), device=cuda_device)
    bc = torch.empty((1, 16, 0), device=cuda_device)
    h0 = normal((1, 32, 16), seed=1, stream=0, device=cuda_device, dtype=torch.float32)
    hl = torch.full_like(h0, float("nan"))
    lib.selective_scan_fwd(e, e, inp["A"], bc, bc, None, h0, torch.empty_like(e), hl)
    torch.cuda.synchronize()
    assert torch.equal(hl, h0)


def test_selective_host_api_matches_device_api(cuda_device):
    inp = _selective_inputs(2, 64, 16, 512, torch.bfloat16, cuda_device, 17)
    y, hl = gpu_selective(inp)
    host = {k: (None if v is None else v.cpu()) for k, v in inp.items()}
    yh = torch.empty_like(host["x"]).pin_memory()
    hlh = torch.empty((2, 64, 16))
    lib.selective_scan_fwd_host(host["x"].pin_memory(), host["delta"].pin_memory(), host["A"],
                                host["B"], host["C"], host["D"], None, yh, hlh)
    assert torch.equal(yh, y.cpu()) and torch.equal(hlh, hl.cpu())


def test_selective_host_api_pipelines_over_several_chunks(cuda_device):
    """x > 16 MB per chunk boundary: batches go through the H2D || kernel || D2H pipeline in
    several chunks (the chunks may take another schedule than the whole problem would)."""
    inp = _selective_inputs(5, 64, 16, 20000, torch.float32, cuda_device, 18, with_h0=True)
    y, hl = gpu_selective(inp)
    host = {k: (None if v is None else v.cpu().pin_memory()) for k, v in inp.items()}
    yh = torch.full_like(host["x"], float("nan")).pin_memory()
    hlh = torch.full((5, 64, 16), float("nan"))
    lib.selective_scan_fwd_host(host["x"], host["delta"], host["A"], host["B"], host["C"],
                                host["D"], host["h0"], yh, hlh)
    assert rel_err(yh, to_f64_numpy(y)) <= 1e-5 and rel_err(hlh, to_f64_numpy(hl)) <= 1e-5
    yh.fill_(float("nan"))
    lib.selective_scan_fwd_host(host["x"], host["delta"], host["A"], host["B"], host["C"],
                                None, None, yh, None)
    sub = {k: (None if k in ("D", "h0") else v) for k, v in inp.items()}
    rows = [(0, 0), (2, 63), (4, 17)]
    yref, _ = oracle_selective_rows(sub, rows)
    for i, (b, d) in enumerate(rows):
        assert_close(yh[b, d], yref[i], torch.float32, "host selective without D/h0/h_last")


def test_runs_on_a_non_default_stream_and_counts_launches(cuda_device):
    inp = _selective_inputs(1, 32, 16, 256, torch.float32, cuda_device, 3)
    s = torch.cuda.Stream()
    n0 = lib.launch_count()
    with torch.cuda.stream(s):
        y, hl = gpu_selective(inp, stream=s)
    assert lib.launch_count() == n0 + 1
    yref, _ = oracle_selective(inp)
    assert_close(y, yref, torch.float32, "stream")


# ======================================================== T2: the five BASELINE configs
def test_config1_affine_fp32_full(cuda_device):
    inp = make_affine_inputs(config(1), device=cuda_device)
    for v in [lib.VARIANT_AUTO] + AFFINE_VARIANTS:
        check_affine(inp, v, f"cfg1 v={v}")
    inp2 = make_affine_inputs(config(1, seed_offset=1), device=cuda_device)
    check_affine(inp2, what="cfg1 seed+1")


def test_config2_selective_fp32_full(cuda_device):
    inp = make_selective_inputs(config(2), device=cuda_device)
    yref, hlref = oracle_selective(inp)
    for v in (lib.VARIANT_AUTO, lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW,
              lib.SELECTIVE_WARP_ROW_TMA):
        y, hl = gpu_selective(inp, v)
        assert_close(y, yref, torch.float32, f"cfg2 y v={v}")
        assert_close(hl, hlref, torch.float32, f"cfg2 h_last v={v}")


def _check_selective_every_element(inp, ref, variant, dtype, what):
    """Every y and h_last element against the oracle at BASELINE.json's per-element bound."""
    yref, hlref = ref
    y, hl = gpu_selective(inp, variant)
    assert y.numel() == yref.size and hl.numel() == hlref.size
    e1 = assert_close_all(y, yref, dtype, f"{what} y")
    e2 = assert_close_all(hl, hlref, dtype, f"{what} h_last")
    return e1, e2


def test_config3_selective_bf16_mamba_scale_every_element(cuda_device):
    """Full size (batch 8 x d_inner 4096 x L 2048 = 67 108 864 outputs), in the launch
    configuration bench.py times (AUTO -> lane_row), every element against the oracle; then
    every other schedule that accepts the shape, also on every element."""
    c = config(3)
    inp = make_selective_inputs(c, device=cuda_device)
    ref = oracle_selective_all_rows(inp)
    assert ref[0].size == c.batch * c.d_inner * c.L
    _check_selective_every_element(inp, ref, lib.VARIANT_AUTO, c.dtype, "cfg3 auto")
    assert lib.last_variant() == lib.SELECTIVE_LANE_ROW
    for v in (lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_WARP_ROW_TMA):
        _check_selective_every_element(inp, ref, v, c.dtype, f"cfg3 {lib.VARIANT_NAMES[v]}")


def test_config4_selective_long_sequence_every_element(cuda_device):
    """batch 1 x d_inner 1536 x L 65536 = 100 663 296 outputs, every element, every schedule."""
    c = config(4)
    inp = make_selective_inputs(c, device=cuda_device)
    ref = oracle_selective_all_rows(inp, rows_per_task=8)
    assert ref[0].size == c.batch * c.d_inner * c.L
    _check_selective_every_element(inp, ref, lib.VARIANT_AUTO, c.dtype, "cfg4 auto")
    auto = lib.last_variant()
    assert auto in FEW_ROWS_VARIANTS
    # SELECTIVE_CHUNKED too: the decoupled look-back BJ names for this config (plain
    # instantiation: no bias, gate or resets), 16 fp32 tiles per row
    for v in SELECTIVE_VARIANTS + [lib.SELECTIVE_CHUNKED]:
        if v != auto:
            _check_selective_every_element(inp, ref, v, c.dtype, f"cfg4 {lib.VARIANT_NAMES[v]}")


@pytest.mark.parametrize("dtype", DTYPES)
def test_selective_chunked_is_what_auto_runs_for_few_rows_and_long_L(cuda_device, dtype):
    """1 x 128 rows x L = 32 768, no bias / gate / reset: AUTO must send this to the plain
    instantiation of the chunked look-back schedule, and every element must match the oracle."""
    inp = _selective_inputs(1, 128, 16, 32768, dtype, cuda_device, seed=4242, with_h0=True)
    ref = oracle_selective_all_rows(inp, rows_per_task=8)
    _check_selective_every_element(inp, ref, lib.VARIANT_AUTO, dtype, f"auto few rows {dtype}")
    assert lib.last_variant() == lib.SELECTIVE_CHUNKED


@pytest.mark.parametrize("dtype,L", [(torch.float32, 65536), (torch.bfloat16, 131072)])
def test_selective_chunked_slow_decay_chain_longer_than_one_lookback_window(cuda_device, dtype, L):
    """Slow decay (A x 0.05, Delta = softplus(N(-4, 1)) ~ 0.02, h0 given): the product of a over a
    whole tile stays far from 0 (e^-0.9 .. e^-0.1; the carry over 33 tiles still weighs up to 1.5 %
    of the state, 150 x the tolerance), so no tile is self-contained and a tile's look-back has to fold
    AGGREGATE descriptors, and a wrong fold anywhere in the chain shows in the result (with BJ's
    fast decay a far tile's carry is ~1e-26 of the state and any fold error is invisible).  With
    ~170 tiles per row, well over the 32 a look-back window covers, the second and later windows
    run whenever a CTA gets ahead of its predecessors' INCLUSIVE publications.  Three runs: each within the parity bound of the oracle
    on every element, and within it of each other (the fold order may differ run to run; the
    header allows exactly that).  (Still slower decay, A x 0.01 with Delta ~ 1e-3, leaves BJ's
    tolerance in EVERY schedule, this one and the register-carry ones alike: fp32 rounding over a
    memory of ~1e5 steps.)"""
    inp = _selective_inputs(1, 64, 16, L, dtype, cuda_device, seed=4343, with_h0=True,
                            delta_shift=-4.0)
    inp["A"] = inp["A"] * 0.05
    ref = oracle_selective_all_rows(inp, rows_per_task=4)
    # the state really survives the whole sequence: h0's contribution at the end is not negligible
    assert float(np.abs(ref[1]).max()) > 1e-3
    outs = []
    for run in range(3):
        y, hl = gpu_selective(inp, lib.SELECTIVE_CHUNKED)
        assert_close_all(y, ref[0], dtype, f"slow decay run {run} y")
        assert_close_all(hl, ref[1], dtype, f"slow decay run {run} h_last")
        outs.append((y, hl))
    for (y, hl) in outs[1:]:
        assert rel_err(y, outs[0][0].double().cpu().numpy()) <= TOL[dtype]
        assert rel_err(hl, outs[0][1].double().cpu().numpy()) <= TOL[dtype]


def test_deterministic_option_keeps_auto_off_the_lookback_schedules(cuda_device):
    """affinescan_set_option(AFFINESCAN_OPT_DETERMINISTIC, 1): AUTO takes a register-carry schedule
    where it would have taken a decoupled look-back, results stay right and are bitwise equal run
    to run; a forced variant is not overridden; 0 restores the default choice."""
    ainp = _affine_inputs(1, 1 << 20, torch.float32, cuda_device, 99)
    sinp = _selective_inputs(1, 128, 16, 32768, torch.float32, cuda_device, seed=98)
    gpu_affine(ainp)
    assert lib.last_variant() == lib.AFFINE_LOOKBACK
    try:
        lib.set_option(lib.OPT_DETERMINISTIC, 1)
        h1, hl1 = gpu_affine(ainp)
        assert lib.last_variant() == lib.AFFINE_CTA_LOOP
        h2, hl2 = gpu_affine(ainp)
        assert torch.equal(h1, h2) and torch.equal(hl1, hl2)
        href, hlref = oracle_affine(ainp)
        assert_close(h1, href, torch.float32, "deterministic affine")
        y1, s1 = gpu_selective(sinp)
        assert lib.last_variant() == lib.SELECTIVE_WARP_ROW_TMA
        y2, s2 = gpu_selective(sinp)
        assert torch.equal(y1, y2) and torch.equal(s1, s2)
        gpu_affine(ainp, lib.AFFINE_LOOKBACK)
        assert lib.last_variant() == lib.AFFINE_LOOKBACK
    finally:
        lib.set_option(lib.OPT_DETERMINISTIC, 0)
    gpu_selective(sinp)
    assert lib.last_variant() == lib.SELECTIVE_CHUNKED


def test_config5_affine_bandwidth_sweep_every_element(cuda_device):
    """2^30 elements re-segmented into L = 2^10 .. 2^20.  ALL 2^30 outputs of each of the six
    lengths are compared with the oracle, streamed slab by slab (2^24 elements, whole sequences)
    so no 8 GB float64 array is materialised; the slabs run on several host
    threads.  Also the forced look-back schedule on the longest and one short length."""
    from concurrent.futures import ThreadPoolExecutor
    total = 1 << 30
    slab = 1 << 24
    flat = make_affine_inputs(config(5, L=total, total=total), device=cuda_device)
    a_flat, u_flat = flat["a"].reshape(-1), flat["u"].reshape(-1)
    h0_all = normal((1 << 20,), seed=config(5).seed, stream=3, device=cuda_device,
                    dtype=torch.float32)
    runs = [(logL, lib.VARIANT_AUTO) for logL in (10, 12, 14, 16, 18, 20)]
    runs += [(20, lib.AFFINE_LOOKBACK), (12, lib.AFFINE_LOOKBACK)]
    outs = []
    for logL, variant in runs:
        L = 1 << logL
        S = total // L
        h = torch.full((S, L), float("nan"), dtype=torch.float32, device=cuda_device)
        hl = torch.full((S,), float("nan"), dtype=torch.float32, device=cuda_device)
        lib.affine_scan_ex(a_flat.view(S, L), u_flat.view(S, L), h0_all[:S], h, hl, variant)
        torch.cuda.synchronize()
        if variant == lib.VARIANT_AUTO:
            # fp32 io: up to 2048 steps one single-warp CTA per sequence; longer
            # ones a CTA each while they fill four waves (r03: whatever their length); else the
            # persistent look-back stream
            sms = torch.cuda.get_device_properties(cuda_device).multi_processor_count
            want = (lib.AFFINE_CTA_LOOP if L <= 2048 or S >= 16 * sms else lib.AFFINE_LOOKBACK)
            assert lib.last_variant() == want
        outs.append((L, S, variant, h, hl))
    h0_host = h0_all.double().cpu().numpy()

    def check_slab(i):
        s0, s1 = i * slab, (i + 1) * slab
        a64 = a_flat[s0:s1].double().cpu().numpy()
        u64 = u_flat[s0:s1].double().cpu().numpy()
        worst = {}
        for (L, S, variant, h, hl) in outs:
            q0, q1 = s0 // L, s1 // L                    # whole sequences: slab % L == 0
            href, hlref = oracle.affine_scan(a64.reshape(-1, L), u64.reshape(-1, L), h0_host[q0:q1])
            e = rel_err_device(h[q0:q1], href)
            e2 = rel_err_device(hl[q0:q1], hlref)
            worst[(L, variant)] = max(e, e2)
        return worst

    compared = 0
    with ThreadPoolExecutor(min(8, host_threads())) as pool:
        for worst in pool.map(check_slab, range(total // slab)):
            compared += slab
            for (L, variant), e in worst.items():
                assert e <= TOL[torch.float32], \
                    f"cfg5 L={L} variant {variant}: max|err|/(1+|ref|) = {e:.3e}"
    assert compared == total


# ============================================================ seeded random shapes (fuzz)
@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_every_variant_against_the_oracle(cuda_device, seed):
    """Seeded random small shapes (ragged L, odd row counts, optional D / h0) through every
    schedule that accepts them; outputs are NaN-prefilled, so an unwritten element fails."""
    rng = np.random.default_rng(seed)
    for _ in range(6):
        dtype = DTYPES[int(rng.integers(2))]
        vec = 4 if dtype == torch.float32 else 8
        batch = int(rng.integers(1, 4))
        L = int(rng.integers(1, 90)) * vec
        d_inner = int(rng.integers(1, 70))
        inp = _selective_inputs(batch, d_inner, 16, L, dtype, cuda_device, int(rng.integers(1 << 20)),
                                with_D=bool(rng.integers(2)), with_h0=bool(rng.integers(2)))
        for v in (lib.VARIANT_AUTO, lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_WARP_ROW_TMA):
            check_selective(inp, v, f"fuzz {batch}x{d_inner}x{L} {dtype} v{v}")
        d32 = 32 * int(rng.integers(1, 4))
        inp = _selective_inputs(batch, d32, 16, L, dtype, cuda_device, int(rng.integers(1 << 20)),
                                with_D=bool(rng.integers(2)), with_h0=bool(rng.integers(2)))
        check_selective(inp, lib.SELECTIVE_LANE_ROW, f"fuzz lane_row {batch}x{d32}x{L} {dtype}")
        S, La = int(rng.integers(1, 40)), int(rng.integers(1, 9000))
        ainp = _affine_inputs(S, La, dtype, cuda_device, int(rng.integers(1 << 20)),
                              with_h0=bool(rng.integers(2)))
        for v in [lib.VARIANT_AUTO] + AFFINE_VARIANTS:
            check_affine(ainp, v, f"fuzz affine {S}x{La} {dtype} v{v}")


def test_release_cache_then_calls_still_work(cuda_device):
    """affinescan_release_cache frees scratch, staging buffers and the host-pipeline streams;
    the next calls re-create what they need."""
    inp = _affine_inputs(3, 20000, torch.float32, cuda_device, 41)
    h, hl = gpu_affine(inp, lib.AFFINE_LOOKBACK)
    a, u = inp["a"].cpu().pin_memory(), inp["u"].cpu().pin_memory()
    hh = torch.empty_like(a).pin_memory()
    lib.affine_scan_host(a, u, inp["h0"].cpu(), hh, None)
    lib.release_cache()
    h2, hl2 = gpu_affine(inp, lib.AFFINE_LOOKBACK)
    hh2 = torch.empty_like(a).pin_memory()
    lib.affine_scan_host(a, u, inp["h0"].cpu(), hh2, None)
    assert torch.equal(h, h2) and torch.equal(hl, hl2) and torch.equal(hh, hh2)


def test_scratch_cache_is_bounded_keyed_by_stream_id_and_skips_the_backward(cuda_device):
    """The look-back descriptors are cached per (device, stream id): (i) 80 short-lived streams,
    each destroyed after its call, leave at most 64 cached buffers (least recently used freed in
    stream order) and every result stays right, including the streams that inherit a recycled
    handle; (ii) selective_scan_bwd takes its large workspace per call and caches nothing."""
    lib.release_cache()
    assert lib.cached_scratch_buffers() == 0
    inp = _affine_inputs(2, 50000, torch.float32, cuda_device, 77)
    href, hlref = oracle_affine(inp)
    outs = []
    for i in range(80):
        s = torch.cuda.Stream(device=cuda_device)
        s.wait_stream(torch.cuda.current_stream())
        h = torch.full_like(inp["a"], float("nan"))
        hl = torch.full((2,), float("nan"), device=cuda_device)
        lib.affine_scan_ex(inp["a"], inp["u"], inp["h0"], h, hl, lib.AFFINE_LOOKBACK, stream=s)
        outs.append((h, hl))
        del s                                   # handle goes back to the driver while work may run
    torch.cuda.synchronize()
    n = lib.cached_scratch_buffers()
    assert 1 <= n <= 64, n
    for (h, hl) in outs[::7] + outs[-3:]:
        assert_close(h, href, torch.float32, "many streams h")
        assert_close(hl, hlref, torch.float32, "many streams h_last")
    # (ii) the backward pass leaves the cache as it found it
    c = config(2, batch=1, d_inner=64, N=16, L=256, dtype=torch.float32, seed=5)
    sel = make_selective_inputs(c, device=cuda_device)
    dy = torch.ones_like(sel["x"])
    dx = torch.empty_like(sel["x"])
    lib.selective_scan_bwd(sel["x"], sel["delta"], sel["A"], sel["B"], sel["C"], sel["D"], None, dy,
                           None, dx, None, None, None, None, None, None, workspace=None)
    torch.cuda.synchronize()
    assert lib.cached_scratch_buffers() == n
    assert bool(torch.isfinite(dx).all())
    lib.release_cache()
    assert lib.cached_scratch_buffers() == 0
