"""GPU parity tests of the rows SURVEY §8(f) adds to the hot path: the fused softplus/bias
prologue and silu(z) gate (f1), resets / packed variable-length sequences (f2) and the
structured-A fast paths (f5), each against the float64 oracle on the same seeded inputs, in
every selective schedule; plus the host-layer promises of §8(b): CUDA-graph capture and
concurrent calls on different streams.
"""
import threading

import numpy as np
import pytest
import torch

import oracle
import paper_2606_00601_b200 as lib
from workloads import config, make_selective_inputs, normal, to_f64_numpy, uniform

from util import TOL, assert_close, assert_close_all, gpu_selective, oracle_selective, rel_err

pytestmark = pytest.mark.gpu

DTYPES = [torch.float32, torch.bfloat16]
VARIANTS = [lib.SELECTIVE_WARP_ROW, lib.SELECTIVE_LANE_ROW, lib.SELECTIVE_WARP_ROW_TMA,
            lib.SELECTIVE_CHUNKED]


def _inputs(batch, d_inner, L, dtype, dev, seed, with_h0=True, N=16):
    c = config(2, batch=batch, d_inner=d_inner, N=N, L=L, dtype=dtype, seed=seed)
    return make_selective_inputs(c, device=dev, with_h0=with_h0)


def _ext_extras(inp, seed, dev, with_z=True, with_bias=True, resets=()):
    x = inp["x"]
    batch, d_inner, L = x.shape
    z = normal(x.shape, std=2.0, seed=seed, stream=20, device=dev, dtype=x.dtype) if with_z else None
    bias = normal((d_inner,), mean=-1.0, seed=seed, stream=21, device=dev, dtype=torch.float32) \
        if with_bias else None
    reset = None
    if resets:
        reset = torch.zeros((batch, L), dtype=torch.uint8, device=dev)
        for (b, t) in resets:
            if b < batch and t < L:
                reset[b, t] = 1
    return z, bias, reset


def gpu_ext(inp, z, bias, reset, softplus, variant=lib.VARIANT_AUTO, a_structure=lib.A_GENERAL):
    x = inp["x"]
    batch, d_inner, _ = x.shape
    N = inp["A"].shape[1]
    y = torch.full_like(x, float("nan"))
    hl = torch.full((batch, d_inner, N), float("nan"), dtype=torch.float32, device=x.device)
    lib.selective_scan_fwd_ext(x, inp["delta"], inp["A"], inp["B"], inp["C"], inp.get("D"), z, bias,
                               reset, inp.get("h0"), y, hl, softplus, a_structure, variant)
    torch.cuda.synchronize()
    return y, hl


def oracle_ext(inp, z, bias, reset, softplus):
    f = to_f64_numpy
    return oracle.selective_scan_fwd_ext(f(inp["x"]), f(inp["delta"]), f(inp["A"]), f(inp["B"]),
                                         f(inp["C"]), f(inp.get("D")), f(z), f(bias), f(reset),
                                         f(inp.get("h0")), softplus)


def _raw_delta(inp, seed, dev):
    """Pre-softplus delta: N(0,1) - 2 in the io dtype (BJ's recipe before the softplus)."""
    x = inp["x"]
    return normal(x.shape, mean=-2.0, seed=seed, stream=22, device=dev, dtype=x.dtype)


# ----------------------------------------------------------- f1: softplus/bias + silu(z) gate
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dtype", DTYPES)
def test_gated_softplus_every_schedule(cuda_device, dtype, variant):
    vec = 4 if dtype == torch.float32 else 8
    seed = 700
    for (batch, d_inner, L) in [(1, 32, vec), (2, 64, 520), (1, 96, 1024 + 2 * vec), (3, 32, 2048)]:
        for (with_z, with_bias, softplus) in [(True, True, True), (False, True, True),
                                              (True, False, False), (False, True, False)]:
            seed += 1
            inp = _inputs(batch, d_inner, L, dtype, cuda_device, seed, with_h0=(seed % 2 == 0))
            if softplus:
                inp["delta"] = _raw_delta(inp, seed, cuda_device)
            z, bias, _ = _ext_extras(inp, seed, cuda_device, with_z, with_bias)
            if not softplus and bias is not None:
                bias = bias.abs() * 0.05            # keep delta + bias positive (a in (0,1))
            y, hl = gpu_ext(inp, z, bias, None, softplus, variant)
            yref, hlref = oracle_ext(inp, z, bias, None, softplus)
            what = f"gated v{variant} {dtype} {batch}x{d_inner}x{L} z{with_z} b{with_bias} sp{softplus}"
            assert_close(y, yref, dtype, what + " y")
            assert_close(hl, hlref, dtype, what + " h_last")


def test_gated_entry_point_equals_ext_and_the_unfused_composition(cuda_device):
    """selective_scan_fwd_gated == ext(softplus, bias, z); and == plain kernel fed
    softplus(raw + bias) with the gate applied afterwards (the two HBM passes it saves)."""
    dev = cuda_device
    inp = _inputs(2, 64, 1024, torch.float32, dev, 31)
    raw = _raw_delta(inp, 31, dev)
    z, bias, _ = _ext_extras(inp, 31, dev)
    y = torch.empty_like(inp["x"])
    hl = torch.empty((2, 64, 16), device=dev)
    lib.selective_scan_fwd_gated(inp["x"], raw, bias, inp["A"], inp["B"], inp["C"], inp["D"], z,
                                 inp["h0"], y, hl)
    torch.cuda.synchronize()
    y2, hl2 = gpu_ext({**inp, "delta": raw}, z, bias, None, True)
    assert torch.equal(y, y2) and torch.equal(hl, hl2)
    delta = torch.nn.functional.softplus((raw + bias[None, :, None]).double()).float()
    y3, hl3 = gpu_selective({**inp, "delta": delta})
    y3 = (y3.double() * torch.nn.functional.silu(z.double())).float()
    # the fused softplus runs on MUFU.EX2/LG2 (~1e-6 relative in Delta); half of BJ's bound
    assert rel_err(y, to_f64_numpy(y3)) <= 5e-5 and rel_err(hl, to_f64_numpy(hl3)) <= 5e-5


def test_softplus_extremes(cuda_device):
    """Large raw delta (softplus -> identity) and very negative (-> exp, tiny Delta keeps full
    relative accuracy so slow channels keep their memory)."""
    dev = cuda_device
    for shift in (-12.0, -6.0, 3.0, 25.0):
        inp = _inputs(1, 32, 512, torch.float32, dev, 41)
        inp["delta"] = normal(inp["x"].shape, mean=shift, std=0.5, seed=41, stream=22, device=dev,
                              dtype=torch.float32)
        if shift > 0:
            inp["A"] = (inp["A"] * 0.02).contiguous()      # keep exp(delta*A) away from underflow
        for v in (lib.SELECTIVE_LANE_ROW, lib.SELECTIVE_WARP_ROW_TMA, lib.SELECTIVE_WARP_ROW):
            y, hl = gpu_ext(inp, None, None, None, True, v)
            yref, hlref = oracle_ext(inp, None, None, None, True)
            assert_close(y, yref, torch.float32, f"softplus shift {shift} v{v} y")
            assert_close(hl, hlref, torch.float32, f"softplus shift {shift} v{v} h_last")


# ------------------------------------------------- f2: resets / packed variable-length sequences
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dtype", DTYPES)
def test_resets_every_schedule(cuda_device, dtype, variant):
    vec = 4 if dtype == torch.float32 else 8
    seed = 800
    for (batch, d_inner, L, resets) in [
        (1, 32, 64, [(0, 0)]),
        (2, 32, 1024, [(1, 1), (1, 2), (1, 500), (0, 1023)]),
        (2, 64, 2048 + vec, [(0, 384), (0, 383), (1, 768), (1, 2048 + vec - 1), (0, 31), (1, 32)]),
        (1, 32, 4096, [(0, t) for t in range(0, 4096, 97)]),
    ]:
        seed += 1
        inp = _inputs(batch, d_inner, L, dtype, cuda_device, seed)
        _, _, reset = _ext_extras(inp, seed, cuda_device, False, False, resets)
        y, hl = gpu_ext(inp, None, None, reset, False, variant)
        yref, hlref = oracle_ext(inp, None, None, reset, False)
        what = f"reset v{variant} {dtype} {batch}x{d_inner}x{L}"
        assert_close(y, yref, dtype, what + " y")
        assert_close(hl, hlref, dtype, what + " h_last")


def test_reset_equals_independent_calls_and_cu_seqlens_helper(cuda_device):
    """One packed call over three sequences == three separate calls (each from h = 0); the mask
    comes from affinescan_reset_mask_from_cu_seqlens."""
    dev = cuda_device
    L = 3000
    inp = _inputs(1, 64, L, torch.float32, dev, 51, with_h0=False)
    starts = [0, 1000, 1776]
    cu = torch.tensor(starts + [L + 5, -1], dtype=torch.int32, device=dev)   # out-of-range ignored
    reset = torch.full((1, L), 7, dtype=torch.uint8, device=dev)
    lib.reset_mask_from_cu_seqlens(cu, reset[0])
    torch.cuda.synchronize()
    expect = torch.zeros(L, dtype=torch.uint8)
    expect[starts] = 1
    assert torch.equal(reset[0].cpu(), expect)
    for v in (lib.VARIANT_AUTO, lib.SELECTIVE_LANE_ROW, lib.SELECTIVE_WARP_ROW_TMA):
        y, hl = gpu_ext(inp, None, None, reset, False, v)
        for lo, hi in zip(starts, starts[1:] + [L]):
            piece = {k: (t[..., lo:hi].contiguous() if k in ("x", "delta", "B", "C") else t)
                     for k, t in inp.items()}
            yp, hp = gpu_selective(piece, v)
            assert rel_err(y[..., lo:hi], to_f64_numpy(yp)) <= 1e-5
        assert rel_err(hl, to_f64_numpy(hp)) <= 1e-5


def test_everything_fused_at_once_and_host_entry_point(cuda_device):
    dev = cuda_device
    for dtype in DTYPES:
        inp = _inputs(2, 64, 1536, dtype, dev, 61)
        inp["delta"] = _raw_delta(inp, 61, dev)
        z, bias, reset = _ext_extras(inp, 61, dev, True, True, [(0, 5), (1, 700), (1, 701)])
        yref, hlref = oracle_ext(inp, z, bias, reset, True)
        for v in VARIANTS:
            y, hl = gpu_ext(inp, z, bias, reset, True, v)
            assert_close(y, yref, dtype, f"all-fused v{v} {dtype} y")
            assert_close(hl, hlref, dtype, f"all-fused v{v} {dtype} h_last")
        host = {k: (None if t is None else t.cpu().pin_memory()) for k, t in inp.items()}
        yh = torch.full_like(host["x"], float("nan")).pin_memory()
        hlh = torch.full((2, 64, 16), float("nan"))
        lib.selective_scan_fwd_ext_host(host["x"], host["delta"], host["A"], host["B"], host["C"],
                                        host["D"], z.cpu(), bias.cpu(), reset.cpu(), host["h0"], yh,
                                        hlh, True)
        assert_close(yh, yref, dtype, f"all-fused host {dtype} y")
        assert_close(hlh, hlref, dtype, f"all-fused host {dtype} h_last")


# ----------------------------------------------------------- lane_row balanced grid (mix)
@pytest.mark.parametrize("dtype", DTYPES)
def test_lane_row_balanced_grid_partial_ctas_rounds_and_fused_steps(cuda_device, dtype):
    """OPT_LANE_ROW_G = 3: one CTA per SM, three 16-row warps and one 8-row warp per
    sub-partition, B/C staged once per CTA by a producer warp.  Shapes: a CTA's 224 rows
    straddling two batches, a last CTA with fewer rows than warps, more rows than one round of
    CTAs holds (with few and with many tiles, so that every barrier is re-armed after use), L not a
    multiple of the staged tile; plain, gated and reset forms."""
    sms = torch.cuda.get_device_properties(cuda_device).multi_processor_count
    vec = 4 if dtype == torch.float32 else 8
    lib.set_option(lib.OPT_LANE_ROW_G, 3)
    try:
        seed = 900
        for (batch, d_inner, L) in [(1, 224, 64), (3, 256, 3 * 32 + vec), (2, 480, 520),
                                    (1, 224 * sms + 96, 40), (5, 1024, 96 + vec),
                                    (2, 224 * sms // 2 + 160, 8 * 64 + vec)]:
            for mode in ("plain", "gated", "reset"):
                seed += 1
                inp = _inputs(batch, d_inner, L, dtype, cuda_device, seed, with_h0=(seed % 2 == 0))
                z = bias = reset = None
                softplus = False
                if mode == "gated":
                    inp["delta"] = _raw_delta(inp, seed, cuda_device)
                    z, bias, _ = _ext_extras(inp, seed, cuda_device)
                    softplus = True
                elif mode == "reset":
                    _, _, reset = _ext_extras(inp, seed, cuda_device, False, False,
                                              resets=[(0, 0), (0, L // 2), (batch - 1, L - 1), (1, 7)])
                y, hl = gpu_ext(inp, z, bias, reset, softplus, lib.SELECTIVE_LANE_ROW)
                assert lib.last_variant() == lib.SELECTIVE_LANE_ROW
                yref, hlref = oracle_ext(inp, z, bias, reset, softplus)
                what = f"lane_mix {mode} {dtype} {batch}x{d_inner}x{L}"
                assert_close(y, yref, dtype, what + " y")
                assert_close(hl, hlref, dtype, what + " h_last")
        # narrower than one CTA's 224 rows: the balanced grid does not apply
        inp = _inputs(2, 192, 64, dtype, cuda_device, 7)
        with pytest.raises(lib.AffineScanError):
            gpu_ext(inp, None, None, None, False, lib.SELECTIVE_LANE_ROW)
    finally:
        lib.set_option(lib.OPT_LANE_ROW_G, -1)


# --------------------------------------------------------------- f5: structured-A fast paths
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("structure", [lib.A_SCALAR_PER_ROW, lib.A_POWERS])
def test_structured_A_fast_paths_match_the_general_oracle(cuda_device, dtype, structure):
    """The fast paths read A[d,0] only; the oracle is the GENERAL one on the full structured A."""
    dev = cuda_device
    vec = 4 if dtype == torch.float32 else 8
    seed = 900
    for (batch, d_inner, L) in [(1, 32, vec), (2, 64, 520), (2, 160, 2048), (1, 4736, 256)]:
        seed += 1
        inp = _inputs(batch, d_inner, L, dtype, dev, seed, with_h0=(seed % 2 == 0))
        a0 = -torch.exp(uniform((d_inner,), -1.0, 0.5, seed=seed, stream=30, device=dev,
                                dtype=torch.float32))
        if structure == lib.A_SCALAR_PER_ROW:
            inp["A"] = a0[:, None].repeat(1, 16).contiguous()
        else:
            a0 = a0 * 0.25                                   # (n+1)*A0 up to 16*A0
            inp["A"] = (a0[:, None] * torch.arange(1, 17, device=dev, dtype=torch.float32)[None, :]
                        ).contiguous()
        yref, hlref = oracle_selective(inp)
        for v in (lib.VARIANT_AUTO, lib.SELECTIVE_LANE_ROW, lib.SELECTIVE_WARP_ROW):
            y, hl = gpu_ext(inp, None, None, None, False, v, structure)
            assert_close(y, yref, dtype, f"A-structure {structure} v{v} {dtype} {batch}x{d_inner}x{L} y")
            assert_close(hl, hlref, dtype, f"A-structure {structure} v{v} h_last")
        # fused with the gate and a reset as well
        z, bias, reset = _ext_extras(inp, seed, dev, True, False, [(0, L // 2)])
        y, hl = gpu_ext(inp, z, None, reset, False, lib.SELECTIVE_LANE_ROW, structure)
        yref2, hlref2 = oracle_ext(inp, z, None, reset, False)
        assert_close(y, yref2, dtype, f"A-structure {structure} fused y")
        assert_close(hl, hlref2, dtype, f"A-structure {structure} fused h_last")


def test_unknown_structure_or_variant_is_rejected(cuda_device):
    inp = _inputs(1, 32, 64, torch.float32, cuda_device, 3)
    with pytest.raises(lib.AffineScanError) as ei:
        gpu_ext(inp, None, None, None, False, lib.VARIANT_AUTO, 7)
    assert ei.value.status == 4


# --------------------------------------------------- §8(b): graph capture, concurrent streams
def test_device_calls_capture_in_a_cuda_graph_and_replay_bitwise(cuda_device):
    """Both device entry points, including the schedules that use library scratch (decoupled
    look-back), captured in one CUDA graph and replayed: results equal the eager calls."""
    dev = cuda_device
    sel = _inputs(2, 64, 4096, torch.float32, dev, 71)
    a = uniform((3, 40000), 0.5, 0.99, seed=71, stream=0, device=dev, dtype=torch.float32)
    u = normal((3, 40000), seed=71, stream=1, device=dev, dtype=torch.float32)
    h0 = normal((3,), seed=71, stream=2, device=dev, dtype=torch.float32)

    def run(outs):
        y, hl, h, hla, yc, hlc = outs
        lib.selective_scan_fwd(sel["x"], sel["delta"], sel["A"], sel["B"], sel["C"], sel["D"],
                               sel["h0"], y, hl)
        lib.affine_scan_ex(a, u, h0, h, hla, lib.AFFINE_LOOKBACK)
        lib.selective_scan_fwd_ex(sel["x"], sel["delta"], sel["A"], sel["B"], sel["C"], sel["D"],
                                  sel["h0"], yc, hlc, lib.SELECTIVE_CHUNKED)

    def fresh():
        return (torch.full_like(sel["x"], float("nan")), torch.full((2, 64, 16), float("nan"), device=dev),
                torch.full_like(a, float("nan")), torch.full((3,), float("nan"), device=dev),
                torch.full_like(sel["x"], float("nan")), torch.full((2, 64, 16), float("nan"), device=dev))

    eager = fresh()
    run(eager)
    torch.cuda.synchronize()
    captured = fresh()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        run(fresh())                     # warm-up on the capture stream (module load, smem attr)
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=s):
            run(captured)
    for rep in range(3):
        for t in captured:
            t.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(captured[0], eager[0]) and torch.equal(captured[1], eager[1]), rep
        # look-back schedules: reproducible up to association order (header)
        assert rel_err(captured[2], to_f64_numpy(eager[2])) <= 1e-5
        assert rel_err(captured[3], to_f64_numpy(eager[3])) <= 1e-5
        assert rel_err(captured[4], to_f64_numpy(eager[4])) <= 1e-5
        assert rel_err(captured[5], to_f64_numpy(eager[5])) <= 1e-5


def test_two_host_threads_on_two_streams_run_concurrently(cuda_device):
    """Device and `_host` entry points from two threads on two streams at the same time."""
    dev = cuda_device
    results, errors = {}, []

    def worker(i):
        try:
            torch.cuda.set_device(dev)
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                inp = _inputs(2, 64, 6000 + 8 * i, torch.float32, dev, 80 + i)
                aa = uniform((2, 300000), 0.9, 0.9999, seed=80 + i, stream=0, device=dev,
                             dtype=torch.float32)
                uu = normal((2, 300000), seed=80 + i, stream=1, device=dev, dtype=torch.float32)
                s.synchronize()
                outs = []
                for rep in range(4):
                    y, hl = gpu_selective(inp, stream=s)
                    h = torch.empty_like(aa)
                    hla = torch.empty(2, device=dev)
                    lib.affine_scan_ex(aa, uu, None, h, hla, lib.AFFINE_LOOKBACK, s)
                    host = {k: (None if t is None else t.cpu()) for k, t in inp.items()}
                    yh = torch.empty_like(host["x"])
                    lib.selective_scan_fwd_host(host["x"], host["delta"], host["A"], host["B"],
                                                host["C"], host["D"], host["h0"], yh, None, s)
                    s.synchronize()
                    outs.append((y.cpu(), h.cpu(), yh))
                results[i] = (inp, aa, uu, outs)
        except Exception as e:           # noqa: BLE001
            errors.append(e)

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for i in range(2):
        inp, aa, uu, outs = results[i]
        yref, _ = oracle_selective(inp)
        href, _ = oracle.affine_scan(to_f64_numpy(aa), to_f64_numpy(uu), None)
        for (y, h, yh) in outs:
            assert_close(y, yref, torch.float32, f"thread {i} y")
            assert_close(yh, yref, torch.float32, f"thread {i} host y")
            assert_close(h, href, torch.float32, f"thread {i} affine h")


def test_persistent_kernels_on_two_streams_share_the_gpu_without_deadlock(cuda_device):
    """The persistent look-back stream and the balanced lane grid launch one or two CTAs per SM and
    wait inside the kernel (tile descriptors, mbarriers).  Two such launches on two streams compete
    for the SMs, so part of each grid may not be resident while the rest runs: tickets are handed
    to running CTAs only, so both must finish, with the same bits as when run alone."""
    dev = cuda_device
    S, L = 3, 6_000_000
    a = uniform((S, L), 0.99, 1.0, seed=5, stream=1, device=dev, dtype=torch.float32)
    u = normal((S, L), seed=5, stream=2, device=dev, dtype=torch.float32)
    inp = _inputs(4, 4096, 512, torch.bfloat16, dev, 11, with_h0=False)
    def affine(stream):
        h = torch.empty_like(a); hl = torch.empty(S, device=dev)
        lib.affine_scan_ex(a, u, None, h, hl, lib.AFFINE_CTA_LOOP if stream is None else lib.AFFINE_LOOKBACK,
                           stream)
        return h, hl
    def selective(stream):
        y = torch.empty_like(inp["x"]); hl = torch.empty((4, 4096, 16), device=dev)
        lib.selective_scan_fwd_ex(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"], inp["D"], None,
                                  y, hl, lib.SELECTIVE_LANE_ROW, stream)
        return y, hl
    lib.set_option(lib.OPT_LANE_ROW_G, 3)
    try:
        s1, s2 = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        torch.cuda.synchronize()
        h_alone, _ = affine(s1); torch.cuda.synchronize()
        y_alone, hl_alone = selective(s2); torch.cuda.synchronize()
        outs = []
        for _ in range(4):                       # interleave launches on the two streams
            outs.append((affine(s1), selective(s2), affine(s2), selective(s1)))
        torch.cuda.synchronize()
        h_ref, _ = affine(None); torch.cuda.synchronize()
        for (ha, _), (ys, hls), (hb, _), (yt, hlt) in outs:
            for h in (ha, hb):                   # look-back: reproducible up to fp association
                assert rel_err(h, to_f64_numpy(h_ref)) <= 1e-4 and rel_err(h, to_f64_numpy(h_alone)) <= 1e-4
            assert torch.equal(ys, y_alone) and torch.equal(hls, hl_alone)
            assert torch.equal(yt, y_alone) and torch.equal(hlt, hl_alone)
    finally:
        lib.set_option(lib.OPT_LANE_ROW_G, -1)



def test_host_entry_point_with_L_zero_writes_h_last(cuda_device):
    """the `_host` form promises the same computation as the device form."""
    inp = _inputs(2, 32, 8, torch.float32, cuda_device, 5)
    h0 = inp["h0"].cpu()
    e = torch.empty((2, 32, 0))
    bc = torch.empty((2, 16, 0))
    hl = torch.full((2, 32, 16), float("nan"))
    lib.selective_scan_fwd_host(e, e, inp["A"].cpu(), bc, bc, None, h0, torch.empty_like(e), hl)
    assert torch.equal(hl, h0)
    lib.selective_scan_fwd_host(e, e, inp["A"].cpu(), bc, bc, None, None, torch.empty_like(e), hl)
    assert torch.equal(hl, torch.zeros_like(hl))


def test_lookback_many_tiles_with_a_close_to_one(cuda_device):
    """with a ~ 1 the tile products never underflow, so every look-back really folds
    its predecessors' aggregates; runs agree with the oracle (and with each other up to the
    association order the header allows)."""
    dev = cuda_device
    # product over a 4096-element tile ~0.3, over a 32-tile look-back window ~1e-17: never 0 in
    # fp32 inside a window (memory ~3000 steps keeps fp32 itself well inside the 1e-4 bound)
    a = uniform((2, 1 << 19), 0.9995, 0.9999, seed=91, stream=0, device=dev, dtype=torch.float32)
    u = normal((2, 1 << 19), std=0.01, seed=91, stream=1, device=dev, dtype=torch.float32)
    h0 = torch.tensor([1.0, -2.0], device=dev)
    href, hlref = oracle.affine_scan(to_f64_numpy(a), to_f64_numpy(u), to_f64_numpy(h0))
    outs = []
    for _ in range(3):
        h = torch.full_like(a, float("nan"))
        hl = torch.full((2,), float("nan"), device=dev)
        lib.affine_scan_ex(a, u, h0, h, hl, lib.AFFINE_LOOKBACK)
        torch.cuda.synchronize()
        assert_close(h, href, torch.float32, "lookback a~1 h")
        assert_close(hl, hlref, torch.float32, "lookback a~1 h_last")
        outs.append(h)
    assert rel_err(outs[1], to_f64_numpy(outs[0])) <= 1e-5


# ------------------------------------------------ f4: L-sharded scan, ranks emulated on one GPU
@pytest.mark.parametrize("dtype", DTYPES)
def test_l_sharded_scan_primitives_ranks_emulated_sequentially(cuda_device, dtype):
    """The CUDA entry points of the multi-GPU L-sharded scan (slice aggregate, compose carry,
    final scan with h0 = h_in) with the R ranks run one after another on one GPU and the
    all-gather replaced by torch.stack: equals the unsharded oracle.  (The torch.distributed
    plumbing itself is covered by tests/test_lshard_gloo.py on CPU.)"""
    from paper_2606_00601_b200.sharding import shard_range_aligned
    dev = cuda_device
    vec = 4 if dtype == torch.float32 else 8
    for (batch, d_inner, L, R) in [(2, 64, 2048, 4), (1, 4736, 512, 2), (2, 33, 1000 + vec, 3)]:
        inp = _inputs(batch, d_inner, L, dtype, dev, 1234 + L)
        yref, hlref = oracle_selective(inp)
        spans = [shard_range_aligned(L, r, R, vec) for r in range(R)]
        slices = [{k: (t[..., lo:hi].contiguous() if k in ("x", "delta", "B", "C") else t)
                   for k, t in inp.items()} for (lo, hi) in spans]
        Ps, Us = [], []
        for s in slices:
            P = torch.full((batch, d_inner, 16), float("nan"), device=dev)
            U = torch.full((batch, d_inner, 16), float("nan"), device=dev)
            lib.selective_scan_slice_aggregate(s["x"], s["delta"], s["A"], s["B"], s["C"], P, U)
            Ps.append(P)
            Us.append(U)
        P_all, U_all = torch.stack(Ps), torch.stack(Us)
        ys = []
        for r, s in enumerate(slices):
            h_in = torch.full((batch, d_inner, 16), float("nan"), device=dev)
            lib.compose_carry(P_all, U_all, inp["h0"], h_in, r)
            y = torch.full_like(s["x"], float("nan"))
            hl = torch.full((batch, d_inner, 16), float("nan"), device=dev)
            lib.selective_scan_fwd(s["x"], s["delta"], s["A"], s["B"], s["C"], s["D"], h_in, y, hl)
            ys.append(y)
        torch.cuda.synchronize()
        what = f"L-sharded {dtype} {batch}x{d_inner}x{L} R={R}"
        assert_close(torch.cat(ys, dim=2), yref, dtype, what + " y")
        assert_close(hl, hlref, dtype, what + " h_last")
