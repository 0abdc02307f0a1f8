#!/usr/bin/env python
"""bench.py — measures BASELINE.json's metric ("selective-scan fwd elements/s and achieved HBM
GB/s (% of B200 peak) at 1 GPU") on the Mamba-scale config (configs[2], "cfg3": batch 8,
d_inner 4096, N 16, L 2048, bf16 io, fp32 state) and prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 1..5] [--L len] [--variant V] [--no-e2e] [--no-cpu-baseline]
                    [--no-all-configs] [--ext gated|powers|scalar]

A "step" is one pass of the whole hot path (one selective_scan_fwd / affine_scan call) over
one batch of seeded synthetic input.  For N > 1 (torchrun) every rank runs the same workload
on its own batch (the path shards over independent rows with no collective: weak scaling),
timing is the max over ranks, and `value` is all ranks' elements / that time.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from workloads import (config, make_affine_inputs, make_selective_inputs,  # noqa: E402
                       to_f64_numpy)

METRIC = "selective_scan_fwd_elements_per_s"
L2_BYTES = 126 * (1 << 20)
FALLBACK_HBM_GBS = 6650.0      # B200_PROFILING.md fallback ("of fallback")
NOMINAL_HBM_GBS = 8000.0       # BASELINE.json north_star "~8 TB/s"
SM_COUNT_FALLBACK = 148        # used only if the device cannot be asked
MUFU_PER_CLK_PER_SM = 16       # NOMINAL: 4 SFU lanes per sub-partition x 4 (ex2 results/clk/SM)
FP32_PER_CLK_PER_SM = 128      # NOMINAL: 32 FP32 lanes per sub-partition x 4 (lane-ops/clk/SM)


# ----------------------------------------------------------------------------- helpers
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            mp = json.load(f)
        return float(mp["hbm_gbs"]), "measured", mp
    except Exception:
        return FALLBACK_HBM_GBS, "fallback", {}


def dtype_name(dt):
    return {torch.float32: "f32", torch.bfloat16: "bf16"}[dt]


def algorithmic_bytes(c, has_h0, has_D=True):
    """SURVEY §8d.3 / DESIGN.md §5: the minimum bytes one call must move."""
    sz = 2 if c.dtype == torch.bfloat16 else 4
    if c.kind == "affine":
        return c.num_seq * c.L * 3 * sz + 4 * c.num_seq * (1 + (1 if has_h0 else 0))
    rows = c.batch * c.d_inner
    return (3 * rows * c.L * sz + 2 * c.batch * c.N * c.L * sz + 4 * c.d_inner * c.N
            + (4 * c.d_inner if has_D else 0) + 4 * rows * c.N * (1 + (1 if has_h0 else 0)))


class ClockSampler:
    """Samples SM clock / power / throttle reasons while the timed region runs (pynvml)."""
    BITS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
            0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
            0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x100: "display_clock"}

    def __init__(self, index, period=0.01):
        self.index, self.period = index, period
        self.samples, self.reasons, self.power = [], set(), []
        self._stop = threading.Event()
        self._thread = None
        self.max_mhz = None
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def _sample(self):
        nv = self.nv
        self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
        except Exception:
            pass
        try:
            mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for bit, name in self.BITS.items():
            if mask & bit and name != "gpu_idle":
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.ok:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        if self._thread:
            try:
                self._sample()
            except Exception:
                pass
            self._stop.set()
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        s = sorted(self.samples)
        out = {"sm_mhz": float(s[len(s) // 2]), "sm_max_mhz": float(self.max_mhz or 0),
               "reasons": sorted(self.reasons), "samples": len(s)}
        if self.power:
            out["power_w_max"] = round(max(self.power), 1)
        return out


# ------------------------------------------------------------------------ the workload
class Workload:
    """One BASELINE.json config (optionally with a forced L, a forced variant, or one of the
    SURVEY §8f extensions) with rotating device input/output sets."""

    def __init__(self, cfg, device, L=0, ext=None, total=None):
        over = {}
        if cfg == 5:
            over["L"] = L or (1 << 16)
            if total:
                over["total"] = total
        elif L:
            over["L"] = L
        self.c = config(cfg, **over)
        self.device = device
        self.kind = self.c.kind
        self.ext = ext if self.kind == "selective" else None
        self.sets = []

    def build_sets(self, nsets, seed_offset=0):
        import paper_2606_00601_b200 as lib
        self.lib = lib
        c = self.c
        for i in range(nsets):
            ci = config_with_seed(c, c.seed + 17 * i + seed_offset)
            if self.kind == "affine":
                inp = make_affine_inputs(ci, device=self.device)
                out = {"h": torch.empty_like(inp["a"]),
                       "h_last": torch.empty(c.num_seq, dtype=torch.float32, device=self.device)}
            else:
                inp = make_selective_inputs(ci, device=self.device)
                self._apply_ext(inp, ci)
                out = {"y": torch.empty_like(inp["x"]),
                       "h_last": torch.empty((c.batch, c.d_inner, c.N), dtype=torch.float32,
                                             device=self.device)}
            self.sets.append((inp, out))
        self.has_h0 = self.sets[0][0].get("h0") is not None
        self.bytes = algorithmic_bytes(c, self.has_h0)
        if self.ext == "gated":       # + z read + bias read
            sz = 2 if c.dtype == torch.bfloat16 else 4
            self.bytes += c.batch * c.d_inner * c.L * sz + 4 * c.d_inner

    def _apply_ext(self, inp, ci):
        """Inputs of the SURVEY §8f rows: "gated" = raw delta (pre-softplus) + bias + z;
        "powers" / "scalar" = structured A (A[d,n] = (n+1) A[d,0] / A[d,n] = A[d,0])."""
        from workloads import normal, uniform
        c, dev = self.c, self.device
        inp["z"] = inp["delta_bias"] = None
        if self.ext == "gated":
            shape = (c.batch, c.d_inner, c.L)
            inp["delta"] = normal(shape, mean=c.delta_shift, seed=ci.seed, stream=22, device=dev,
                                  dtype=c.dtype)               # softplus is applied by the kernel
            inp["z"] = normal(shape, seed=ci.seed, stream=20, device=dev, dtype=c.dtype)
            inp["delta_bias"] = normal((c.d_inner,), std=0.1, seed=ci.seed, stream=21, device=dev,
                                       dtype=torch.float32)
        elif self.ext in ("powers", "scalar"):
            a0 = -torch.exp(uniform((c.d_inner,), -1.0, 0.5, seed=ci.seed, stream=30, device=dev,
                                    dtype=torch.float32))
            if self.ext == "scalar":
                inp["A"] = a0[:, None].repeat(1, c.N).contiguous()
            else:
                n1 = torch.arange(1, c.N + 1, device=dev, dtype=torch.float32)
                inp["A"] = (0.25 * a0[:, None] * n1[None, :]).contiguous()

    def launch(self, i, variant=0):
        inp, out = self.sets[i % len(self.sets)]
        lib = self.lib
        if self.kind == "affine":
            lib.affine_scan_ex(inp["a"], inp["u"], inp["h0"], out["h"], out["h_last"], variant)
        elif self.ext:
            structure = {"gated": lib.A_GENERAL, "powers": lib.A_POWERS,
                         "scalar": lib.A_SCALAR_PER_ROW}[self.ext]
            lib.selective_scan_fwd_ext(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"], inp["D"],
                                       inp["z"], inp["delta_bias"], None, inp["h0"], out["y"],
                                       out["h_last"], self.ext == "gated", structure, variant)
        else:
            lib.selective_scan_fwd_ex(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"],
                                      inp["D"], inp["h0"], out["y"], out["h_last"], variant)

    # end-to-end through the C-ABI with HOST buffers (pinned)
    def build_host(self):
        inp, out = self.sets[0]
        self.h_in = {k: (None if v is None else v.cpu().pin_memory()) for k, v in inp.items()}
        self.h_out = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
        self.h2d = sum(v.numel() * v.element_size() for v in self.h_in.values() if v is not None)
        self.d2h = sum(v.numel() * v.element_size() for v in self.h_out.values())

    def launch_host(self):
        i, o = self.h_in, self.h_out
        if self.kind == "affine":
            self.lib.affine_scan_host(i["a"], i["u"], i["h0"], o["h"], o["h_last"])
        else:
            self.lib.selective_scan_fwd_host(i["x"], i["delta"], i["A"], i["B"], i["C"], i["D"],
                                             i["h0"], o["y"], o["h_last"])

    def describe(self, world):
        c = self.c
        d = {"workload": c.name + (f"+{self.ext}" if self.ext else ""),
             "call": "affine_scan" if self.kind == "affine"
             else ("selective_scan_fwd_ext" if self.ext else "selective_scan_fwd"), "seed": c.seed}
        if self.kind == "affine":
            d.update(num_seq=c.num_seq, L=c.L)
        else:
            d.update(batch=c.batch, d_inner=c.d_inner, N=c.N, L=c.L)
        d["io_dtype"] = dtype_name(c.dtype)
        d["parallelism"] = f"independent_batches_x{world}" if world > 1 else "single_gpu"
        return d


def config_with_seed(c, seed):
    from dataclasses import replace
    return replace(c, seed=seed)


# ----------------------------------------------------------------- CPU baseline (oracle)
def oracle_sample_runner(c, device_inputs, seed=0):
    """Returns (run(n_units) -> elements processed, unit name, max units).  The sample is the
    first n rows / sequences of the SAME workload; the oracle runs as it stands (1 thread)."""
    import oracle
    inp = device_inputs
    if c.kind == "affine":
        a, u = inp["a"], inp["u"]
        h0 = inp["h0"]

        def run(n):
            n = max(1, min(n, c.num_seq))
            ha, hu = to_f64_numpy(a[:n]), to_f64_numpy(u[:n])
            hh = None if h0 is None else to_f64_numpy(h0[:n])
            t0 = time.perf_counter()
            oracle.affine_scan(ha, hu, hh)
            return n * c.L, time.perf_counter() - t0
        return run, "sequences", c.num_seq

    cache = {}

    def host_batch(b):
        """float64 host copy of batch b (exact widening), made outside the timed calls."""
        if b not in cache:
            cache.clear()           # one batch at a time: cfg3 is 2 x 64 MB of float64 per batch
            cache[b] = {k: (None if v is None else
                            to_f64_numpy(v[b:b + 1] if k in ("x", "delta", "B", "C", "h0") else v))
                        for k, v in inp.items()}
        return cache[b]

    def run(n):
        """Oracle over the first n (b, d) rows of the workload; returns (elements, seconds)."""
        n = max(1, min(n, c.batch * c.d_inner))
        done, secs = 0, 0.0
        for b in range(c.batch):
            rows = min(c.d_inner, n - done)
            if rows <= 0:
                break
            h = host_batch(b)
            t0 = time.perf_counter()
            oracle.selective_scan_fwd(h["x"][:, :rows], h["delta"][:, :rows], h["A"][:rows],
                                      h["B"], h["C"], h["D"][:rows],
                                      None if h["h0"] is None else h["h0"][:, :rows])
            secs += time.perf_counter() - t0
            done += rows
        return done * c.L, secs
    return run, "rows (b,d order)", c.batch * c.d_inner


def time_oracle(c, inputs, target_s):
    """The oracle as it stands on a bounded sample of the workload: (i) 1 thread, the plain loop;
    (ii) all host cores: the identical loop, the sample's outer rows / sequences split over
    T = os.cpu_count() threads by THIS harness (oracle.c itself stays one-threaded;
    ctypes releases the GIL).  Returns (one_thread, all_cores) records."""
    from concurrent.futures import ThreadPoolExecutor
    run, unit, max_units = oracle_sample_runner(c, inputs)
    probe = max(1, min(max_units, 8))
    run(1)                                   # load/compile the C oracle outside the timing
    el, dt = run(probe)
    n = int(max(1, min(max_units, probe * target_s / max(dt, 1e-6))))
    el, dt = run(n)
    one = {"value": el / dt, "unit": "elements/s", "cores": 1, "kind": "oracle",
           "sample": f"first {n} {unit} of the workload ({el} elements, {dt:.2f} s of oracle "
                     f"time, float64, 1 thread)"}
    T = max(1, os.cpu_count() or 1)
    runners = [oracle_sample_runner(c, inputs)[0] for _ in range(T)]   # a host cache per thread
    per = max(1, min(max_units, n) // T)
    for r in runners:
        r(1)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(T) as pool:
        done = list(pool.map(lambda r: r(per), runners))
    wall = time.perf_counter() - t0
    el_all = sum(d[0] for d in done)
    allc = {"value": el_all / wall, "unit": "elements/s", "cores": T, "kind": "oracle",
            "sample": f"{T} threads x the first {per} {unit} of the workload each ({el_all} elements, "
                      f"{wall:.2f} s wall incl. per-thread float64 widening, float64)"}
    return one, allc


# ------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    w = Workload(args.config, "cpu", args.L)
    c = w.c
    inputs = (make_affine_inputs if c.kind == "affine" else make_selective_inputs)(
        c if c.elements <= (1 << 24) else shrink_for_cpu(c), device="cpu")
    run, unit, max_units = oracle_sample_runner(c if c.elements <= (1 << 24) else shrink_for_cpu(c),
                                                inputs)
    # size the per-step sample so that (steps + warmup) steps end within ~2 minutes
    run(1)
    _, t4 = run(4)
    per_unit = t4 / 4
    budget = 120.0 / max(1, args.steps + args.warmup)
    n = int(max(1, min(max_units, budget / max(per_unit, 1e-9))))
    for _ in range(args.warmup):
        run(n)
    elements, dt = 0, 0.0
    for _ in range(args.steps):
        e, t = run(n)               # t = seconds inside the oracle (host widening excluded)
        elements += e
        dt += t
    value = elements / dt
    sample = f"{n} {unit} per step ({elements // max(1, args.steps)} elements/step), float64, 1 thread"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "elements/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, workloads/gen.py)",
        "config": w.describe(1),
        "io_dtype": dtype_name(c.dtype),
        "cpu_baseline": {"value": value, "unit": "elements/s", "cores": 1, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "elements/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def shrink_for_cpu(c):
    """Host-side stand-in for the big configs: same distributions and L, fewer rows, so the
    reference arm never materialises hundreds of MB it will not scan."""
    from dataclasses import replace
    if c.kind == "affine":
        return replace(c, num_seq=min(c.num_seq, max(1, (1 << 22) // c.L)))
    return replace(c, batch=1, d_inner=min(c.d_inner, 512))


# ------------------------------------------------------------------------------ our arm
def sm_count(device):
    try:
        return torch.cuda.get_device_properties(device).multi_processor_count
    except Exception:
        return SM_COUNT_FALLBACK


def alu_ceiling(c, mhz, sms):
    """NOMINAL two-pipe arithmetic ceiling of the fused selective scan: per
    state-step one 2^x and 4 FP32 lane-ops; a share f of the 2^x evaluated on the FP32 pipe as a
    degree-DEG polynomial (2 + DEG extra lane-ops), the rest on the SFU; the pipes balance at
    (1 - f) / 16 = (4 + (2 + DEG) f) / 128 cycles per state-step per SM, with the NOMINAL unit
    counts 16 SFU and 128 FP32 lanes per SM (4 and 32 per sub-partition)."""
    deg = 3 if c.dtype == torch.bfloat16 else 5
    f = (FP32_PER_CLK_PER_SM - 4 * MUFU_PER_CLK_PER_SM) / (
        FP32_PER_CLK_PER_SM + (2 + deg) * MUFU_PER_CLK_PER_SM)
    per_clk_sm = MUFU_PER_CLK_PER_SM / (1.0 - f)          # state-steps / clk / SM
    return f, per_clk_sm, per_clk_sm * sms * mhz * 1e6     # state-steps / s


def measure(w, variant, K, warm, device, local, barrier, max_over_ranks, world=1):
    """W warm-up launches, then K timed launches: device time of the whole region (t_begin..t_end,
    max over ranks) and a CUDA-event pair around every launch, with the clocks sampled meanwhile."""
    lib = w.lib
    for i in range(max(warm, 3)):
        w.launch(i, variant)
    torch.cuda.synchronize()
    chosen = lib.last_variant()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(K)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = lib.launch_count()
    barrier()
    torch.cuda.profiler.start()      # ncu --profile-from-start off sees the timed region only
    with ClockSampler(local) as clocks:
        # Keep the GPU busy while the host enqueues the K launches, so that the device never
        # waits for the host inside the timed region (short kernels: cfg1, cfg2).
        torch.cuda._sleep(min(int(K * 6e4), int(4e8)))
        t_begin.record()
        for i in range(K):
            ev[i][0].record()
            w.launch(i, variant)
            ev[i][1].record()
        t_end.record()
        torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    barrier()
    launches = lib.launch_count() - launches0
    total_ms = max_over_ranks(t_begin.elapsed_time(t_end), device)
    per_launch_ms = sorted(a.elapsed_time(b) for a, b in ev)
    return {"chosen": chosen, "launches": launches, "total_ms": total_ms,
            "kernel_ms": sum(per_launch_ms) / K, "kernel_ms_min": per_launch_ms[0],
            "kernel_ms_median": per_launch_ms[K // 2], "clocks": clocks.summary()}


def nsets_for(step_bytes):
    """Rotating input/output sets so that > 126 MB (L2) of other data passes between reuses."""
    n = max(2, -(-4 * L2_BYTES // step_bytes)) if step_bytes < 4 * L2_BYTES else 2
    return min(n, 64)


def summarize(w, m, peak, sms):
    """Per-config record of the all_configs block."""
    c = w.c
    achieved = w.bytes / (m["kernel_ms"] * 1e-3) / 1e9
    clk = m["clocks"]
    rec = {"workload": w.describe(1)["workload"], "kernel": w.lib.VARIANT_NAMES.get(m["chosen"], "?"),
           "kernel_ms": round(m["kernel_ms"], 5), "kernel_ms_min": round(m["kernel_ms_min"], 5),
           "elements_per_s": c.elements / (m["kernel_ms"] * 1e-3),
           "algorithmic_bytes": w.bytes, "hbm_gbs": round(achieved, 1),
           "hbm_frac": round(achieved / peak, 4),
           "hbm_frac_of_nominal_8TBps": round(achieved / NOMINAL_HBM_GBS, 4),
           "clocks": {"sm_mhz": clk.get("sm_mhz"), "reasons": clk.get("reasons")}}
    if c.kind == "selective":
        mhz = clk.get("sm_mhz") or clk.get("sm_max_mhz") or 1965.0
        steps_state = c.elements * c.N
        mufu_ms = steps_state / (MUFU_PER_CLK_PER_SM * sms * mhz * 1e6) * 1e3
        rec["frac_of_mufu_only_wall"] = round(mufu_ms / m["kernel_ms"], 4)
    return rec


def time_backward(cfg, device, local, peak, barrier, K, W):
    """selective_scan_bwd on a selective config's shape.  Algorithmic bytes: reads
    x, delta, dy (io dtype) and B, C; writes dx, ddelta (fp32), dB, dC, dA, dD."""
    import paper_2606_00601_b200 as lib
    from workloads import normal
    c = config(cfg)
    inp = make_selective_inputs(c, device=device)
    dy = normal(inp["x"].shape, seed=c.seed, stream=40, device=device, dtype=c.dtype)
    f32 = dict(dtype=torch.float32, device=device)
    bdl, bnl = (c.batch, c.d_inner, c.L), (c.batch, c.N, c.L)
    g = [torch.empty(bdl, **f32), torch.empty(bdl, **f32), torch.empty((c.d_inner, c.N), **f32),
         torch.empty(bnl, **f32), torch.empty(bnl, **f32), torch.empty((c.d_inner,), **f32),
         torch.empty((c.batch, c.d_inner, c.N), **f32)]

    def launch():
        lib.selective_scan_bwd(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"], inp["D"], None,
                               dy, None, *g)
    for _ in range(W):
        launch()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(K)]
    barrier()
    torch.cuda.profiler.start()      # as in measure(): a profiler sees the timed launches only
    with ClockSampler(local) as clocks:
        for a, b in ev:
            a.record()
            launch()
            b.record()
        torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    ms = sorted(a.elapsed_time(b) for a, b in ev)
    kernel_ms = sum(ms) / K
    sz = 2 if c.dtype == torch.bfloat16 else 4
    rows = c.batch * c.d_inner
    nbytes = (3 * rows * c.L * sz + 2 * c.batch * c.N * c.L * sz + 2 * rows * c.L * 4
              + 2 * c.batch * c.N * c.L * 4 + 4 * c.d_inner * (2 * c.N + 2) + 4 * rows * c.N)
    achieved = nbytes / (kernel_ms * 1e-3) / 1e9
    clk = clocks.summary()
    return {"workload": c.name + "+backward", "kernel": "selective_scan_bwd (3 launches)",
            "kernel_ms": round(kernel_ms, 5), "kernel_ms_min": round(ms[0], 5),
            "elements_per_s": c.elements / (kernel_ms * 1e-3), "algorithmic_bytes": nbytes,
            "hbm_gbs": round(achieved, 1), "hbm_frac": round(achieved / peak, 4),
            "hbm_frac_of_nominal_8TBps": round(achieved / NOMINAL_HBM_GBS, 4),
            "clocks": {"sm_mhz": clk.get("sm_mhz"), "reasons": clk.get("reasons")},
            "note": "library scratch (checkpoints + dB/dC partials) is not counted as algorithmic"}


def run_all_configs(args, device, local, peak, sms, barrier, max_over_ranks):
    """cfg1, cfg2, cfg4 (+ the forced chunked schedule), the six cfg5 lengths (+ forced look-back
    on one long sequence and on 64 sequences), and the §8f rows on the cfg3 shape — about 10 timed
    launches each, so the per-config claims of BASELINE.md are driver-timed."""
    import paper_2606_00601_b200 as lib
    out = []
    K, W = args.all_configs_steps, 3

    def one(w, variant=0, note=None):
        m = measure(w, variant, K, W, device, local, barrier, max_over_ranks)
        rec = summarize(w, m, peak, sms)
        if variant:
            rec["forced_variant"] = lib.VARIANT_NAMES.get(variant, str(variant))
        if note:
            rec["note"] = note
        out.append(rec)

    def selective(cfg, variants=(0,), ext=None):
        w = Workload(cfg, device, ext=ext)
        sb = algorithmic_bytes(w.c, False)
        w.build_sets(nsets_for(sb))
        for v in variants:
            one(w, v)
        del w
        torch.cuda.empty_cache()

    w = Workload(1, device)
    w.build_sets(64)
    one(w, note="197 KB: launch-latency-bound; 64 rotating sets still fit L2")
    del w
    selective(2)
    selective(4, (0, lib.SELECTIVE_CHUNKED))
    selective(3, (0,), "gated")
    selective(3, (0,), "powers")
    selective(3, (0,), "scalar")
    out.append(time_backward(3, device, local, peak, barrier, K, W))
    # cfg5: one flat 2^30-element pair of arrays re-segmented for every L (12.9 GB >> L2)
    total = 1 << 30
    w5 = Workload(5, device, L=total, total=total)
    w5.build_sets(1)
    inp, outp = w5.sets[0]
    from workloads import normal
    h0_all = normal((1 << 20,), seed=w5.c.seed, stream=3, device=device, dtype=torch.float32)

    def resegment(L, variant=0, note=None):
        S = total // L
        ws = Workload(5, device, L=L, total=total)
        ws.lib = lib
        ws.sets = [({"a": inp["a"].view(S, L), "u": inp["u"].view(S, L), "h0": h0_all[:S]},
                    {"h": outp["h"].view(S, L),
                     "h_last": torch.empty(S, dtype=torch.float32, device=device)})]
        ws.has_h0 = True
        ws.bytes = algorithmic_bytes(ws.c, True)
        one(ws, variant, note)

    for logL in (10, 12, 14, 16, 18, 20):
        resegment(1 << logL)
    resegment(1 << 24, lib.AFFINE_LOOKBACK, "64 sequences of 2^24, forced decoupled look-back")
    resegment(1 << 30, lib.AFFINE_LOOKBACK, "ONE sequence of 2^30, forced decoupled look-back")
    del w5, inp, outp
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py (impl ours) needs a CUDA device; there is no CPU fallback")
    if local >= torch.cuda.device_count():
        raise RuntimeError(f"rank {rank}: LOCAL_RANK {local} but only {torch.cuda.device_count()} "
                           "CUDA devices are visible")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    from paper_2606_00601_b200.sharding import max_over_ranks

    from paper_2606_00601_b200 import build as libbuild
    if not os.path.exists(libbuild.LIB_PATH):
        libbuild.build()             # fresh checkout: the built library is git-ignored
    import paper_2606_00601_b200 as lib
    lib.set_option(lib.OPT_LANE_ROW_G, args.lane_row_g)
    lib.set_option(lib.OPT_LANE_ROW_POLY16, args.lane_row_poly16)
    sms = sm_count(device)
    w = Workload(args.config, device, args.L, args.ext)
    c = w.c
    step_bytes = algorithmic_bytes(c, c.kind == "affine" and c.h0_recipe == "normal")
    nsets = nsets_for(step_bytes)
    w.build_sets(nsets, seed_offset=1000 * rank)
    variant = args.variant

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    K = args.steps
    m = measure(w, variant, K, args.warmup, device, local, barrier, max_over_ranks, world)
    kernel_ms = m["kernel_ms"]
    ms_per_step = m["total_ms"] / K
    elements = c.elements * world
    value = elements / (ms_per_step * 1e-3)

    peak, peak_kind, mp = measured_peaks()
    achieved = w.bytes / (kernel_ms * 1e-3) / 1e9
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.txt")) as f:
            for ln in f:
                parts = ln.split()
                if len(parts) >= 2 and parts[0] == w.describe(1)["workload"]:
                    traffic = int(parts[1])
    except Exception:
        pass
    clk = m["clocks"]
    kernel_name = lib.VARIANT_NAMES.get(m["chosen"], str(m["chosen"]))
    hbm = {"bound": "hbm", "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
           "frac": round(achieved / peak, 4), "traffic": traffic,
           "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum of the committed "
                             "--set full capture (profiles/traffic.txt), not measured in this run",
           "peak_kind": peak_kind,
           "algorithmic_bytes": w.bytes, "kernel_ms": round(kernel_ms, 5),
           "kernel_ms_min": round(m["kernel_ms_min"], 5),
           "kernel_ms_median": round(m["kernel_ms_median"], 5),
           "frac_of_nominal_8TBps": round(achieved / NOMINAL_HBM_GBS, 4),
           "kernel": kernel_name}
    if args.lane_row_g != -1 or args.lane_row_poly16 != -1:
        hbm["ablation"] = {"lane_row_g": args.lane_row_g, "lane_row_poly16": args.lane_row_poly16}
    line = {
        "metric": METRIC, "value": value, "unit": "elements/s", "n_gpus": world, "steps": K,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "io_dtype": dtype_name(c.dtype),
        "data": "synthetic (seeded, workloads/gen.py; BASELINE.json distributions)",
        "config": {**w.describe(world),
                   "l2": f"{nsets} rotating input/output sets x {step_bytes / 1e6:.1f} MB "
                         f"(> 126 MB L2 between reuses)"},
        "clocks": clk, "gpu_launches": m["launches"], "sm_count": sms,
        "hbm_gbs_achieved": round(achieved, 1),
        # BASELINE.json's own yardstick, stated at top level: fraction of HBM peak and its target
        "hbm_frac_of_measured_peak": hbm["frac"],
        "hbm_frac_of_nominal_8TBps": hbm["frac_of_nominal_8TBps"],
        "target_70pct_of_hbm_peak_met": bool(achieved / NOMINAL_HBM_GBS >= 0.70),
    }
    if c.kind == "selective" and args.ext in (None, "gated"):
        # The binding roofline of the general-A path is arithmetic, not HBM.
        mhz = clk.get("sm_mhz") or clk.get("sm_max_mhz") or 1965.0
        f, per_clk_sm, alu_peak = alu_ceiling(c, mhz, sms)
        steps_state = c.elements * c.N
        mufu_ms = steps_state / (MUFU_PER_CLK_PER_SM * sms * mhz * 1e6) * 1e3
        fp32_floor_ms = 4 * steps_state / (FP32_PER_CLK_PER_SM * sms * mhz * 1e6) * 1e3
        alu_achieved = steps_state / (kernel_ms * 1e-3)
        # BASELINE.json's metric is the HBM fraction, so `roofline` stays the HBM view;
        # the arithmetic ceiling that actually binds this path is reported beside it.
        line["roofline"] = hbm
        line["roofline_alu"] = {
            "bound": "alu", "achieved": alu_achieved, "peak": alu_peak, "unit": "state-steps/s",
            "frac": round(alu_achieved / alu_peak, 4),
            "peak_kind": "nominal: 16 SFU (MUFU.EX2) + 128 FP32 lanes per clock per SM "
                         f"x {sms} SMs x sampled SM clock, balanced polynomial offload "
                         "(derivation: DESIGN.md §11)",
            "poly_share_at_balance": round(f, 4), "state_steps_per_clk_per_sm": round(per_clk_sm, 2),
            "kernel_ms": hbm["kernel_ms"], "kernel": hbm["kernel"],
            "mufu_only_wall_ms": round(mufu_ms, 4),
            "frac_of_mufu_only_wall": round(mufu_ms / kernel_ms, 4),
            "fp32_only_floor_ms": round(fp32_floor_ms, 4),
            "alu_wall_ms": round(steps_state / alu_peak * 1e3, 4), "sm_mhz_used": mhz,
            "note": "the general-A selective scan needs N exp and 4N FP32 lane-ops per element: "
                    "its arithmetic floor lies above the HBM floor (DESIGN.md §6.2)"}
        if "ablation" in hbm:
            line["roofline_alu"]["ablation"] = hbm["ablation"]
    else:
        line["roofline"] = hbm

    # ---- end to end through the C-ABI with host buffers
    if not args.no_e2e and not args.ext:
        w.build_host()
        for _ in range(2):
            w.launch_host()
        barrier()
        ke = max(3, min(args.e2e_steps, K))
        t0 = time.perf_counter()
        for _ in range(ke):
            w.launch_host()          # synchronises the stream before returning
        torch.cuda.synchronize()
        e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / ke, device)
        line["e2e"] = {"value": elements / (e2e_ms * 1e-3), "unit": "elements/s",
                       "h2d_bytes_per_step": w.h2d, "d2h_bytes_per_step": w.d2h,
                       "steps": ke, "ms_per_step": e2e_ms,
                       "api": f"{'affine_scan' if c.kind == 'affine' else 'selective_scan_fwd'}"
                              "_host (pinned host buffers, H2D + kernel + D2H per step)"}

    # ---- the oracle timed beside it (rank 0, N=1 only): one thread and all host cores
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        one, allc = time_oracle(c, w.sets[0][0], args.cpu_seconds)
        line["cpu_baseline"] = one
        line["cpu_baseline_all_cores"] = allc

    # ---- every other config, driver-timed (rank 0, N=1, default workload only)
    if (rank == 0 and world == 1 and not args.no_all_configs and args.config == 3
            and not args.ext and not args.variant):
        del w
        torch.cuda.empty_cache()
        line["all_configs"] = run_all_configs(args, device, local, peak, sms, barrier,
                                              max_over_ranks)
        # compact digest LAST in the line (dict order is print order): a log that keeps only the
        # tail of stdout still shows every config: [workload, kernel, ms, frac of measured HBM,
        # frac of the MUFU-only wall or null]
        line["configs_summary"] = [
            [r["workload"].replace("_selective", "").replace("_affine", ""), r["kernel"],
             round(r["kernel_ms"], 4), r["hbm_frac"], r.get("frac_of_mufu_only_wall")]
            for r in line["all_configs"]]

    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` (N > 1) outside torchrun: start the N ranks ourselves, one per
    GPU, exactly as the driver would; refuse (non-zero) when the box has fewer GPUs."""
    import socket
    import subprocess
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        print(f"bench.py: --gpus {args.gpus} requested but {have} CUDA device(s) visible; "
              "refusing to time fewer GPUs than asked", file=sys.stderr)
        return 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
           f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port", str(port),
           os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config 1..5 (default 3)")
    ap.add_argument("--L", type=int, default=0, help="sequence length override (config 5 sweep)")
    ap.add_argument("--variant", type=int, default=0, help="force an affinescan_variant")
    ap.add_argument("--lane-row-g", type=int, default=-1, help="ablation: lanes per row (1, 2, 4)")
    ap.add_argument("--lane-row-poly16", type=int, default=-1,
                    help="ablation: sixteenths of the exps on the fma-pipe polynomial (0, 3..6)")
    ap.add_argument("--ext", default=None, choices=["gated", "powers", "scalar"],
                    help="SURVEY §8f rows on the chosen selective config: fused softplus/bias + "
                         "silu(z) gate, or a structured-A fast path")
    ap.add_argument("--no-all-configs", action="store_true",
                    help="skip the per-config block (cfg1, 2, 4, cfg5 sweep, §8f rows)")
    ap.add_argument("--all-configs-steps", type=int, default=10)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    args = ap.parse_args()
    if args.steps < 1:
        ap.error("--steps must be >= 1")
    if args.impl == "reference":
        sys.exit(run_reference(args))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))           # never silently time one GPU for --gpus N
    if args.gpus != world:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}", file=sys.stderr)
        sys.exit(2)
    sys.exit(run_ours(args))


if __name__ == "__main__":
    main()
