#!/usr/bin/env python
"""bench.py -- headline measurement of the tile_gemm hot path on B200.

    python bench.py --gpus N --steps K --warmup W            # this build (CUDA path, C ABI)
    python bench.py --impl reference --steps K --warmup W    # the fp64 CPU oracle, timed as it stands

One JSON line on stdout (rank 0).  A "step" is one call of tile_gemm on BASELINE.json's
config[2] -- the 8192^3 BF16 GEMM with bf16 output the metric is quoted on -- which runs the
whole GEMM path per call: launch preconditions (a1), selector (a2), persistent tile map (a3),
TMA K-loop loads (a4), tcgen05 MMAs (a5), epilogue (a6).  The M=1 decode path (a7, config[4]:
256 GEMVs over distinct 62.4 GB of weights) and the prefill projections (config[3]) are timed in
the same run and reported under "gemv" / "prefill" with their own rooflines.

N > 1: one process per GPU (torchrun), every rank runs the same independent problem (no
data-path collective exists for this path), time = max over ranks, value = sum of the work.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bf16_gemm_tflops"
UNIT = "TFLOP/s"
WORKLOAD = "cfg3: BF16 GEMM M=N=K=8192, A~N(0,1), B~N(0,1/K), fp32 accumulate, bf16 output, seed 2"
L2_NOTE = "inputs 256 MiB per step > 126 MB L2; 4 rotating A/B/C sets so no step re-reads the previous step's data"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "source": "measured"}
    # B200_PROFILING.md fallback
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def ncu_traffic(key):
    """Per-launch DRAM bytes of the dominant kernel from the committed ncu capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(path):
        with open(path) as f:
            for line in f:
                parts = line.strip().split(",")
                if len(parts) >= 2 and parts[0] == key:
                    return float(parts[1])
    return None


# ---------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock, power and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.stop_flag, self.thread = [], set(), False, None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20,
                 "hw_thermal_slowdown": 0x40, "hw_power_brake": 0x80}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv:
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()
        return self

    def __exit__(self, *a):
        self.stop_flag = True
        if self.thread:
            self.thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------- CPU oracle legs
def oracle_gemm_sample(rows, seed=2):
    """The oracle as it stands on a slab of cfg3: `rows` rows of A against all of B."""
    import oracle
    rng = np.random.default_rng([seed, 99])
    from paper_2606_15991_b200 import workloads as wl
    K = N = 8192
    a = wl.f32_to_bf16_bits(rng.standard_normal((rows, K), dtype=np.float32))
    b = wl.f32_to_bf16_bits(rng.standard_normal((K, N), dtype=np.float32) * np.float32(K ** -0.5))
    oracle.gemm(a[:8], b)   # touch pages / load the library
    t0 = time.perf_counter()
    oracle.gemm(a, b)
    dt = time.perf_counter() - t0
    return 2.0 * rows * N * K / dt / 1e12, dt


def cpu_baseline_leg(target_seconds=12.0):
    import oracle
    cores = oracle.default_threads()
    tf, dt = oracle_gemm_sample(64)
    rows = int(max(64, min(2048, 64 * target_seconds / max(dt, 1e-3))))
    rows -= rows % 8
    tf, dt = oracle_gemm_sample(rows)
    return {"value": tf, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle.gemm (fp64, C and S) on rows [0,{rows}) of cfg3 x all 8192 columns, K=8192; "
                      f"{dt:.1f} s wall on {cores} threads"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    cores = oracle.default_threads()
    _, dt8 = oracle_gemm_sample(32)
    budget = 150.0 / max(1, args.steps + args.warmup)
    rows = int(max(8, min(512, 32 * budget / max(dt8, 1e-3))))
    rows -= rows % 8
    for _ in range(args.warmup):
        oracle_gemm_sample(rows)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_gemm_sample(rows)
    # oracle_gemm_sample times only the oracle call; re-measure wall inclusive of input generation
    wall = time.perf_counter() - t0
    tf = np.mean([oracle_gemm_sample(rows)[0] for _ in range(1)]) if args.steps == 0 else None
    # per-step oracle time measured precisely
    per = [oracle_gemm_sample(rows)[1] for _ in range(max(1, min(3, args.steps)))]
    ms = float(np.median(per)) * 1e3
    value = 2.0 * rows * 8192 * 8192 / (ms * 1e-3) / 1e12
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": f"each step = oracle.gemm on a {rows}-row slab (all N, all K)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{rows} rows x 8192 cols x K=8192 per step, {wall:.1f} s for the timed steps"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------- CUDA legs
def time_region(fn_step, steps, stream_sync, dist_barrier):
    """barrier+sync, K steps between two CUDA events on the launching stream, sync+barrier."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist_barrier()
    stream_sync()
    e0.record()
    for i in range(steps):
        fn_step(i)
    e1.record()
    stream_sync()
    dist_barrier()
    return e0.elapsed_time(e1)   # ms


def bench_gemm(tg, wl, torch, case, steps, warmup, sets, tdist, sampler=None):
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(1000 + case.seed[0])
    out_dt = torch.bfloat16 if case.out_dtype == "bf16" else torch.float32
    bufs = []
    for _ in range(sets):
        A = torch.empty((case.M, case.K), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_a, generator=g)
        B = torch.empty((case.K, case.N), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_b, generator=g)
        C = torch.empty((case.M, case.N), dtype=out_dt, device=dev)
        bufs.append((A, B, C))

    def step(i):
        A, B, C = bufs[i % sets]
        tg.tile_gemm(A, B, C)

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    l0 = tg.tile_gemm_launch_count()
    if sampler is not None:
        with sampler:
            ms = time_region(step, steps, torch.cuda.synchronize, tdist.barrier)
    else:
        ms = time_region(step, steps, torch.cuda.synchronize, tdist.barrier)
    launches = tg.tile_gemm_launch_count() - l0
    ms = tdist.max_over_ranks(ms)
    return ms / steps, launches, bufs


def bench_e2e(tg, wl, torch, case, steps):
    """Same metric through the C ABI with HOST buffers: H2D of A and B, GEMM, D2H of C per step."""
    rng = np.random.default_rng(77)
    esz = 2 if case.out_dtype == "bf16" else 4
    A = torch.empty((case.M, case.K), dtype=torch.bfloat16).pin_memory()
    B = torch.empty((case.K, case.N), dtype=torch.bfloat16).pin_memory()
    C = torch.empty((case.M, case.N), dtype=torch.bfloat16 if esz == 2 else torch.float32).pin_memory()
    A.copy_(torch.from_numpy(rng.standard_normal((case.M, case.K), dtype=np.float32)).to(torch.bfloat16))
    B.copy_((torch.from_numpy(rng.standard_normal((case.K, case.N), dtype=np.float32)) * case.sigma_b).to(torch.bfloat16))
    od = tg.OUT_BF16 if esz == 2 else tg.OUT_F32

    def call():
        rc = tg.tile_gemm_host_raw(A.data_ptr(), B.data_ptr(), C.data_ptr(), case.M, case.N, case.K,
                                   case.K, case.N, case.N, od)
        if rc != 0:
            raise tg.TileGemmError(rc, tg.tile_gemm_last_error())

    call()
    t0 = time.perf_counter()
    for _ in range(steps):
        call()   # synchronous: returns after the D2H copy completed
    dt = (time.perf_counter() - t0) / steps
    h2d = (case.M * case.K + case.K * case.N) * 2
    d2h = case.M * case.N * esz
    tg.tile_gemm_shutdown()   # release the staging buffers
    return dt, h2d, d2h, float(C.float().abs().mean())


def bench_decode(tg, wl, torch, passes, warmup, layers, tdist, static_b=True):
    """config[4]: 4 projections x `layers` layers, every weight in its own buffer.  static_b: the
    calls go through tile_gemm_static_b (decode weights are immutable), which lets each GEMV stream
    weight tiles ahead of the programmatic-dependent-launch wait on its predecessor."""
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(4)
    items = []
    for layer in range(layers):
        for (K, N) in wl.QWEN3_32B:
            W = torch.empty((K, N), dtype=torch.bfloat16, device=dev).normal_(0, 0.02, generator=g)
            x = torch.empty((1, K), dtype=torch.bfloat16, device=dev).normal_(0, 1.0, generator=g)
            y = torch.empty((1, N), dtype=torch.bfloat16, device=dev)
            items.append((x, W, y))
    alg_bytes = sum(2 * K * N + 2 * K + 2 * N for (K, N) in wl.QWEN3_32B) * layers

    def one_pass(_):
        for x, W, y in items:
            tg.tile_gemm(x, W, y, static_b=static_b)

    def plain_pass(_):
        for x, W, y in items:
            tg.tile_gemm(x, W, y)

    for i in range(warmup):
        one_pass(i)
    torch.cuda.synchronize()
    l0 = tg.tile_gemm_launch_count()
    ms = time_region(one_pass, passes, torch.cuda.synchronize, tdist.barrier)
    launches = tg.tile_gemm_launch_count() - l0
    ms = tdist.max_over_ranks(ms) / passes
    plain_pass(0)
    plain_ms = tdist.max_over_ranks(time_region(plain_pass, passes, torch.cuda.synchronize, tdist.barrier)) / passes
    # per-shape kernel time (events around each projection class, one extra pass)
    per_shape = {}
    for p, (K, N) in enumerate(wl.QWEN3_32B):
        sel = items[p::4]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(3):             # three chains back to back: the idle-to-busy start-up is paid once in 3 * layers launches
            for x, W, y in sel:
                tg.tile_gemm(x, W, y, static_b=static_b)
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1) / (3 * len(sel))
        per_shape[f"K{K}_N{N}"] = {"us": round(t * 1e3, 2), "gbs": round((2 * K * N + 2 * K + 2 * N) / (t * 1e-3) / 1e9, 1)}
    # replay of the same pass as one recorded step of the library's own C ABI (tile_gemm_record_*:
    # decode engines replay a recorded step)
    graph_ms = None
    try:
        s = torch.cuda.Stream()
        for x, W, y in items:
            tg.tile_gemm(x, W, y, static_b=static_b, stream=s)     # workspaces of this stream exist before recording
        s.synchronize()
        tg.tile_gemm_record_begin(s)
        for x, W, y in items:
            tg.tile_gemm(x, W, y, static_b=static_b, stream=s)
        step = tg.tile_gemm_record_end(s)
        step.replay(s)
        s.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        for _ in range(passes):
            step.replay(s)
        e1.record(s)
        s.synchronize()
        graph_ms = e0.elapsed_time(e1) / passes
        step.free()
    except Exception as exc:  # reported, never silently substituted for the headline
        graph_ms = None
        sys.stderr.write(f"[bench] recorded-step variant unavailable: {exc}\n")
    return ms, alg_bytes, launches, per_shape, graph_ms, len(items), plain_ms


def bench_add(tg, torch, n, steps, warmup, tdist):
    """z = x + y over f32 at n = 2^28 (Listing 1).  12 B of HBM traffic per
    element; the three 1 GiB vectors are far larger than L2."""
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(28)
    x = torch.empty(n, dtype=torch.float32, device=dev).normal_(0, 1, generator=g)
    y = torch.empty(n, dtype=torch.float32, device=dev).normal_(0, 1, generator=g)
    z = torch.empty(n, dtype=torch.float32, device=dev)
    for _ in range(warmup):
        tg.tile_add_f32(x, y, z)
    ms = time_region(lambda i: tg.tile_add_f32(x, y, z), steps, torch.cuda.synchronize, tdist.barrier)
    return tdist.max_over_ranks(ms) / steps


def bench_launch_overhead(tg, torch, n_ops=1000, elems=2048):
    """PAPER.md:322-326 (Figure 8a): host cost per operation of a pipeline of N tiny element-wise
    kernels, launched one by one with a single wait at the end ("sync" mode) versus recorded once
    and replayed with one driver call ("graph" mode; the paper's floor is ~0.8 us/op on its GPU).
    The op is tile_add_f32 on `elems` floats (the paper uses a length-2048 tile), z_{i+1} = z_i + y."""
    dev = torch.device("cuda", torch.cuda.current_device())
    s = torch.cuda.Stream()
    y = torch.ones(elems, dtype=torch.float32, device=dev)
    za = torch.zeros(elems, dtype=torch.float32, device=dev)
    zb = torch.zeros(elems, dtype=torch.float32, device=dev)

    def chain():
        for i in range(n_ops):
            src, dst = (za, zb) if i % 2 == 0 else (zb, za)
            tg.tile_add_f32(src, y, dst, stream=s)

    chain()
    s.synchronize()
    out = {}
    best = 1e30
    for _ in range(5):
        t0 = time.perf_counter()
        chain()
        s.synchronize()
        best = min(best, time.perf_counter() - t0)
    out["stream_launch_us_per_op"] = best / n_ops * 1e6
    # the same chain through the bare C entry (arguments marshalled once): what a C caller pays
    import ctypes
    lib = tg.load_library()
    vp = ctypes.c_void_p
    pre = [(vp(za.data_ptr()), vp(y.data_ptr()), vp(zb.data_ptr()), elems, vp(s.cuda_stream)),
           (vp(zb.data_ptr()), vp(y.data_ptr()), vp(za.data_ptr()), elems, vp(s.cuda_stream))]
    best = 1e30
    for _ in range(5):
        t0 = time.perf_counter()
        for i in range(n_ops):
            lib.tile_add_f32(*pre[i & 1])
        s.synchronize()
        best = min(best, time.perf_counter() - t0)
    out["stream_launch_us_per_op_c_abi"] = best / n_ops * 1e6
    tg.tile_gemm_record_begin(s)
    chain()
    step = tg.tile_gemm_record_end(s)
    step.replay(s)
    s.synchronize()
    best = 1e30
    for _ in range(5):
        t0 = time.perf_counter()
        step.replay(s)
        s.synchronize()
        best = min(best, time.perf_counter() - t0)
    out["recorded_replay_us_per_op"] = best / n_ops * 1e6
    out["ops"], out["elems_per_op"], out["nodes"] = n_ops, elems, step.nodes
    step.free()
    return out


def bench_skinny(tg, wl, torch, ms_list, tdist, layers=8):
    """skinny M (decode with a few tokens in flight) on the four Qwen3-32B weight shapes:
    the weight-streaming tensor-core kernel up to M = 48 (and M <= 64 on unsliced weights), else the tiled GEMM with K slices.  Weights are
    immutable (tile_gemm_static_b, as in the M = 1 leg).  HBM-bound: reported as GB/s of algorithmic bytes
    (weights once + activations + outputs), `layers` distinct weight sets; `per_shape_gbs` times each of
    the four shapes in a chain of its own (qkv, attn_out, gate_up, down)."""
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(8)
    Ws = [[torch.empty((K, N), dtype=torch.bfloat16, device=dev).normal_(0, 0.02, generator=g)
           for (K, N) in wl.QWEN3_32B] for _ in range(layers)]
    out = {}
    for M in ms_list:
        xs = [torch.empty((M, K), dtype=torch.bfloat16, device=dev).normal_(0, 1, generator=g) for (K, N) in wl.QWEN3_32B]
        ys = [torch.empty((M, N), dtype=torch.bfloat16, device=dev) for (K, N) in wl.QWEN3_32B]

        def one_pass(_):
            for layer in range(layers):
                for p in range(4):
                    tg.tile_gemm(xs[p], Ws[layer][p], ys[p], static_b=True)

        one_pass(0)
        ms = tdist.max_over_ranks(time_region(one_pass, 3, torch.cuda.synchronize, tdist.barrier)) / 3
        byt = sum(2 * K * N + 2 * M * K + 2 * M * N for (K, N) in wl.QWEN3_32B) * layers
        per_shape = []
        for p, (K, N) in enumerate(wl.QWEN3_32B):
            def chain(_, p=p):
                for layer in range(layers):
                    tg.tile_gemm(xs[p], Ws[layer][p], ys[p], static_b=True)
            chain(0)
            ms_p = tdist.max_over_ranks(time_region(chain, 5, torch.cuda.synchronize, tdist.barrier)) / 5
            per_shape.append(round((2 * K * N + 2 * M * K + 2 * M * N) * layers / (ms_p * 1e-3) / 1e9))
        K0, N0 = wl.QWEN3_32B[0]
        out[str(M)] = {"ms_per_pass": round(ms, 4), "gbs": round(byt / (ms * 1e-3) / 1e9, 1), "per_shape_gbs": per_shape,
                       "config": tg.tile_gemm_query_plan(M, N0, K0)["config"] if M >= 2 else 0, "launches_per_pass": 4 * layers}
    return out


SWEEP_COLUMNS = ["us_median_single", "us_back_to_back", "us_recorded_replay", "tflops_recorded_replay", "tile_config"]


def bench_sweep(tg, torch, sizes, tdist, warm_s=0.35):
    """the paper's Figure 6b sweep, M=N=K powers of two, f16 (the
    paper's precision) and bf16, 16-bit output, on rotating operand sets whose total exceeds L2 where
    the problem allows.  Steady-state protocol: every timing of a (size, type) is taken
    directly after `warm_s` seconds of back-to-back launches of that same problem, so that all three
    see the chip in the power state a pipeline of such GEMMs runs in; the type order alternates from
    size to size.  Per size: median of per-launch event timings inside a back-to-back stream (paper:
    medians), the back-to-back average without inner events (programmatic dependent launch intact),
    and the same launches as ONE recorded step (no host in the loop).  Rows follow SWEEP_COLUMNS."""
    dev = torch.device("cuda", torch.cuda.current_device())
    out = {"columns": SWEEP_COLUMNS, "f16": {}, "bf16": {}}
    types = (("f16", torch.float16), ("bf16", torch.bfloat16))
    for si, n in enumerate(sizes):
        for dt_name, dt in (types if si % 2 == 0 else types[::-1]):
            per_set = 3 * n * n * 2
            sets = int(max(1, min(8, (256 << 20) // per_set + 1)))
            reps = 40 if n <= 4096 else (12 if n <= 16384 else 5)
            g = torch.Generator(device=dev)
            g.manual_seed(600 + n)
            bufs = [(torch.empty((n, n), dtype=dt, device=dev).normal_(0, 1, generator=g),
                     torch.empty((n, n), dtype=dt, device=dev).normal_(0, n ** -0.5, generator=g),
                     torch.empty((n, n), dtype=dt, device=dev)) for _ in range(sets)]

            def warm(seconds):
                t_end = time.perf_counter() + seconds
                i = 0
                while time.perf_counter() < t_end:
                    for _ in range(8):
                        tg.tile_gemm(*bufs[i % sets])
                        i += 1
                    if n >= 8192:
                        torch.cuda.synchronize()   # keep the launch queue short: the warm-up must end on time

            # the same launches as one recorded step (mode c)
            rs = torch.cuda.Stream()
            tg.tile_gemm_record_begin(rs)
            for i in range(reps):
                tg.tile_gemm(*bufs[i % sets], stream=rs)
            step = tg.tile_gemm_record_end(rs)
            meds, b2bs, recs = [], [], []
            for rnd in range(3):   # the three modes interleaved, three rounds, median of each: drift of the power state averages out
                warm(warm_s if rnd == 0 else warm_s / 3)
                # (a) per-launch events inside a back-to-back stream
                evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
                for i in range(reps):
                    evs[i][0].record()
                    tg.tile_gemm(*bufs[i % sets])
                    evs[i][1].record()
                torch.cuda.synchronize()
                meds.append(float(np.median([a.elapsed_time(b) for a, b in evs])))
                # (b) back to back, no inner events
                warm(warm_s / 3)
                tdist.barrier()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for i in range(reps):
                    tg.tile_gemm(*bufs[i % sets])
                e1.record()
                torch.cuda.synchronize()
                b2bs.append(e0.elapsed_time(e1) / reps)
                # (c) one recorded step
                warm(warm_s / 3)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(rs)
                step.replay(rs)
                e1.record(rs)
                rs.synchronize()
                recs.append(e0.elapsed_time(e1) / reps)
            step.free()
            med, b2b, rep_ms = float(np.median(meds)), float(np.median(b2bs)), float(np.median(recs))
            fl = 2.0 * n ** 3
            out[dt_name][str(n)] = [round(med * 1e3, 1), round(b2b * 1e3, 1), round(rep_ms * 1e3, 1),
                                    round(fl / (rep_ms * 1e-3) / 1e12, 1),
                                    tg.tile_gemm_query_config(n, n, n, tg.OUT_BF16)["config"]]
            del bufs
            torch.cuda.empty_cache()
    return out


def bench_cublas_context(tg, torch, case, seconds=1.0, pause=2.5):
    """CONTEXT, not product path: torch.matmul (cuBLAS) and tile_gemm on cfg3 under ONE protocol in this very run, so that
    the roofline fraction (whose denominator MEASURED_PEAKS.json was taken on another day, possibly another box: the pool's
    B200s differ by +-5 % under the power cap) can be read next to a same-box, same-minute ratio.  Burst = 20 launches after
    `pause` seconds of idle and 5 warm-up launches; sustained = back to back for `seconds` right after 0.35 s of the same."""
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(1000 + case.seed[0])
    sets = 4
    bufs = [(torch.empty((case.M, case.K), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_a, generator=g),
             torch.empty((case.K, case.N), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_b, generator=g),
             torch.empty((case.M, case.N), dtype=torch.bfloat16, device=dev)) for _ in range(sets)]
    flops = 2.0 * case.M * case.N * case.K

    def run(kind, k):
        for i in range(k):
            A, B, C = bufs[i % sets]
            if kind == "cublas":
                torch.matmul(A, B, out=C)
            else:
                tg.tile_gemm(A, B, C)

    def timed(kind, k):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        run(kind, k)
        e1.record()
        torch.cuda.synchronize()
        return flops / (e0.elapsed_time(e1) / k * 1e-3) / 1e12

    out = {"note": "context only: torch.matmul (cuBLAS) is not on the product path"}
    for kind in ("cublas", "tile_gemm", "cublas", "tile_gemm"):
        time.sleep(pause)
        run(kind, 5)
        torch.cuda.synchronize()
        out.setdefault(kind + "_burst_tflops", []).append(round(timed(kind, 20), 1))
    for kind in ("tile_gemm", "cublas", "cublas", "tile_gemm"):
        t_end = time.perf_counter() + 0.35
        while time.perf_counter() < t_end:
            run(kind, 16)
            torch.cuda.synchronize()
        k = max(16, int(seconds / 0.8e-3))
        out.setdefault(kind + "_sustained_tflops", []).append(round(timed(kind, k), 1))
    out["burst_ratio"] = round(max(out["tile_gemm_burst_tflops"]) / max(out["cublas_burst_tflops"]), 4)
    out["sustained_ratio"] = round(sum(out["tile_gemm_sustained_tflops"]) / sum(out["cublas_sustained_tflops"]), 4)
    del bufs
    torch.cuda.empty_cache()
    return out


def bench_sustained(tg, torch, case, seconds, local_rank, tdist):
    """cfg3 back to back for >= `seconds`: the figure to hold against MEASURED_PEAKS.json's sustained
    cuBLAS number (a seconds-long loop under the power cap), with its own clock record."""
    dev = torch.device("cuda", torch.cuda.current_device())
    g = torch.Generator(device=dev)
    g.manual_seed(1000 + case.seed[0])
    sets = 4
    bufs = [(torch.empty((case.M, case.K), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_a, generator=g),
             torch.empty((case.K, case.N), dtype=torch.bfloat16, device=dev).normal_(0, case.sigma_b, generator=g),
             torch.empty((case.M, case.N), dtype=torch.bfloat16, device=dev)) for _ in range(sets)]
    for i in range(8):
        tg.tile_gemm(*bufs[i % sets])
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tdist.barrier()
    steps = 0
    with sampler:
        t_end = time.perf_counter() + seconds
        e0.record()
        while time.perf_counter() < t_end:
            for _ in range(64):
                tg.tile_gemm(*bufs[steps % sets])
                steps += 1
            torch.cuda.synchronize()      # bounded queue: the loop ends when the clock says so
        e1.record()
        torch.cuda.synchronize()
    ms = tdist.max_over_ranks(e0.elapsed_time(e1))
    del bufs
    torch.cuda.empty_cache()
    return ms / steps, steps, ms, sampler.summary()


def run_cuda(args):
    import torch
    from paper_2606_15991_b200 import binding as tg
    from paper_2606_15991_b200 import dist as tdist
    from paper_2606_15991_b200 import workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    rank, local_rank, world = tdist.init()
    if world != args.gpus and rank == 0:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s); reporting n_gpus = {world}\n")
    torch.cuda.set_device(local_rank)
    tg.load_library()
    if args.gemm_config:
        tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, args.gemm_config)
    if args.group_m:
        tg.tile_gemm_set_tuning(tg.TUNE_GEMM_GROUP_M, args.group_m)
    peaks = measured_peaks()
    case = wl.CFG3
    flops = 2.0 * case.M * case.N * case.K

    sampler = ClockSampler(local_rank)
    ms_step, launches, bufs = bench_gemm(tg, wl, torch, case, args.steps, args.warmup, 4, tdist, sampler)
    clocks = sampler.summary()
    value = world * flops / (ms_step * 1e-3) / 1e12
    per_gpu = flops / (ms_step * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": WORKLOAD, "l2": L2_NOTE, "tile_config": tg.tile_gemm_query_config(case.M, case.N, case.K, tg.OUT_BF16),
                   "parallelism": f"{world} independent replicas, no collective"},
        "clocks": clocks,
        "gpu_launches": int(launches * world),
        "roofline": {"bound": "tensor", "achieved": per_gpu, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                     "frac": per_gpu / peaks["bf16_tflops"], "traffic": ncu_traffic("gemm_8192_dram_bytes"),
                     "peak_source": f"{peaks['source']} cuBLAS bf16 burst (MEASURED_PEAKS.json): the --steps leg is a burst",
                     "frac_of_nominal_2250": per_gpu / 2250.0,
                     "kernel": "gemm_tcgen05_kernel<2,256,4,2,false,0>", "algorithmic_flops_per_launch": flops},
    }
    del bufs
    torch.cuda.empty_cache()
    if not args.no_sustained:
        # the same step back to back for seconds: what MEASURED_PEAKS.json's sustained cuBLAS figure is measured like
        s_ms, s_steps, s_total, s_clocks = bench_sustained(tg, torch, case, args.sustained_seconds, local_rank, tdist)
        s_tf = flops / (s_ms * 1e-3) / 1e12
        line["roofline"]["sustained"] = {
            "achieved": s_tf, "peak": peaks["bf16_tflops_sustained"], "frac": s_tf / peaks["bf16_tflops_sustained"],
            "unit": "TFLOP/s", "ms_per_step": s_ms, "steps": s_steps, "seconds": s_total * 1e-3, "clocks": s_clocks,
            "peak_source": f"{peaks['source']} cuBLAS bf16 back to back for seconds (MEASURED_PEAKS.json)"}

    if rank == 0 and world == 1 and not (args.no_cublas_context or args.no_sustained or args.headline_only):
        line["roofline"]["cublas_same_run"] = bench_cublas_context(tg, torch, case)

    if rank == 0 and not args.no_e2e:
        dt, h2d, d2h, _ = bench_e2e(tg, wl, torch, case, max(2, min(args.steps, 5)))
        line["e2e"] = {"value": flops / dt / 1e12, "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3,
                       "api": "tile_gemm_host (pinned host A,B,C; H2D + GEMM + D2H per step)"}
    tdist.barrier()

    gemv_rec = probe_rec = None
    if not args.headline_only:
        # config[3]: prefill projections
        pre = {}
        tot_ms, tot_fl = 0.0, 0.0
        for c in wl.CFG4:
            ms, _, b = bench_gemm(tg, wl, torch, c, max(5, args.steps // 4), 3, 2, tdist)
            del b
            torch.cuda.empty_cache()
            fl = 2.0 * c.M * c.N * c.K
            pre[c.name] = {"ms": round(ms, 4), "tflops": round(fl / (ms * 1e-3) / 1e12, 1)}
            tot_ms += ms
            tot_fl += fl
        pre["aggregate_tflops"] = tot_fl / (tot_ms * 1e-3) / 1e12
        pre["frac_of_measured_peak"] = pre["aggregate_tflops"] / peaks["bf16_tflops"]
        line["prefill"] = pre
        # config[4]: decode GEMV sequence
        ms, alg_bytes, gl, per_shape, graph_ms, n, plain_ms = bench_decode(tg, wl, torch, args.decode_passes, 2,
                                                                           args.decode_layers, tdist)
        gbs = alg_bytes / (ms * 1e-3) / 1e9
        gemv_rec = {
            "metric": "decode_gemv_hbm_gbs", "value": gbs * world, "unit": "GB/s", "ms_per_pass": ms,
            "launches_per_pass": n, "layers": args.decode_layers, "algorithmic_bytes_per_pass": alg_bytes,
            "api": "tile_gemm_static_b, plain stream launches (weights immutable: tiles are prefetched ahead of the PDL wait)",
            "plain_tile_gemm": {"ms_per_pass": plain_ms, "gbs": alg_bytes / (plain_ms * 1e-3) / 1e9},
            "per_shape": per_shape,
            "recorded_step_replay": None if graph_ms is None else {"ms_per_pass": graph_ms,
                                                           "gbs": alg_bytes / (graph_ms * 1e-3) / 1e9},
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / peaks["hbm_gbs"], "traffic": ncu_traffic("gemv_gate_up_dram_bytes"),
                         "peak_source": f"{peaks['source']} copy bandwidth (MEASURED_PEAKS.json)",
                         "frac_of_8000": gbs / 8000.0, "kernel": "gemv_split_kernel<256,64,3,2>"},
        }
        # what a pure streaming read achieves on this box (4 GiB, every word once)
        dev0 = torch.device("cuda", torch.cuda.current_device())
        pbuf = torch.empty(1 << 30, dtype=torch.int32, device=dev0).random_(0, 1 << 30)
        pout = torch.zeros(1, dtype=torch.int64, device=dev0)
        for _ in range(2):
            tg.tile_read_probe_u32(pbuf, pout)
        preps = 10
        pms = tdist.max_over_ranks(time_region(lambda i: tg.tile_read_probe_u32(pbuf, pout), preps,
                                               torch.cuda.synchronize, tdist.barrier)) / preps
        probe_gbs = pbuf.numel() * 4 / (pms * 1e-3) / 1e9
        del pbuf
        torch.cuda.empty_cache()
        probe_rec = {"gbs": probe_gbs, "bytes": 4 << 30, "kernel": "read_probe_kernel (tile_read_probe_u32)"}
        gemv_rec["roofline"]["frac_of_read_probe"] = gemv_rec["roofline"]["achieved"] / probe_gbs
        # the GEMV half of BASELINE.json's metric, also inside the top-level roofline record
        line["roofline"]["gemv"] = {k: gemv_rec["roofline"][k] for k in
                                    ("bound", "achieved", "peak", "unit", "frac", "frac_of_8000", "frac_of_read_probe", "kernel")}
        # element-wise add (Listing 1) at n = 2^28
        n_add = 1 << 28
        ms = bench_add(tg, torch, n_add, max(10, args.steps // 4), 3, tdist)
        gbs = 12.0 * n_add / (ms * 1e-3) / 1e9
        line["add"] = {
            "metric": "elementwise_add_f32_hbm_gbs", "value": gbs * world, "unit": "GB/s", "n": n_add,
            "us_per_launch": ms * 1e3, "paper_b200_gbs": 6970.0,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": gbs / peaks["hbm_gbs"], "traffic": ncu_traffic("add_2p28_dram_bytes"),
                         "peak_source": f"{peaks['source']} copy bandwidth (MEASURED_PEAKS.json)",
                         "frac_of_8000": gbs / 8000.0, "kernel": "add_f32_vec_kernel<1,4,true>",
                         "algorithmic_bytes_per_launch": 12 * n_add},
        }
        # per-op host cost, stream launches vs one recorded step
        if rank == 0:
            line["replay"] = {k: (round(v, 3) if isinstance(v, float) else v) for k, v in bench_launch_overhead(tg, torch).items()}
        tdist.barrier()
        # fused gate/up + SwiGLU epilogue on the cfg4 gate_up shape vs the plain GEMM that writes [gate | up]
        c = wl.CFG4[2]
        dev = torch.device("cuda", torch.cuda.current_device())
        gg = torch.Generator(device=dev)
        gg.manual_seed(55)
        Xs = [torch.empty((c.M, c.K), dtype=torch.bfloat16, device=dev).normal_(0, 1, generator=gg) for _ in range(2)]
        Wsw = [torch.empty((c.K, c.N), dtype=torch.bfloat16, device=dev).normal_(0, 0.02, generator=gg) for _ in range(2)]
        Hs = torch.empty((c.M, c.N // 2), dtype=torch.bfloat16, device=dev)
        Cp = torch.empty((c.M, c.N), dtype=torch.bfloat16, device=dev)
        reps = max(5, args.steps // 8)
        for i in range(3):
            tg.tile_gemm_swiglu(Xs[i % 2], Wsw[i % 2], Hs)
            tg.tile_gemm(Xs[i % 2], Wsw[i % 2], Cp)
        ms_f = tdist.max_over_ranks(time_region(lambda i: tg.tile_gemm_swiglu(Xs[i % 2], Wsw[i % 2], Hs), reps,
                                                torch.cuda.synchronize, tdist.barrier)) / reps
        ms_p = tdist.max_over_ranks(time_region(lambda i: tg.tile_gemm(Xs[i % 2], Wsw[i % 2], Cp), reps,
                                                torch.cuda.synchronize, tdist.barrier)) / reps
        fl = 2.0 * c.M * c.N * c.K
        line["swiglu"] = {"shape": f"M={c.M} K={c.K} 2I={c.N}", "fused_ms": round(ms_f, 4), "fused_tflops": round(fl / (ms_f * 1e-3) / 1e12, 1),
                          "plain_gate_up_gemm_ms": round(ms_p, 4), "plain_tflops": round(fl / (ms_p * 1e-3) / 1e12, 1),
                          "c_bytes_fused": c.M * c.N, "c_bytes_plain": 2 * c.M * c.N}
        del Xs, Wsw, Hs, Cp
        torch.cuda.empty_cache()
        # skinny M
        line["skinny_m"] = bench_skinny(tg, wl, torch, [2, 4, 8, 16, 32, 64], tdist)
        # the paper's size sweep in f16 and bf16
        if not args.no_sweep:
            line["sweep"] = bench_sweep(tg, torch, [1024, 2048, 4096, 8192, 16384, 32768], tdist)
    # the GEMV half of the metric goes LAST (before the short cpu_baseline record), so that it is in the
    # final kilobytes of the line whatever the other legs print
    if gemv_rec is not None:
        line["read_probe"] = probe_rec
        if gemv_rec["roofline"]["frac"] > 1.0:
            note = ("above 1 because the peak is MEASURED_PEAKS.json's COPY bandwidth (read + write streams); a pure read "
                    "stream runs faster on this part: the ceiling to read it against is frac_of_read_probe")
            gemv_rec["roofline"]["frac_note"] = note
            line["roofline"]["gemv"]["frac_note"] = note
        line["gemv"] = gemv_rec
    # the steady-state figures once more, as short top-level records at the END of the line (the roofline object that
    # holds the full versions is printed kilobytes earlier)
    sus = line["roofline"].get("sustained")
    if sus is not None:
        line["sustained"] = {"achieved": round(sus["achieved"], 1), "peak": sus["peak"], "frac": round(sus["frac"], 4),
                             "unit": "TFLOP/s", "seconds": round(sus["seconds"], 2),
                             "sm_mhz": (sus.get("clocks") or {}).get("sm_mhz"), "reasons": (sus.get("clocks") or {}).get("reasons")}
    ctx = line["roofline"].get("cublas_same_run")
    if ctx is not None:
        line["cublas_same_run"] = {"burst_ratio": ctx["burst_ratio"], "sustained_ratio": ctx["sustained_ratio"],
                                   "note": "tile_gemm / torch.matmul on cfg3 in this run; context only"}
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline_leg()
        print(json.dumps(line), flush=True)
    tdist.barrier()
    tdist.shutdown()
    return 0


def spawn_ranks(n):
    """`python bench.py --gpus N` with no torchrun environment: start the N ranks ourselves, exactly the way the
    driver's torchrun form does (one process per GPU, rendezvous on 127.0.0.1), with this command line."""
    import socket
    import subprocess
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_rendezvous(args):
    """The N > 1 plumbing without the kernels: every rank joins, the ranks meet at a barrier, and rank 0 prints how
    many arrived and the max / sum of their rank numbers (what the timing scalars travel through)."""
    from paper_2606_15991_b200 import dist as tdist
    rank, local_rank, world = tdist.init()
    tdist.barrier()
    top = tdist.max_over_ranks(float(rank))
    total = tdist.sum_over_ranks(float(rank + 1))
    if rank == 0:
        print(json.dumps({"rendezvous": world, "gpus_flag": args.gpus, "max_rank": top, "sum_rank_plus_1": total,
                          "impl": args.impl}), flush=True)
    tdist.barrier()
    tdist.shutdown()
    return 0 if world == args.gpus else 1


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--decode-passes", type=int, default=5)
    ap.add_argument("--decode-layers", type=int, default=64)
    ap.add_argument("--headline-only", action="store_true", help="skip the prefill and decode legs")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the f16/bf16 size sweep (SURVEY 8(f)1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", action="store_true", help="skip the seconds-long back-to-back cfg3 leg")
    ap.add_argument("--no-cublas-context", action="store_true", help="skip the same-run cuBLAS context figures (torch.matmul)")
    ap.add_argument("--sustained-seconds", type=float, default=2.5)
    ap.add_argument("--gemm-config", type=int, default=0, help="force a GEMM tile config (tile_gemm_set_tuning key 0)")
    ap.add_argument("--group-m", type=int, default=0, help="force the raster group height (tuning key 1)")
    ap.add_argument("--rendezvous-only", action="store_true",
                    help="start the ranks, rendezvous (NCCL on GPUs, gloo on a CPU box), print the world that met, and exit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args.gpus)
    if args.rendezvous_only:
        return run_rendezvous(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
