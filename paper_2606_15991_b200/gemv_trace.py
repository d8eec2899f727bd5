"""Timeline of the M = 1 decode kernel inside a chain of launches (tile_gemm_debug_trace).

    python -m paper_2606_15991_b200.gemv_trace [--fixup 0|1|2|3] [--l2-post N] [--layers L] [--shapes 0,1,2,3]

For each of the four Qwen3-32B weight shapes (BASELINE.json config 5) it records one step of L
back-to-back GEMVs on distinct weight buffers (tile_gemm_static_b, programmatic dependent launch),
with a fresh trace buffer per launch, replays it, and prints per launch where the CTAs were in
time -- kernel entry, first tile in shared memory, last tile consumed, partial sums handed over,
CTA done -- as min / p10 / median / p90 / max microseconds relative to the moment the launch's
dependency wait released.  The period (last CTA done of launch k-1 to last CTA done of launch k)
is the launch's real cost inside the stream.  PAPER.md:347 gives decode its roofline (weights
streamed once); this shows what separates a launch from it: the hand-over of the split-K partial
sums after the last tile, the spread of the CTAs' finish times, and the gap between launches.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import binding as tg
from . import workloads as wl


def pct(a, rel):
    a = (a - rel) / 1e3
    return f"{a.min():6.2f}/{np.percentile(a, 10):6.2f}/{np.median(a):6.2f}/{np.percentile(a, 90):6.2f}/{a.max():6.2f}"


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--fixup", type=int, default=0, help="tuning key 8: 0 auto, 1 tickets, 2 tagged slots, 3 cluster")
    ap.add_argument("--l2-post", type=int, default=0, help="tuning key 9 (n >= 1: n - 1 tiles into L2 behind the wait)")
    ap.add_argument("--layers", type=int, default=10)
    ap.add_argument("--shapes", default="0,1,2,3")
    args = ap.parse_args(argv)
    dev = torch.device("cuda", torch.cuda.current_device())
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, args.fixup)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_L2_POST, args.l2_post)
    names = {0: "automatic", 1: "tickets", 2: "tagged slots (else tickets)", 3: "cluster + DSMEM (else tickets)"}
    print(f"split-K hand-over: {names.get(args.fixup, args.fixup)}; columns are min/p10/median/p90/max in us after the "
          f"launch's dependency wait released")
    g = torch.Generator(device=dev)
    g.manual_seed(4)
    for p in [int(v) for v in args.shapes.split(",")]:
        K, N = wl.QWEN3_32B[p]
        L = args.layers
        items = [(torch.empty((1, K), dtype=torch.bfloat16, device=dev).normal_(0, 1, generator=g),
                  torch.empty((K, N), dtype=torch.bfloat16, device=dev).normal_(0, 0.02, generator=g),
                  torch.empty((1, N), dtype=torch.bfloat16, device=dev)) for _ in range(L)]
        bufs = [torch.zeros((4096, 8), dtype=torch.int64, device=dev) for _ in range(L)]
        s = torch.cuda.Stream()
        tg.tile_gemm_record_begin(s)
        for (x, W, y), b in zip(items, bufs):
            tg.tile_gemm_debug_trace(b)
            tg.tile_gemm(x, W, y, static_b=True, stream=s)
        step = tg.tile_gemm_record_end(s)
        tg.tile_gemm_debug_trace(None)
        for _ in range(3):
            step.replay(s)
        s.synchronize()
        T = [b.cpu().numpy() for b in bufs]
        T = [t[t[:, 1] > 0] for t in T]
        byt = 2 * K * N + 2 * K + 2 * N
        slices = int((T[0][:, 0] >> 32).max()) + 1
        print(f"\n## K={K} N={N}: {len(T[0])} CTAs = {len(T[0]) // slices} column blocks x {slices} slices, {byt / 1e6:.1f} MB per launch")
        print("| launch | period us | GB/s | previous launch's last CTA done | CTA start | first tile | last tile consumed | partials handed over | CTA done | combiner CTAs: done |")
        print("|---|---|---|---|---|---|---|---|---|---|")
        periods = []
        for k in range(3, L):
            t = T[k]
            rel = t[:, 2].min()
            prev_end = T[k - 1][:, 5].max()
            per = (t[:, 5].max() - prev_end) / 1e3
            periods.append(per)
            handed = t[:, 7][t[:, 7] > 0]
            comb = t[(t[:, 7] > 0) & ((t[:, 5] - t[:, 7]) > 500)]
            print(f"| {k} | {per:.2f} | {byt / per / 1e3:.0f} | {(prev_end - rel) / 1e3:.2f} | {pct(t[:, 1], rel)} | {pct(t[:, 3], rel)} | "
                  f"{pct(t[:, 4], rel)} | {pct(handed, rel) if len(handed) else '-'} | {pct(t[:, 5], rel)} | "
                  f"{pct(comb[:, 5], rel) if len(comb) else '-'} |")
        per = float(np.median(periods))
        print(f"\nmedian period {per:.2f} us = {byt / per / 1e3:.0f} GB/s")
        step.free()
        del items, bufs
        torch.cuda.empty_cache()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
