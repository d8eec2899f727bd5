"""Where a tiled-GEMM launch spends its time, from the kernel's own clock (tile_gemm_debug_trace).

    python -m paper_2606_15991_b200.gemm_trace [N ...]        # default: 4096 8192 16384, bf16 in / bf16 out

For every size and tile configuration it prints, averaged over the clusters of one launch (after warm-up): how long
the MMA issuer's loop ran, what share of it the issuer waited for accumulator slots (the epilogue drain that a
two-slot tile cannot hide), clock cycles per k-tile against the tensor pipe's 1024 (8 MMAs of
128 cycles), and how long one epilogue warp needs from "accumulator full" to "slot handed back".  Needs a B200.
"""
from __future__ import annotations

import sys

import torch

from . import binding as tg


def trace_once(n: int, cfg: int, dev) -> str:
    g = torch.Generator(device=dev)
    g.manual_seed(3)
    A = torch.empty((n, n), dtype=torch.bfloat16, device=dev).normal_(0, 1, generator=g)
    B = torch.empty((n, n), dtype=torch.bfloat16, device=dev).normal_(0, n ** -0.5, generator=g)
    C = torch.empty((n, n), dtype=torch.bfloat16, device=dev)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    for _ in range(30):
        tg.tile_gemm(A, B, C)
    torch.cuda.synchronize()
    rec = torch.zeros((256, 8), dtype=torch.int64, device=dev)
    tg.tile_gemm_debug_trace(rec)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    tg.tile_gemm(A, B, C)
    e1.record()
    torch.cuda.synchronize()
    tg.tile_gemm_debug_trace(None)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, 0)
    r = rec.cpu().double()
    r = r[r[:, 2] > 0]
    _, acc, tot, nk, drain, tiles = (r[:, i] for i in range(6))
    us = e0.elapsed_time(e1) * 1e3
    return (f"| {n} | {cfg} | {us:.0f} | {len(r)} | {tot.mean():.0f} | {100 * (acc / tot).mean():.1f} % | {(acc / tiles).mean():.0f} | "
            f"{(drain / tiles).mean():.0f} | {(tot / nk).mean():.0f} | {tot.mean() / us / 1e3:.2f} |")


def main(argv):
    sizes = [int(a) for a in argv] or [4096, 8192, 16384]
    dev = torch.device("cuda", torch.cuda.current_device())
    print("| M=N=K | tile config | launch us | clusters | issuer loop clk | waiting for accumulator slots | clk per tile | "
          "epilogue drain clk per tile | clk per k-tile | SM clock GHz |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for n in sizes:
        for cfg in (4, 3):
            print(trace_once(n, cfg, dev), flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
