"""Lifetime and liveness of the library's own state, on a B200 through the C ABI:

* a recorded step owns its workspaces ("replayed nodes do not depend on addresses that change
  across replays") -- it survives larger shapes on the recording stream, replays on
  another stream and overlaps with direct calls;
* the lockstep producers of the persistent GEMM never hang when their clusters are not all
  resident (the lockstep is a locality hint, PAPER.md:161-163 only needs one owner per tile);
* tile_gemm_host is safe to call from several host threads.
Every result is compared with the fp64 oracle (integer-valued inputs: bit-exact).
"""
import threading
import time

import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl
from parity import check_bit_exact

pytestmark = pytest.mark.gpu
DEV = "cuda"


@pytest.fixture(autouse=True)
def _reset_tuning():
    yield
    for key in range(tg.NUM_TUNE_KEYS):
        tg.tile_gemm_set_tuning(key, 0)
    torch.cuda.synchronize()


def _int_case(M, N, K, seed):
    a, b = wl.make_inputs_custom(M, N, K, "int4", seed=seed)
    ref, _ = oracle.gemm(a, b)
    return wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV), ref


def test_recorded_step_owns_its_workspaces():
    """Record (with NO warm-up on the stream) a K-sliced GEMM, a split-K GEMV, a skinny-M weight-streaming
    GEMM (cluster hand-over: no workspace at all) and a GEMM whose B has an odd row stride (repack workspace); then run 4x larger split shapes directly on
    the recording stream, which regrows that stream's workspaces; then replay -- on the recording
    stream, and on a second stream while direct split-K calls keep the first one busy."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, 5)        # K slices for the GEMV column blocks and the GEMM's last wave
    s, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    A1, B1, ref1 = _int_case(130, 384, 2048, 301)         # GEMM, partial last wave cut into 5 slices
    x2, B2, ref2 = _int_case(1, 1536, 2560, 302)          # M = 1, 5 slices per column block
    A3, B3, ref3 = _int_case(3, 1024, 1280, 303)          # M = 3: the weight-streaming tensor-core kernel
    a4, b4 = wl.make_inputs_custom(140, 200, 264, "int4", seed=304)
    ref4, _ = oracle.gemm(a4, b4)
    A4 = wl.bits_to_torch(a4, DEV)
    B4full = torch.zeros((264, 203), dtype=torch.bfloat16, device=DEV)   # ldb = 203: not TMA-addressable
    B4full[:, :200] = wl.bits_to_torch(b4, DEV)
    B4 = B4full[:, :200]
    outs = [torch.empty(r.shape, dtype=torch.float32, device=DEV) for r in (ref1, ref2, ref3, ref4)]

    def chain(stream):
        tg.tile_gemm(A1, B1, outs[0], stream=stream)
        tg.tile_gemm(x2, B2, outs[1], stream=stream, static_b=True)
        tg.tile_gemm(A3, B3, outs[2], stream=stream)
        tg.tile_gemm(A4, B4, outs[3], stream=stream)

    def check(tag):
        for i, ref in enumerate((ref1, ref2, ref3, ref4)):
            check_bit_exact(outs[i].cpu().numpy(), ref, f"{tag}: call {i}")
            outs[i].fill_(float("nan"))
        torch.cuda.synchronize()

    tg.tile_gemm_record_begin(s)
    chain(s)
    step = tg.tile_gemm_record_end(s)
    assert step.nodes >= 4
    step.replay(s)
    s.synchronize()
    check("first replay")

    # larger split shapes directly on the recording stream: its own workspaces are created / regrown
    Ab, Bb, refb = _int_case(260, 1536, 4096, 305)
    xb, Wb, refg = _int_case(1, 6144, 5120, 306)
    Cb = torch.empty(refb.shape, dtype=torch.float32, device=DEV)
    yb = torch.empty(refg.shape, dtype=torch.float32, device=DEV)
    for _ in range(2):
        tg.tile_gemm(Ab, Bb, Cb, stream=s)
        tg.tile_gemm(xb, Wb, yb, stream=s, static_b=True)
    s.synchronize()
    check_bit_exact(Cb.cpu().numpy(), refb, "direct large GEMM")
    check_bit_exact(yb.cpu().numpy(), refg, "direct large GEMV")
    step.replay(s)
    s.synchronize()
    check("replay after the stream's workspaces grew")

    # replay on another stream while direct split-K calls run on the recording stream
    for _ in range(6):
        tg.tile_gemm(Ab, Bb, Cb, stream=s)
        tg.tile_gemm(xb, Wb, yb, stream=s, static_b=True)
        step.replay(s2)
    s.synchronize()
    s2.synchronize()
    check_bit_exact(Cb.cpu().numpy(), refb, "direct large GEMM next to a replay")
    check_bit_exact(yb.cpu().numpy(), refg, "direct large GEMV next to a replay")
    check("replay on a second stream next to direct calls")
    step.free()
    assert step.nodes == -1
    # and the stream still works after the step is gone
    chain(s)
    s.synchronize()
    check("direct calls after record_free")


def test_record_state_errors():
    lib = tg.load_library()
    import ctypes
    s = torch.cuda.Stream()
    out = ctypes.c_void_p()
    assert lib.tile_gemm_record_end(ctypes.c_void_p(s.cuda_stream), ctypes.byref(out)) == tg.E_PATH   # not recording
    tg.tile_gemm_record_begin(s)
    assert lib.tile_gemm_record_begin(ctypes.c_void_p(s.cuda_stream)) == tg.E_PATH                     # already recording
    step = tg.tile_gemm_record_end(s)
    assert step.nodes == 0
    step.free()


def test_caller_capture_uses_the_stream_workspaces_and_refuses_to_grow():
    """A stream captured by the caller (not through tile_gemm_record_*) keeps the round-1 contract:
    the workspaces must exist beforehand; a call that would grow one fails with a clear message."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, 4)
    s = torch.cuda.Stream()
    x, W, ref = _int_case(1, 1024, 2048, 311)
    y = torch.empty((1, 1024), dtype=torch.float32, device=DEV)
    NL = 1 << 18                                          # 1024 column blocks x 4 slices of partial sums: beyond the first 1 MB
    xl = torch.ones((1, 256), dtype=torch.bfloat16, device=DEV)
    Wl = torch.ones((256, NL), dtype=torch.bfloat16, device=DEV)
    yl = torch.empty((1, NL), dtype=torch.float32, device=DEV)
    tg.tile_gemm(x, W, y, stream=s)                      # the small shape's workspace exists
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s, capture_error_mode="relaxed"):
        tg.tile_gemm(x, W, y, stream=s)
        with pytest.raises(tg.TileGemmError) as ei:
            tg.tile_gemm(xl, Wl, yl, stream=s)            # would have to grow under a foreign capture
        assert ei.value.status == tg.E_CUDA and "capture" in ei.value.message
    y.fill_(float("nan"))
    tg.tile_gemm(xl, Wl, yl, stream=s)                   # grows the pinned set: the old buffer is retired, not freed
    g.replay()
    torch.cuda.synchronize()
    check_bit_exact(y.cpu().numpy(), ref, "caller-captured GEMV after the workspace grew")
    assert torch.all(yl == 256.0)


@pytest.mark.parametrize("cfg", [3, 4])
def test_lockstep_does_not_hang_when_clusters_are_not_resident(cfg):
    """60 SMs are held by another kernel for 40 ms; a persistent GEMM with lockstep producers forced
    on (window 4) starts next to it, so a good part of its clusters cannot be resident.  The
    producers that are running give up waiting for the missing ones after GEMM_LOCKSTEP_PATIENCE_NS
    and the launch completes with the same bits."""
    M, N, K = 2048, 4096, 1024
    A, B, ref = _int_case(M, N, K, 320 + cfg)
    C = torch.empty((M, N), dtype=torch.float32, device=DEV)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, 4 | (4 << 8))
    plan = tg.tile_gemm_query_plan(M, N, K)
    assert plan["lockstep_rounds"] >= 1
    tg.tile_gemm(A, B, C)                                 # alone: all clusters resident
    torch.cuda.synchronize()
    check_bit_exact(C.cpu().numpy(), ref, "lockstep GEMM alone")
    C.fill_(float("nan"))
    blocker, worker = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    tg.tile_gemm_debug_occupy(60, 40_000_000, stream=blocker)
    tg.tile_gemm(A, B, C, stream=worker)
    worker.synchronize()
    dt_gemm = time.perf_counter() - t0
    blocker.synchronize()
    check_bit_exact(C.cpu().numpy(), ref, "lockstep GEMM next to a kernel holding 60 SMs")
    assert dt_gemm < 1.0, f"the GEMM took {dt_gemm:.3f} s next to the blocker"


def test_host_entry_from_two_threads():
    """tile_gemm_host serialises concurrent callers: two host threads, different shapes, 6 calls each."""
    cases = []
    for i, (M, N, K) in enumerate([(2304, 640, 512), (700, 1100, 300)]):
        a, b = wl.make_inputs_custom(M, N, K, "int4", seed=330 + i)
        ref, _ = oracle.gemm(a, b)
        cases.append((a, b, ref))
    errors = []

    def worker(idx):
        try:
            a, b, ref = cases[idx]
            for _ in range(6):
                out = np.full(ref.shape, np.nan, dtype=np.float32)
                tg.tile_gemm_host(a, b, out)
                check_bit_exact(out, ref, f"host thread {idx}")
        except BaseException as exc:  # noqa: BLE001 - reported by the main thread
            errors.append((idx, exc))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


@pytest.mark.parametrize("fix,split", [(1, 10), (2, 10), (3, 4)])
def test_gemv_trace_on_leaves_the_result_alone_and_fills_sane_records(fix, split):
    """tile_gemm_debug_trace on an M = 1 launch in each hand-over protocol (tickets, tagged slots, cluster):
    y keeps its bits, every CTA of the launch writes its record, the time stamps are ordered, and the
    tiles the CTAs report add up to column blocks x k-tiles.  The binding holds the buffer while it is set."""
    K, N = 2560, 2048                                   # 8 column blocks of 256, 40 k-tiles of 64
    x, B, ref = _int_case(1, N, K, 411)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, fix)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, split)
    y0 = tg.tile_gemm(x, B)
    torch.cuda.synchronize()
    rec = torch.zeros((128, 8), dtype=torch.int64, device=DEV)
    tg.tile_gemm_debug_trace(rec)
    assert tg._trace_ref is rec
    try:
        y1 = tg.tile_gemm(x, B)
        torch.cuda.synchronize()
    finally:
        tg.tile_gemm_debug_trace(None)
    assert tg._trace_ref is None
    check_bit_exact(y1.cpu().numpy(), ref, f"traced GEMV, fix-up {fix}")
    assert torch.equal(y0, y1)
    r = rec.cpu().numpy()
    ctas = 8 * split
    used, rest = r[:ctas], r[ctas:]
    assert (rest == 0).all(), "records past the launch's CTAs were written"
    assert sorted((int(w) >> 16) & 0xFFFF | ((int(w) >> 32) << 16) for w in used[:, 0]) == \
        sorted(bx | (by << 16) for by in range(split) for bx in range(8))
    t = used[:, 1:6]
    assert (t > 0).all() and (np.diff(t, axis=1) >= 0).all(), "time stamps out of order"
    assert (t[:, 4] - t[:, 0] < 5_000_000).all(), "a CTA of a 10 MB GEMV took more than 5 ms"
    assert int(used[:, 6].sum()) == 8 * 40
    assert ((used[:, 7] >= t[:, 3]) & (used[:, 7] <= t[:, 4])).all(), "hand-over stamp outside [last tile, done]"
    # a later launch without tracing leaves the buffer alone
    rec.zero_()
    tg.tile_gemm(x, B)
    torch.cuda.synchronize()
    assert (rec == 0).all()


@pytest.mark.parametrize("cfg", [3, 4])
def test_gemm_trace_on_leaves_the_result_alone_and_counts_the_k_tiles(cfg):
    M, N, K = 1024, 1024, 1024
    A, B, ref = _int_case(M, N, K, 412)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, 1)      # whole tiles only
    q = tg.tile_gemm_query_config(M, N, K)
    tiles = -(-M // (q["BM"] * q["cta_group"])) * -(-N // q["BN"])
    rec = torch.zeros((256, 8), dtype=torch.int64, device=DEV)
    tg.tile_gemm_debug_trace(rec)
    try:
        C = tg.tile_gemm(A, B)
        torch.cuda.synchronize()
    finally:
        tg.tile_gemm_debug_trace(None)
    check_bit_exact(C.cpu().numpy(), ref, f"traced GEMM, config {cfg}")
    r = rec.cpu().numpy()
    live = r[r[:, 2] > 0]
    assert len(live) == min(tiles, q["ctas"] // q["cta_group"])
    assert (live[:, 1] <= live[:, 2]).all() and (live[:, 2] < 50_000_000).all()
    assert int(live[:, 3].sum()) == tiles * (K // q["BK"])
    assert int(live[:, 5].sum()) >= tiles and (live[:, 4] > 0).all()


def test_recorded_step_takes_no_trace_pointer():
    """A step recorded while tracing is on must not keep the trace buffer's address: after the buffer is gone
    a replay would write into freed memory.  Launches under record_begin get a null trace pointer."""
    x, B, ref = _int_case(1, 1536, 2560, 413)
    A2, B2, ref2 = _int_case(256, 512, 512, 414)
    y = torch.empty((1, 1536), dtype=torch.float32, device=DEV)
    C2 = torch.empty((256, 512), dtype=torch.float32, device=DEV)
    tg.tile_gemm(x, B, y)                                # workspaces exist before the recording
    tg.tile_gemm(A2, B2, C2)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    rec = torch.zeros((256, 8), dtype=torch.int64, device=DEV)
    tg.tile_gemm_debug_trace(rec)
    try:
        tg.tile_gemm_record_begin(s)
        tg.tile_gemm(x, B, y, stream=s)
        tg.tile_gemm(A2, B2, C2, stream=s)
        step = tg.tile_gemm_record_end(s)
    finally:
        tg.tile_gemm_debug_trace(None)
    y.fill_(float("nan"))
    C2.fill_(float("nan"))
    step.replay(s)
    s.synchronize()
    assert (rec == 0).all(), "a recorded launch wrote trace records"
    check_bit_exact(y.cpu().numpy(), ref, "replayed GEMV")
    check_bit_exact(C2.cpu().numpy(), ref2, "replayed GEMM")
    step.free()
