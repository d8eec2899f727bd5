"""CPU tests of the boundary: the C-ABI library loads and exports every symbol the header
declares, launch preconditions and the selector behave as include/tile_gemm.h states (pure
host, fake pointers, nothing dereferenced), the schedule function covers C exactly once, and
the N>1 helpers work over gloo with world_size 2.  No compute call is made (no GPU here)."""
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest
import torch

import parity
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
A0, B0, C0 = 0x10000, 0x7000_0000_0000, 0x7100_0000_0000   # fake, well separated, 16-byte aligned


def test_library_exports_every_declared_symbol():
    header = "".join(open(os.path.join(ROOT, "include", h)).read() for h in ("tile_gemm.h", "tile_gemm_debug.h"))
    declared = set(re.findall(r"\b(tile_(?:gemm|gemv|add|read)\w*)\s*\(", header))
    assert declared == set(tg.EXPORTS), declared ^ set(tg.EXPORTS)
    lib = tg.load_library()
    for name in declared:
        assert hasattr(lib, name), name


def test_status_strings_are_distinct():
    names = [tg.tile_gemm_status_string(i) for i in range(16)]
    assert len(set(names)) == 16 and names[0] == "ok"
    assert tg.tile_gemm_status_string(99) == "unknown status"


def sel(M, N, K, lda=None, ldb=None, ldc=None, A=A0, B=B0, C=C0, out=tg.OUT_F32):
    return tg.tile_gemm_select(M, N, K, K if lda is None else lda, N if ldb is None else ldb,
                               N if ldc is None else ldc, A, B, C, out)


def test_selector_paths_for_baseline_configs():
    assert sel(256, 256, 256) == tg.PATH_GEMM_TMA
    assert sel(1023, 1537, 769) == tg.PATH_GEMM_REPACK            # packed rows are not 16-byte multiples
    assert sel(1023, 1537, 769, 776, 1544, 1544) == tg.PATH_GEMM_TMA
    assert sel(8192, 8192, 8192, out=tg.OUT_BF16) == tg.PATH_GEMM_TMA
    for (K, N) in wl.QWEN3_32B:
        assert sel(4096, N, K, out=tg.OUT_BF16) == tg.PATH_GEMM_TMA
        assert sel(1, N, K, out=tg.OUT_BF16) == tg.PATH_GEMV
    assert sel(256, 256, 256, A=A0 + 2) == tg.PATH_GEMM_REPACK     # misaligned base
    assert sel(1, 1537, 769) == tg.PATH_GEMV                       # GEMV needs no alignment
    assert sel(5, 7, 0) == tg.PATH_ZERO
    assert sel(0, 7, 3) == tg.PATH_NOOP and sel(7, 0, 3) == tg.PATH_NOOP


@pytest.mark.parametrize("kwargs,code,fragment", [
    (dict(M=-1, N=4, K=4), tg.E_EXTENT, "negative extent"),
    (dict(M=4, N=4, K=4, lda=3), tg.E_LDA, "lda=3 < K=4"),
    (dict(M=4, N=4, K=4, ldb=3), tg.E_LDB, "ldb=3 < N=4"),
    (dict(M=4, N=4, K=4, ldc=3), tg.E_LDC, "ldc=3 < N=4"),
    (dict(M=4, N=4, K=4, out=7), tg.E_DTYPE, "out_dtype=7"),
    (dict(M=4, N=4, K=4, A=0), tg.E_NULL, "A is NULL"),
    (dict(M=4, N=4, K=4, B=0), tg.E_NULL, "B is NULL"),
    (dict(M=4, N=4, K=4, C=0), tg.E_NULL, "C is NULL"),
    (dict(M=4, N=4, K=4, A=A0 + 1), tg.E_ALIGN, "2-byte aligned"),
    (dict(M=4, N=4, K=4, C=C0 + 2), tg.E_ALIGN, "4-byte aligned"),
    (dict(M=4, N=4, K=4, C=A0 + 8), tg.E_ALIAS, "overlaps A"),
    (dict(M=4, N=4, K=4, C=B0), tg.E_ALIAS, "overlaps B"),
    (dict(M=2 ** 31, N=4, K=4), tg.E_OVERFLOW, "extent above"),
    (dict(M=2 ** 20, N=4, K=4, lda=2 ** 45), tg.E_OVERFLOW, "overflow"),
])
def test_each_precondition_has_its_own_error(kwargs, code, fragment):
    """'each rejected on the host with its own message'."""
    assert sel(**kwargs) == -code
    assert fragment in tg.tile_gemm_last_error()


def test_bf16_output_alignment_is_two_bytes():
    assert sel(4, 4, 4, C=C0 + 2, out=tg.OUT_BF16) > 0
    assert sel(4, 4, 4, C=C0 + 1, out=tg.OUT_BF16) == -tg.E_ALIGN


def test_strided_operands_that_only_touch_do_not_alias():
    a_bytes = (4 - 1) * 4 * 2 + 4 * 2
    assert sel(4, 4, 4, C=A0 + a_bytes + 2, out=tg.OUT_BF16) > 0      # directly after A's span
    assert sel(4, 4, 4, C=A0 + a_bytes - 2, out=tg.OUT_BF16) == -tg.E_ALIAS


def test_compute_entries_fail_loudly_without_a_gpu():
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    rc = tg.tile_gemm_raw(A0, B0, C0, 4, 4, 4, 4, 4, 4, 0)
    assert rc == tg.E_DEVICE
    assert "no CPU fallback" in tg.tile_gemm_last_error()
    rc = tg.tile_gemm_host_raw(A0, B0, C0, 4, 4, 4, 4, 4, 4, 0)
    assert rc == tg.E_DEVICE


def test_bad_force_path_and_tuning_key():
    assert tg.tile_gemm_raw(A0, B0, C0, 4, 4, 4, 4, 4, 4, 0, 0, 9) == tg.E_PATH
    with pytest.raises(tg.TileGemmError):
        tg.tile_gemm_set_tuning(99, 0)


@pytest.mark.parametrize("cfg", [
    dict(BM=128, BN=128, cta_group=1, ctas=148, group_m=16),
    dict(BM=128, BN=256, cta_group=1, ctas=56, group_m=16),
    dict(BM=128, BN=256, cta_group=2, ctas=148, group_m=8),
    dict(BM=128, BN=256, cta_group=2, ctas=8, group_m=3),
    dict(BM=128, BN=512, cta_group=2, ctas=132, group_m=8, config=6),    # two CTA pairs per cluster: a unit is two tile rows
    dict(BM=128, BN=512, cta_group=2, ctas=12, group_m=2, config=6),
])
@pytest.mark.parametrize("shape", [(1023, 1537), (8192, 8192), (130, 70), (4096, 5120)])
def test_schedule_function_covers_every_element_once(cfg, shape):
    """The tile -> owner map restated on the host is a function onto [0,M) x [0,N): every
    element has exactly one owning tile and CTA ids stay below the launched count."""
    M, N = shape
    own = parity.expected_owner_map(M, N, cfg)
    assert own.min() >= 0
    tile_m = cfg["BM"] * cfg["cta_group"] * (2 if cfg.get("config") == 6 else 1)      # rows of a work unit
    tiles = -(-M // tile_m) * -(-N // cfg["BN"])
    ids = np.unique(own >> 8)
    assert ids.size == tiles and ids.max() == tiles - 1
    assert (own & 0xFF).max() < cfg["ctas"]
    # each unit id occupies one rectangle of unit rows x BN, every CTA of its cluster a BM-row band of it
    t = int(ids[len(ids) // 2])
    rr, cc = np.where((own >> 8) == t)
    assert rr.max() - rr.min() < tile_m and cc.max() - cc.min() < cfg["BN"]
    for cta in np.unique(own[rr, cc] & 0xFF):
        r2 = rr[(own[rr, cc] & 0xFF) == cta]
        assert r2.max() - r2.min() < cfg["BM"]


def test_workload_shapes_match_baseline_json():
    assert (wl.CFG1.M, wl.CFG1.N, wl.CFG1.K) == (256, 256, 256)
    assert (wl.CFG2.M, wl.CFG2.N, wl.CFG2.K) == (1023, 1537, 769)
    assert (wl.CFG3.M, wl.CFG3.N, wl.CFG3.K) == (8192, 8192, 8192)
    assert [(c.K, c.N) for c in wl.CFG4] == [(5120, 10240), (5120, 8192), (5120, 51200), (25600, 5120)]
    assert all(c.M == 4096 for c in wl.CFG4)
    a, b = wl.make_inputs(wl.CFG1)
    a2, _ = wl.make_inputs(wl.CFG1)
    assert np.array_equal(a, a2)
    vals = wl.bits_to_torch(a).float().numpy()
    assert set(np.unique(vals)) <= set(range(-4, 5))
    r, c = wl.stratified_samples(8192, 8192, 128, seed=2)
    assert r.size == 4096 and len(set(zip((r // 128).tolist(), (c // 128).tolist()))) == 4096


def test_gloo_world_size_two_bench_helpers():
    """bench.py's N>1 plumbing (unit sharding, max-over-ranks timing) over gloo on CPU."""
    script = os.path.join(ROOT, "tests", "gloo_worker.py")
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29541", PYTHONPATH=ROOT)
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29541", script],
                         env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    assert "GLOO_OK rank0" in res.stdout


# ------------------------------------------------------------------ SURVEY 8(f) entries: launch preconditions on the host
def test_add_preconditions_are_checked_before_any_device_call():
    X, Y, Z = 0x10000, 0x7000_0000_0000, 0x7100_0000_0000
    assert tg.tile_add_f32_raw(X, Y, Z, -1) == tg.E_EXTENT
    assert tg.tile_add_f32_raw(X, Y, Z, 0) == tg.E_OK                      # empty: success, nothing to do
    assert tg.tile_add_f32_raw(X, Y, Z, (1 << 40) + 1) == tg.E_OVERFLOW
    assert tg.tile_add_f32_raw(0, Y, Z, 8) == tg.E_NULL
    assert tg.tile_add_f32_raw(X, Y, 0, 8) == tg.E_NULL
    assert tg.tile_add_f32_raw(X + 2, Y, Z, 8) == tg.E_ALIGN
    assert tg.tile_add_f32_raw(X, Y, X + 16, 8) == tg.E_ALIAS             # z overlaps x: the output is exclusively owned
    assert tg.tile_add_f32_raw(X, Y, Y - 16, 8) == tg.E_ALIAS
    assert tg.tile_add_f32_raw(X, Y, Y + 32, 8) != tg.E_ALIAS             # adjacent, not overlapping
    assert "z" in tg.tile_gemm_last_error() or not torch.cuda.is_available()
    if not torch.cuda.is_available():                                        # no CPU fallback: the device check fails loudly
        assert tg.tile_add_f32_raw(X, X, Z, 8) == tg.E_DEVICE


def test_typed_entry_preconditions():
    args = (A0, B0, C0, 8, 8, 8, 8, 8, 8)
    assert tg.tile_gemm_typed_raw(*args, 2, tg.OUT_F32) == tg.E_IN_DTYPE
    assert tg.tile_gemm_typed_raw(*args, -1, tg.OUT_F32) == tg.E_IN_DTYPE
    assert tg.tile_gemm_typed_raw(*args, tg.IN_F16, 3) == tg.E_DTYPE
    assert tg.tile_gemm_typed_raw(A0, B0, C0, 8, 8, 8, 7, 8, 8, tg.IN_F16, tg.OUT_F16) == tg.E_LDA
    # a 16-bit C (bf16 or f16) must be 2-byte aligned, an fp32 C 4-byte aligned
    assert tg.tile_gemm_typed_raw(A0, B0, C0 + 2, 8, 8, 8, 8, 8, 8, tg.IN_F16, tg.OUT_F16) != tg.E_ALIGN
    assert tg.tile_gemm_typed_raw(A0, B0, C0 + 2, 8, 8, 8, 8, 8, 8, tg.IN_F16, tg.OUT_F32) == tg.E_ALIGN
    if not torch.cuda.is_available():
        assert tg.tile_gemm_typed_raw(*args, tg.IN_F16, tg.OUT_F16) == tg.E_DEVICE


def test_record_entries_reject_bad_handles_without_a_device():
    lib = tg.load_library()
    assert lib.tile_gemm_replay(None, None) == tg.E_NULL
    assert lib.tile_gemm_recorded_nodes(None) == -1
    assert lib.tile_gemm_record_free(None) == tg.E_OK
    import ctypes
    out = ctypes.c_void_p(1)
    assert lib.tile_gemm_record_end(ctypes.c_void_p(0x1000), ctypes.byref(out)) == tg.E_PATH   # that stream is not recording
    assert out.value is None and "not recording" in tg.tile_gemm_last_error()
    assert lib.tile_gemm_record_end(ctypes.c_void_p(0x1000), None) == tg.E_NULL
    if not torch.cuda.is_available():
        assert lib.tile_gemm_record_begin(None) == tg.E_DEVICE


def test_debug_entries_check_their_arguments_on_the_host():
    lib = tg.load_library()
    import ctypes
    assert lib.tile_gemm_debug_trace(ctypes.c_void_p(0x1004), 4) == tg.E_ALIGN
    assert lib.tile_gemm_debug_trace(ctypes.c_void_p(0x1000), -1) == tg.E_EXTENT
    assert lib.tile_gemm_debug_trace(None, 0) == tg.E_OK
    assert lib.tile_gemm_debug_occupy(-1, 10, None) == tg.E_EXTENT
    assert lib.tile_gemm_debug_occupy(1, 3_000_000_000, None) == tg.E_OVERFLOW
    for key in range(tg.NUM_TUNE_KEYS):
        tg.tile_gemm_set_tuning(key, 0)


def test_swiglu_preconditions_on_the_host():
    a = (A0, B0, C0)
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 31, 16, tg.OUT_F32) == tg.E_LDB          # ldw < 2I
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 63, 32, 16, tg.OUT_F32) == tg.E_LDA
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 32, 15, tg.OUT_F32) == tg.E_LDC
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 32, 16, 9) == tg.E_DTYPE
    assert tg.tile_gemm_swiglu_raw(*a, 8, 12, 64, 64, 32, 16, tg.OUT_F32) == tg.E_PATH         # I % 8 != 0
    assert tg.tile_gemm_swiglu_raw(A0 + 2, B0, C0, 8, 16, 64, 64, 32, 16, tg.OUT_F32) == tg.E_PATH   # X not TMA-addressable
    assert tg.tile_gemm_swiglu_raw(A0, B0, B0 + 64 * 2 * 16 + 32, 8, 16, 64, 64, 64, 16, tg.OUT_BF16) == tg.E_ALIAS  # H inside the up half
    assert tg.tile_gemm_swiglu_raw(*a, 0, 16, 64, 64, 32, 16, tg.OUT_F32) == tg.E_OK           # M == 0: no-op
    if not torch.cuda.is_available():
        assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 32, 16, tg.OUT_F32) == tg.E_DEVICE


def test_selector_routes_a_few_rows_to_the_tensor_cores():
    # only M = 1 is the CUDA-core GEMV; from M = 2 on the tensor-core path (in place through TMA where A and B
    # are 16-byte addressable -- the weight-streaming kernel up to M = 64 where its plan allows -- else after a repack)
    assert sel(1, 10240, 5120) == tg.PATH_GEMV
    for M in (2, 3, 4, 5, 32, 33):
        assert sel(M, 10240, 5120) == tg.PATH_GEMM_TMA
        assert sel(M, 10240, 5120, lda=5121) == tg.PATH_GEMM_REPACK
        assert sel(M, 10240, 5120, A=A0 + 2) == tg.PATH_GEMM_REPACK
    st = tg.tile_gemm_raw(A0, B0, C0, 2, 64, 64, 64, 64, 64, tg.OUT_F32, force_path=tg.PATH_GEMV)
    assert st == tg.E_PATH and "M == 1" in tg.tile_gemm_last_error()


@pytest.mark.parametrize("G", [2, 8])
def test_selector_on_column_shards(G):
    """column shard g of a row-major B (K x N) is the pointer B + g*N/G with ldb = N.
    For the Qwen3 shapes every shard stays TMA-addressable (16-byte aligned start, ldb % 8 == 0) and
    disjoint from the other shards' C columns, so the selector takes the same paths as unsharded."""
    for (K, N) in wl.QWEN3_32B:
        w = N // G
        for g in (0, G - 1):
            Bg, Cg = B0 + 2 * g * w, C0 + 2 * g * w
            assert tg.tile_gemm_select(4096, w, K, K, N, N, A0, Bg, Cg, tg.OUT_BF16) == tg.PATH_GEMM_TMA
            assert tg.tile_gemm_select(1, w, K, K, N, N, A0, Bg, Cg, tg.OUT_BF16) == tg.PATH_GEMV
    # a shard whose first column is not 16-byte aligned falls back to the repack path, still legal
    assert tg.tile_gemm_select(64, 100, 256, 256, 1004, 1004, A0, B0 + 2 * 100, C0 + 4 * 100, tg.OUT_F32) == tg.PATH_GEMM_REPACK


def test_truncation_model_on_the_hand_worked_cases():
    """parity.tcgen05_accumulate_model (the statement of how the tensor core sums) gives
    the hand-worked values of parity.TRUNCATION_CASES; the GPU test then holds the kernel to both."""
    for groups, exact, nearest, want in parity.TRUNCATION_CASES:
        v = []
        for g in groups:
            v += list(g) + [0.0] * (16 - len(g))
        a = np.array([v])
        assert a.sum() == exact
        assert np.float64(np.float32(exact)) == nearest or abs(exact) % 1 == 0.5   # RNE of the exact sum (ties listed by hand)
        got = parity.tcgen05_accumulate_model(a, np.ones((len(v), 1)))[0, 0]
        assert got == want



def test_bench_gpus_flag_starts_that_many_ranks():
    """`python bench.py --gpus 2` without a torchrun environment (the driver's plain form) must start two ranks
    itself: the self-spawn path re-launches the same command line under torch.distributed.run, the two ranks
    rendezvous (gloo here, NCCL on a GPU box) and rank 0 reports the world that met.  --rendezvous-only stops
    there, before any kernel, so this runs on the CPU box."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env["PYTHONPATH"] = ROOT
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rendezvous-only"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stdout + res.stderr
    lines = [json.loads(ln) for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout                      # rank 0 alone prints
    assert lines[0]["rendezvous"] == 2 and lines[0]["gpus_flag"] == 2
    assert lines[0]["max_rank"] == 1.0 and lines[0]["sum_rank_plus_1"] == 3.0
    # one rank: no spawn, no process group
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--rendezvous-only"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0 and json.loads(res.stdout.strip().splitlines()[-1])["rendezvous"] == 1
