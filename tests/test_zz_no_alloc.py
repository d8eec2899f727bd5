"""tile_gemv_no_alloc: the M = 1 product for callers that cannot allocate device memory.

Who that is: a serving process whose own pool took all of HBM at start-up (a cudaMalloc made by a
library would find nothing left), a plug-in whose host forbids allocations once it is initialised, a
decode loop that cannot take cudaMalloc's device-wide synchronisation in the middle of a token.  For
them the library has ONE entry whose split-K scratch (fp32 partial sums + arrival tickets) is a fixed
1 MiB + 4 KiB array inside the library image, shared by every call on a GPU and never cleared between
calls by anyone but the entry itself.

What is checked here, against the ordinary path (tile_gemm at M = 1, which takes its workspace from
cudaMalloc) and against the fp64 oracle, always on TWO calls in a row, because the second call is the
one that meets the first call's leftovers in the shared array:
  * normal inputs: both paths inside the suite's gates (tests/parity.py) of the oracle, and within the
    fp32 summation-order term 2K * 2^-24 * S of each other;
  * integer-valued inputs: all three bit-identical;
  * a second call that is narrower, shallower and sliced differently than the first (stale partial
    sums and stale ticket slots around it), and a second call of the same shape queued without any
    synchronisation in between;
  * requests beyond the fixed scratch fail with E_LIMIT, launch nothing and leave y alone.
The file is named test_zz_* so that pytest collects it last: `pytest -x` then never hides another
test behind a failure here.  It runs alone in a fresh process as well as after the rest of the suite
(the entry reads no tuning key; the ordinary path is used with its automatic plan).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl
from parity import check_bit_exact, check_close

X0, B0, Y0 = 0x10000, 0x7000_0000_0000, 0x7100_0000_0000   # fake, well separated, 16-byte aligned


# ------------------------------------------------------------------ host logic (no GPU needed)
def test_no_alloc_limits_are_checked_before_anything_is_queued():
    raw = tg.tile_gemv_no_alloc_raw
    assert tg.NO_ALLOC_SCRATCH_BYTES == tg.NO_ALLOC_MAX_TILES * (256 * 4 + 4)
    # wider than the scratch has tickets for
    st = raw(X0, B0, Y0, tg.NO_ALLOC_MAX_N + 1, 64, tg.NO_ALLOC_MAX_N + 8, tg.IN_BF16, tg.OUT_F32)
    assert st == tg.E_LIMIT and "TILE_GEMV_NO_ALLOC_MAX_N" in tg.tile_gemm_last_error()
    assert tg.tile_gemm_status_string(tg.E_LIMIT).startswith("request exceeds the fixed scratch")
    # 32 column blocks x 64 slices = 2048 partial-sum tiles > 1024
    st = raw(X0, B0, Y0, 8192, 4096, 8192, tg.IN_BF16, tg.OUT_F32, split=64)
    assert st == tg.E_LIMIT and "2048 partial-sum tiles" in tg.tile_gemm_last_error()
    # ... but a slice count above ceil(K / 64) means ceil(K / 64): 32 x 2 tiles fit
    if not torch.cuda.is_available():
        assert raw(X0, B0, Y0, 8192, 128, 8192, tg.IN_BF16, tg.OUT_F32, split=64) == tg.E_DEVICE
    # the remaining preconditions
    assert raw(X0, B0, Y0, 512, 512, 512, tg.IN_BF16, tg.OUT_F32, split=-1) == tg.E_EXTENT
    assert raw(X0, B0 + 2, Y0, 512, 512, 512, tg.IN_BF16, tg.OUT_F32) == tg.E_PATH      # B not 16-byte aligned
    assert raw(X0, B0, Y0, 512, 512, 516, tg.IN_BF16, tg.OUT_F32) == tg.E_PATH          # ldb not a multiple of 8
    assert "allocated copy" in tg.tile_gemm_last_error()
    assert raw(X0, B0, Y0, 512, 512, 504, tg.IN_BF16, tg.OUT_F32) == tg.E_LDB
    assert raw(X0, B0, Y0, 512, 512, 512, 7, tg.OUT_F32) == tg.E_IN_DTYPE
    assert raw(X0, B0, Y0, 512, 512, 512, tg.IN_BF16, 9) == tg.E_DTYPE
    assert raw(0, B0, Y0, 512, 512, 512, tg.IN_BF16, tg.OUT_F32) == tg.E_NULL
    assert raw(X0, B0, B0 + 64, 512, 512, 512, tg.IN_BF16, tg.OUT_F32) == tg.E_ALIAS     # y inside B
    assert raw(X0, B0, Y0, 0, 512, 512, tg.IN_BF16, tg.OUT_F32) == tg.E_OK               # N == 0: no-op
    if not torch.cuda.is_available():   # no CPU fallback: a valid request needs the device
        assert raw(X0, B0, Y0, 512, 512, 512, tg.IN_BF16, tg.OUT_F32) == tg.E_DEVICE


# ------------------------------------------------------------------ GPU: two calls in a row
def _padded_weights(b_bits, ldb, dtype):
    """(K, N) bit patterns as a row-major device tensor with row stride ldb >= N (padding = NaN patterns)."""
    K, N = b_bits.shape
    full = np.full((K, ldb), 0x7FC0 if dtype == torch.bfloat16 else 0x7E00, dtype=np.uint16)
    full[:, :N] = b_bits
    return wl.bits_to_torch(full, "cuda", dtype)[:, :N]


def _inputs(N, K, dist, seed, dtype=torch.bfloat16, sigma_b=1.0):
    if dtype == torch.bfloat16:
        x_bits, b_bits = wl.make_inputs_custom(1, N, K, dist=dist, sigma_b=sigma_b, seed=seed)
    else:
        x_bits, b_bits = wl.make_inputs_f16(1, N, K, dist=dist, sigma_b=sigma_b, seed=seed)
    return x_bits, b_bits


def _both_paths(x_bits, b_bits, ldb, out_dtype, split, dtype=torch.bfloat16):
    """Runs the no-alloc entry and the ordinary path on the same device tensors; nothing is synchronised here."""
    K, N = b_bits.shape
    x = wl.bits_to_torch(x_bits, "cuda", dtype)
    B = _padded_weights(b_bits, ldb, dtype)
    y_new = torch.full((N + 16,), float("nan"), dtype=out_dtype, device="cuda")   # 16 guard elements behind y
    before = tg.tile_gemm_launch_count()
    tg.tile_gemv_no_alloc(x, B, y_new[:N], split=split)
    assert tg.tile_gemm_launch_count() == before + 1
    y_old = tg.tile_gemm(x, B, out_dtype=out_dtype)
    return y_new, y_old


def _check_pair(y_new, y_old, x_bits, b_bits, out_name, exact, what, dtype=torch.bfloat16):
    K, N = b_bits.shape
    assert torch.isnan(y_new[N:].float()).all(), f"{what}: wrote past y[N)"
    new = y_new[:N].float().cpu().numpy().astype(np.float64)[None, :]
    old = y_old.float().cpu().numpy().astype(np.float64)
    ref, S = oracle.gemm(x_bits, b_bits, in_dtype=oracle.IN_BF16 if dtype == torch.bfloat16 else oracle.IN_F16)
    if exact:
        check_bit_exact(new, ref, what + " (no-alloc vs oracle)")
        assert np.array_equal(new, old), f"{what}: no-alloc and ordinary path differ on integer inputs"
        return
    check_close(new, ref, S, K, out_name, what + " (no-alloc vs oracle)")
    check_close(old, ref, S, K, out_name, what + " (ordinary path vs oracle)")
    # the two CUDA paths against each other: fp32 summation order (the `acc` term of parity.check_close),
    # plus one rounding step of the 16-bit output types
    acc = 2.0 * K * 2.0 ** -24 * S
    step = {"f32": 0.0, "bf16": 2.0 ** -7, "f16": 2.0 ** -10}[out_name] * np.abs(ref)
    bad = np.abs(new - old) > acc + step + 1e-300
    assert not bad.any(), f"{what}: paths differ beyond the suite's tolerance at {np.argwhere(bad)[:5].tolist()}"


@pytest.mark.gpu
def test_no_alloc_matches_the_ordinary_path_on_two_calls_in_a_row():
    # call 1: a decode-sized shape, automatic slices (the scratch fills with 32 x S tiles of partial sums)
    x1, b1 = _inputs(8192, 5120, "normal", seed=11, sigma_b=0.02)
    n1, o1 = _both_paths(x1, b1, 8192, torch.float32, split=0)
    # call 2, queued right behind it: narrower, shallower, ragged in N and K, padded rows, forced to 7 slices --
    # it lands in the middle of call 1's leftovers and must not see them
    x2, b2 = _inputs(1001, 1000, "int4", seed=12)
    n2, o2 = _both_paths(x2, b2, 1008, torch.float32, split=7)
    torch.cuda.synchronize()
    _check_pair(n1, o1, x1, b1, "f32", False, "call 1 (8192 x 5120, normal)")
    _check_pair(n2, o2, x2, b2, "f32", True, "call 2 (1001 x 1000, int4, 7 slices)")


@pytest.mark.gpu
@pytest.mark.parametrize("out_dtype,out_name", [(torch.float32, "f32"), (torch.bfloat16, "bf16")])
def test_no_alloc_same_shape_twice_without_synchronising(out_dtype, out_name):
    # the same (B, N, K) twice, different activations, no host synchronisation in between: the second launch
    # re-uses every ticket and every partial-sum slot of the first
    x1, b = _inputs(5120, 3136, "normal", seed=21, sigma_b=0.05)
    x2, _ = _inputs(5120, 3136, "normal", seed=22, sigma_b=0.05)
    n1, o1 = _both_paths(x1, b, 5120, out_dtype, split=0)
    n2, o2 = _both_paths(x2, b, 5120, out_dtype, split=0)
    torch.cuda.synchronize()
    _check_pair(n1, o1, x1, b, out_name, False, f"first call ({out_name})")
    _check_pair(n2, o2, x2, b, out_name, False, f"second call ({out_name})")
    # reproducible: the same call a third time gives the second call's bits
    n3, _ = _both_paths(x2, b, 5120, out_dtype, split=0)
    torch.cuda.synchronize()
    assert torch.equal(n3[:5120], n2[:5120])


@pytest.mark.gpu
def test_no_alloc_f16_inputs_and_output():
    x1, b1 = _inputs(4104, 2048, "normal", seed=41, dtype=torch.float16, sigma_b=0.05)
    n1, o1 = _both_paths(x1, b1, 4104, torch.float16, split=0, dtype=torch.float16)
    x2, b2 = _inputs(520, 777, "int4", seed=42, dtype=torch.float16)
    n2, o2 = _both_paths(x2, b2, 520, torch.float32, split=5, dtype=torch.float16)
    torch.cuda.synchronize()
    _check_pair(n1, o1, x1, b1, "f16", False, "f16 in, f16 out", dtype=torch.float16)
    _check_pair(n2, o2, x2, b2, "f32", True, "f16 in, fp32 out, int4", dtype=torch.float16)


@pytest.mark.gpu
@pytest.mark.parametrize("split", [1, 2, 3, 16, 40])
def test_no_alloc_integer_inputs_bit_exact_over_slice_counts(split):
    # S = 1 uses no scratch at all; S = 40 > 8 is beyond what a thread-block cluster could carry
    x1, b1 = _inputs(2600, 2500, "int4", seed=30 + split)
    n1, o1 = _both_paths(x1, b1, 2608, torch.float32, split=split)
    x2, b2 = _inputs(300, 4100, "int4", seed=60 + split)
    n2, o2 = _both_paths(x2, b2, 304, torch.float32, split=split)
    torch.cuda.synchronize()
    _check_pair(n1, o1, x1, b1, "f32", True, f"split {split}, first")
    _check_pair(n2, o2, x2, b2, "f32", True, f"split {split}, second")


@pytest.mark.gpu
def test_no_alloc_rejects_what_the_fixed_scratch_cannot_hold():
    K = 4096
    x = torch.ones((K,), dtype=torch.bfloat16, device="cuda")
    B = torch.ones((K, 8192), dtype=torch.bfloat16, device="cuda")
    y = torch.full((8192,), -7.0, dtype=torch.float32, device="cuda")
    before = tg.tile_gemm_launch_count()
    with pytest.raises(tg.TileGemmError) as e:
        tg.tile_gemv_no_alloc(x, B, y, split=64)          # 32 column blocks x 64 slices > 1024 tiles
    assert e.value.status == tg.E_LIMIT and "TILE_GEMV_NO_ALLOC_MAX_TILES" in e.value.message
    wide = tg.NO_ALLOC_MAX_N + 256
    Bw = torch.ones((64, wide), dtype=torch.bfloat16, device="cuda")
    yw = torch.full((wide,), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(tg.TileGemmError) as e:
        tg.tile_gemv_no_alloc(x[:64], Bw, yw)
    assert e.value.status == tg.E_LIMIT and "TILE_GEMV_NO_ALLOC_MAX_N" in e.value.message
    torch.cuda.synchronize()
    assert tg.tile_gemm_launch_count() == before
    assert (y == -7.0).all() and (yw == -7.0).all()
    # the widest legal output and the fullest legal slicing still run, and right after the failures
    tg.tile_gemv_no_alloc(x[:64], Bw[:, :tg.NO_ALLOC_MAX_N], yw[:tg.NO_ALLOC_MAX_N])
    tg.tile_gemv_no_alloc(x, B, y, split=32)              # 32 x 32 = 1024 tiles: exactly the scratch
    torch.cuda.synchronize()
    assert (yw[:tg.NO_ALLOC_MAX_N] == 64.0).all() and (yw[tg.NO_ALLOC_MAX_N:] == -7.0).all()
    assert (y == float(K)).all()
