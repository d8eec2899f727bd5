"""Parity on the configurations bench.py reports that the earlier files do not reach (round 3):

  * the large points of the paper's square sweep -- 16384^3 in bf16 and f16, 32768^3 in
    bf16: the lockstep producers cover 27 and 110 whole rounds there (tile_gemm_query_plan), a path the other
    tests reach only at K = 16384 on 4096 rows;
  * the weight-streaming tensor-core kernel (2 <= M <= 64) in its AUTOMATIC plan, weights declared immutable
    as bench.py's skinny_m leg does, on the four Qwen3-32B decode shapes -- including the
    K-slice counts 4 and 6 that plan picks there and the 400-block unsliced launch of N = 51200;
  * the tiled kernel on 2 <= M <= 64 (its short A box and its split-K of a launch below one wave), which the
    selector only reaches for 49..64 rows on sliced weights unless tuning key 11 says "never skinny".

Inputs are generated on the device by the seeded generators of workloads.py and read back for the oracle.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl
from parity import check_bit_exact, check_close
from test_gpu_parity import SKINNY_SHAPES, rne_bf16, run_case

pytestmark = pytest.mark.gpu
DEV = "cuda"


@pytest.fixture(autouse=True)
def _reset_tuning():
    yield
    for key in range(tg.NUM_TUNE_KEYS):
        tg.tile_gemm_set_tuning(key, 0)
    torch.cuda.synchronize()


# ------------------------------------------------------------------ the sweep's large sizes
@pytest.mark.parametrize("n,dtype", [(16384, torch.bfloat16), (16384, torch.float16), (32768, torch.bfloat16)])
def test_sweep_large_sizes_sampled(n, dtype):
    """One sample in every 256 x 512 output tile (4096 samples at 16384^2, 8192 at 32768^2) against
    oracle.gemm_sampled, on normal inputs (tolerance gates) and on integer inputs (bit-exact: sums stay below
    2^24); the 16-bit result is RNE of the fp32 result bit for bit on the whole matrix; run-to-run bits equal."""
    name = "bf16" if dtype == torch.bfloat16 else "f16"
    in_dtype = oracle.IN_BF16 if dtype == torch.bfloat16 else oracle.IN_F16
    plan = tg.tile_gemm_query_plan(n, n, n)
    assert plan["config"] == 4 and plan["lockstep_rounds"] >= (100 if n == 32768 else 20)
    rows, cols = wl.stratified_samples(n, n, (256, 512), seed=n)
    assert rows.size == (n // 256) * (n // 512)
    ri, ci = torch.from_numpy(rows).to(DEV), torch.from_numpy(cols).to(DEV)
    C32 = torch.empty((n, n), dtype=torch.float32, device=DEV)
    C16 = torch.empty((n, n), dtype=dtype, device=DEV)
    C16b = torch.empty((n, n), dtype=dtype, device=DEV)

    # normal inputs, the distribution bench.py's sweep draws (A ~ N(0, 1), B ~ N(0, 1/n))
    g = torch.Generator(device=DEV)
    g.manual_seed(1000 + n)
    A = torch.empty((n, n), dtype=dtype, device=DEV).normal_(0, 1, generator=g)
    B = torch.empty((n, n), dtype=dtype, device=DEV).normal_(0, n ** -0.5, generator=g)
    tg.tile_gemm(A, B, C32)
    tg.tile_gemm(A, B, C16)
    tg.tile_gemm(A, B, C16b)
    torch.cuda.synchronize()
    assert torch.equal(C16.view(torch.int16), C16b.view(torch.int16)), "run-to-run bits differ"
    assert torch.equal(C32.to(dtype).view(torch.int16), C16.view(torch.int16)), f"{name} output is not RNE(fp32 output)"
    a, b = wl.torch_to_bits(A), wl.torch_to_bits(B)
    c_ref, s_ref = oracle.gemm_sampled(a, b, rows, cols, in_dtype=in_dtype)
    check_close(C32[ri, ci].cpu().numpy(), c_ref, s_ref, n, "f32", f"{n}^3 {name} in, fp32 samples")
    check_close(C16[ri, ci].float().cpu().numpy(), c_ref, s_ref, n, name, f"{n}^3 {name} samples")
    del a, b, C16, C16b

    # integer inputs: |sum| <= 16 n < 2^24, every partial sum exact -> the fp32 result is the exact result
    Ai, Bi = wl.make_int_inputs_device(n, n, n, seed=n, device=DEV, dtype=dtype)
    A.copy_(Ai)
    B.copy_(Bi)
    del Ai, Bi
    tg.tile_gemm(A, B, C32)
    torch.cuda.synchronize()
    a, b = wl.torch_to_bits(A), wl.torch_to_bits(B)
    c_ref, _ = oracle.gemm_sampled(a, b, rows, cols, in_dtype=in_dtype)
    check_bit_exact(C32[ri, ci].cpu().numpy(), c_ref, f"{n}^3 {name} integer samples")
    # every row sum of C against A (B 1): exact in int64, covers every output tile row of the whole matrix
    ones = B.double().sum(dim=1)                                   # (K,) exact: |.| <= 4 n
    want = (A.double() @ ones)                                     # exact: integers below 2^53
    got = C32.double().sum(dim=1)
    assert torch.equal(got, want), "row sums of the integer result differ from A (B 1)"


# ------------------------------------------------------------------ skinny M on the decode shapes, automatic plan
def _decode_weights(K, N, seed, integer):
    if integer:
        _, W = wl.make_int_inputs_device(1, N, K, seed=seed, device=DEV)
        return W
    g = torch.Generator(device=DEV)
    g.manual_seed(seed)
    return torch.empty((K, N), dtype=torch.bfloat16, device=DEV).normal_(0, 0.02, generator=g)


@pytest.mark.parametrize("proj", [0, 1, 2, 3])
def test_skinny_decode_shapes_automatic_plan(proj):
    """M in {8, 32, 48, 64} on one decode shape with the plan bench.py times (automatic, static_b): integer
    inputs bit-exact on the full output, normal inputs inside the gates, bf16 output = RNE(fp32 output),
    nothing written past row M - 1 or column N - 1."""
    K, N = wl.QWEN3_32B[proj]
    Wi = _decode_weights(K, N, 500 + proj, True)
    Wn = _decode_weights(K, N, 600 + proj, False)
    wi_bits, wn_bits = wl.torch_to_bits(Wi), wl.torch_to_bits(Wn)
    Xi, _ = wl.make_int_inputs_device(64, 1, K, seed=700 + proj, device=DEV)
    g = torch.Generator(device=DEV)
    g.manual_seed(800 + proj)
    Xn = torch.empty((64, K), dtype=torch.bfloat16, device=DEV).normal_(0, 1, generator=g)
    seen = set()
    for M in (8, 32, 48, 64):
        p = tg.tile_gemm_query_plan(M, N, K)
        seen.add((p["config"], p["split"]))
        for X, W, w_bits, integer in ((Xi, Wi, wi_bits, True), (Xn, Wn, wn_bits, False)):
            if not integer and M not in (32, 64):
                continue
            C32 = torch.full((M + 1, N + 8), float("nan"), dtype=torch.float32, device=DEV)
            Cb = torch.full((M + 1, N + 8), float("nan"), dtype=torch.bfloat16, device=DEV)
            tg.tile_gemm(X[:M], W, C32[:M, :N], static_b=True)
            tg.tile_gemm(X[:M], W, Cb[:M, :N], static_b=True)
            torch.cuda.synchronize()
            for C in (C32, Cb):
                assert torch.isnan(C[M]).all() and torch.isnan(C[:, N:]).all(), f"M={M}: wrote outside C"
                assert not torch.isnan(C[:M, :N]).any(), f"M={M}: elements of C left unwritten"
            ref, S = oracle.gemm(wl.torch_to_bits(X[:M]), w_bits)
            got32 = C32[:M, :N].cpu().numpy()
            gotb = Cb[:M, :N].float().cpu().numpy().astype(np.float64)
            what = f"{wl.QWEN3_32B_NAMES[proj]} M={M} plan={p['config']}/{p['split']}"
            if integer:
                check_bit_exact(got32, ref, what)
                assert np.array_equal(gotb, rne_bf16(ref)), what + ": bf16 output"
            else:
                check_close(got32, ref, S, K, "f32", what)
                check_close(gotb, ref, S, K, "bf16", what + " bf16")
                assert np.array_equal(gotb, rne_bf16(got32)), what + ": bf16 output is not RNE(fp32 output)"
    assert any(c == 5 for c, _ in seen), "the weight-streaming kernel was never selected"


# ------------------------------------------------------------------ the tiled kernel on 2 <= M <= 64
@pytest.mark.parametrize("M", [2, 5, 16, 33, 64])
@pytest.mark.parametrize("split", [0, 3])
def test_tiled_kernel_on_few_rows_integer_bit_exact_and_canary(M, split):
    """Tuning key 11 = 1 ("never the weight-streaming kernel"): the tiled kernel takes M <= 64 with its short A
    box, and below one wave cuts K -- automatically or into the forced number of slices -- on ragged N and K
    and padded strides.  Integer inputs are exact whatever the slicing; the canary sees every element
    written and nothing outside."""
    tg.tile_gemm_set_tuning(tg.TUNE_SKINNY, 1)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, split)
    for (K, N), pads in SKINNY_SHAPES:
        a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=91 + M)
        ref, _ = oracle.gemm(a, b)
        pads_ok = (pads[0] + (-(K + pads[0])) % 8, pads[1] + (-(N + pads[1])) % 8, pads[2])   # A and B stay TMA-addressable
        p = tg.tile_gemm_query_plan(M, N, K)
        assert p["config"] in (1, 2, 3, 4) and p["a_box_rows"] <= 64
        got = run_case(a, b, "f32", pads=pads_ok, force=tg.PATH_GEMM_TMA, what=f"tiled M={M}")
        check_bit_exact(got.astype(np.float32), ref, f"tiled M={M} K={K} N={N} split={split} plan={p}")
        gotb = run_case(a, b, "bf16", pads=pads_ok, what=f"tiled M={M} bf16")
        assert np.array_equal(gotb, rne_bf16(ref))
