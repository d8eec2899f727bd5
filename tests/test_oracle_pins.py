"""Pins for the fp64 CPU oracle (north_star names
identity, all-ones C_ij = K, 8x8x8 brute force and exact small-integer results).

Each pin fixes the oracle against something other than itself: closed forms,
special cases, a separately written brute-force loop, numpy's float64 matmul,
algebraic invariants, torch / ml_dtypes bf16 casts.  A dropped term, wrong
sign, wrong index or transposed operand fails at least one of them.
All CPU; no CUDA code is touched.
"""
import os

import ml_dtypes
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def bits(x):
    """float array whose values are exactly representable in bf16 -> bit patterns
    (through torch's cast, not the oracle's)."""
    b = wl.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))
    back = wl.bits_to_torch(b).to(torch.float32).numpy()
    assert np.array_equal(back, np.asarray(x, dtype=np.float32)), "test input not bf16-exact"
    return b


def ints(rng, shape, lo=-4, hi=4):
    return rng.integers(lo, hi + 1, size=shape).astype(np.float32)


# ---------------------------------------------------------------- bf16 codec
def test_bf16_decode_all_patterns_against_torch():
    allbits = np.arange(65536, dtype=np.uint16)
    ours = oracle.bf16_decode(allbits)
    ref = wl.bits_to_torch(allbits).to(torch.float64).numpy()
    both_nan = np.isnan(ours) & np.isnan(ref)
    assert np.array_equal(ours[~both_nan], ref[~both_nan])
    assert np.array_equal(np.isnan(ours), np.isnan(ref))
    # and against ml_dtypes, a second independent library
    ref2 = allbits.view(ml_dtypes.bfloat16).astype(np.float64)
    assert np.array_equal(ours[~both_nan], ref2[~both_nan])


def test_bf16_encode_roundtrip_all_patterns():
    allbits = np.arange(65536, dtype=np.uint16)
    vals = oracle.bf16_decode(allbits).astype(np.float32)
    nan = np.isnan(vals)
    enc = oracle.bf16_encode(vals)
    assert np.array_equal(enc[~nan], allbits[~nan])
    assert np.all((enc[nan] & 0x7FC0) == 0x7FC0)


def test_bf16_encode_ties_golden():
    # tests/golden/bf16_rne.txt: IEEE-754 round-to-nearest-even facts, hex in/out.
    rows = [l.split() for l in open(os.path.join(GOLDEN, "bf16_rne.txt")) if l.strip() and l[0] != "#"]
    f32 = np.array([int(r[0], 16) for r in rows], dtype=np.uint32).view(np.float32)
    want = np.array([int(r[1], 16) for r in rows], dtype=np.uint16)
    assert np.array_equal(oracle.bf16_encode(f32), want)


def test_bf16_encode_random_against_torch_and_ml_dtypes():
    rng = np.random.default_rng(11)
    x = np.concatenate([
        rng.standard_normal(600_000).astype(np.float32),
        (rng.standard_normal(200_000) * 1e-30).astype(np.float32),
        (rng.standard_normal(200_000) * 1e30).astype(np.float32),
        rng.integers(0, 2 ** 32, size=100_000, dtype=np.uint64).astype(np.uint32).view(np.float32),
    ])
    x = x[~np.isnan(x)]
    ours = oracle.bf16_encode(x)
    assert np.array_equal(ours, wl.f32_to_bf16_bits(x))
    assert np.array_equal(ours, x.astype(ml_dtypes.bfloat16).view(np.uint16))


# ---------------------------------------------------------------- special cases
def test_identity_left_and_right():
    rng = np.random.default_rng(1)
    n = 96
    eye = bits(np.eye(n))
    Bm = wl.f32_to_bf16_bits(rng.standard_normal((n, 130)).astype(np.float32))
    C, S = oracle.gemm(eye, Bm)
    assert np.array_equal(C, oracle.bf16_decode(Bm))        # I @ B == B exactly
    assert np.array_equal(S, np.abs(oracle.bf16_decode(Bm)))
    Am = wl.f32_to_bf16_bits(rng.standard_normal((70, n)).astype(np.float32))
    C, S = oracle.gemm(Am, eye)
    assert np.array_equal(C, oracle.bf16_decode(Am))        # A @ I == A exactly


@pytest.mark.parametrize("M,N,K", [(5, 7, 1), (33, 17, 257), (64, 64, 769), (3, 300, 4096)])
def test_all_ones_gives_K(M, N, K):
    C, S = oracle.gemm(bits(np.ones((M, K))), bits(np.ones((K, N))))
    assert np.all(C == K) and np.all(S == K)


def test_all_ones_bf16_output_rounding_golden():
    # RNE_bf16(K) for the all-ones product (SURVEY.md 8(c) pin table): 257 -> 256, 769 -> 768.
    rows = [l.split() for l in open(os.path.join(GOLDEN, "allones_bf16_out.txt")) if l.strip() and l[0] != "#"]
    for k, want in rows:
        K = int(k)
        C, _ = oracle.gemm(bits(np.ones((2, K))), bits(np.ones((K, 3))))
        got = oracle.bf16_decode(oracle.bf16_encode(C.astype(np.float32)))
        assert np.all(got == float(want)), (K, want)


def test_rank_one_closed_form():
    rng = np.random.default_rng(2)
    M, N, K = 41, 53, 37
    alpha = ints(rng, (M, 1))
    beta = ints(rng, (1, N))
    C, S = oracle.gemm(bits(np.repeat(alpha, K, axis=1)), bits(np.repeat(beta, K, axis=0)))
    assert np.array_equal(C, K * alpha.astype(np.float64) * beta.astype(np.float64))
    assert np.array_equal(S, K * np.abs(alpha).astype(np.float64) * np.abs(beta))


def test_k_mod_8_closed_form():
    M, N, K = 9, 11, 1003
    A = np.tile((np.arange(K) % 8).astype(np.float32), (M, 1))
    C, _ = oracle.gemm(bits(A), bits(np.ones((K, N))))
    full, rem = divmod(K, 8)
    assert np.all(C == full * 28 + sum(range(rem)))


def test_one_hot_rows_select_rows_of_B():
    # a_{i,pi(i)} = 1: C_i. = B_{pi(i)}. exactly; catches any k pairing / transposition error.
    rng = np.random.default_rng(3)
    M, N, K = 50, 67, 129
    pi = rng.integers(0, K, size=M)
    A = np.zeros((M, K), dtype=np.float32)
    A[np.arange(M), pi] = 1.0
    Bm = wl.f32_to_bf16_bits(rng.standard_normal((K, N)).astype(np.float32))
    C, _ = oracle.gemm(bits(A), Bm)
    assert np.array_equal(C, oracle.bf16_decode(Bm)[pi])


def test_one_hot_columns_select_columns_of_A():
    rng = np.random.default_rng(4)
    M, N, K = 31, 40, 77
    pj = rng.integers(0, K, size=N)
    Bm = np.zeros((K, N), dtype=np.float32)
    Bm[pj, np.arange(N)] = -2.0
    Am = wl.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    C, S = oracle.gemm(Am, bits(Bm))
    assert np.array_equal(C, -2.0 * oracle.bf16_decode(Am)[:, pj])
    assert np.array_equal(S, 2.0 * np.abs(oracle.bf16_decode(Am)[:, pj]))


# ---------------------------------------------------------------- brute force
def brute_force(a, b):
    """Separately written triple loop over Python floats (fp64)."""
    M, K = a.shape
    N = b.shape[1]
    c = [[0.0] * N for _ in range(M)]
    s = [[0.0] * N for _ in range(M)]
    for i in range(M):
        for j in range(N):
            acc = 0.0
            sacc = 0.0
            for k in range(K):
                acc += float(a[i, k]) * float(b[k, j])
                sacc += abs(float(a[i, k])) * abs(float(b[k, j]))
            c[i][j] = acc
            s[i][j] = sacc
    return np.array(c), np.array(s)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_8x8x8_ints(seed):
    rng = np.random.default_rng(seed)
    a, b = ints(rng, (8, 8)), ints(rng, (8, 8))
    C, S = oracle.gemm(bits(a), bits(b))
    cb, sb = brute_force(a, b)
    assert np.array_equal(C, cb) and np.array_equal(S, sb)


def test_brute_force_ragged_normals():
    rng = np.random.default_rng(5)
    ab = wl.f32_to_bf16_bits(rng.standard_normal((7, 13)).astype(np.float32))
    bb = wl.f32_to_bf16_bits(rng.standard_normal((13, 5)).astype(np.float32))
    a = wl.bits_to_torch(ab).to(torch.float64).numpy()
    b = wl.bits_to_torch(bb).to(torch.float64).numpy()
    C, S = oracle.gemm(ab, bb)
    cb, sb = brute_force(a, b)
    assert np.array_equal(C, cb) and np.array_equal(S, sb)   # same k order => same bits


# ---------------------------------------------------------------- library routine
@pytest.mark.parametrize("M,N,K", [(256, 256, 256), (129, 517, 1000), (1, 900, 1024), (1023, 64, 769)])
def test_against_numpy_float64_matmul(M, N, K):
    ab, bb = wl.make_inputs_custom(M, N, K, "normal", seed=M + N + K)
    a = wl.bits_to_torch(ab).to(torch.float64).numpy()
    b = wl.bits_to_torch(bb).to(torch.float64).numpy()
    C, S = oracle.gemm(ab, bb)
    assert np.all(np.abs(C - a @ b) <= 1e-12 * S + 1e-300)
    assert np.all(np.abs(S - np.abs(a) @ np.abs(b)) <= 1e-12 * S)


def test_integer_inputs_exact_vs_numpy_int64():
    rng = np.random.default_rng(6)
    M, N, K = 100, 90, 3000
    a, b = ints(rng, (M, K)), ints(rng, (K, N))
    C, S = oracle.gemm(bits(a), bits(b))
    assert np.array_equal(C, (a.astype(np.int64) @ b.astype(np.int64)).astype(np.float64))
    assert np.array_equal(S, (np.abs(a).astype(np.int64) @ np.abs(b).astype(np.int64)).astype(np.float64))


# ---------------------------------------------------------------- invariants
def test_blocks_and_threads_do_not_change_bits():
    ab, bb = wl.make_inputs_custom(150, 140, 333, "normal", seed=8)
    ref = oracle.gemm(ab, bb, threads=1, blocks=(1, 1, 1))
    for threads in (1, 3, 8):
        for blocks in ((7, 7, 7), (64, 256, 512), (1000, 1000, 1000)):
            C, S = oracle.gemm(ab, bb, threads=threads, blocks=blocks)
            assert np.array_equal(C, ref[0]) and np.array_equal(S, ref[1])


def test_gemv_column_partition_matches_row_partition():
    # M=1 takes the column-range thread partition; M=8 rows of the same x take the row one.
    ab, bb = wl.make_inputs_custom(1, 2000, 700, "normal", seed=9)
    C1, S1 = oracle.gemm(ab, bb, threads=8)
    C8, S8 = oracle.gemm(np.repeat(ab, 8, axis=0), bb, threads=8)
    assert all(np.array_equal(C8[r], C1[0]) for r in range(8))
    assert all(np.array_equal(S8[r], S1[0]) for r in range(8))


def test_transpose_identity_ints():
    rng = np.random.default_rng(10)
    a, b = ints(rng, (37, 91)), ints(rng, (91, 23))
    C, _ = oracle.gemm(bits(a), bits(b))
    Ct, _ = oracle.gemm(bits(b.T.copy()), bits(a.T.copy()))
    assert np.array_equal(C.T, Ct)


def test_k_permutation_invariance_ints():
    rng = np.random.default_rng(12)
    a, b = ints(rng, (20, 300)), ints(rng, (300, 30))
    p = rng.permutation(300)
    C, S = oracle.gemm(bits(a), bits(b))
    Cp, Sp = oracle.gemm(bits(a[:, p].copy()), bits(b[p].copy()))
    assert np.array_equal(C, Cp) and np.array_equal(S, Sp)


def test_padded_leading_dimensions_are_honoured():
    rng = np.random.default_rng(13)
    M, N, K = 19, 21, 45
    a, b = ints(rng, (M, K)), ints(rng, (K, N))
    apad = np.full((M, K + 11), 0x7FC0, dtype=np.uint16)   # NaN padding must never be read
    bpad = np.full((K, N + 5), 0x7FC0, dtype=np.uint16)
    apad[:, :K] = bits(a)
    bpad[:, :N] = bits(b)
    C, _ = oracle.gemm(apad[:, :K], bpad[:, :N])
    assert np.array_equal(C, (a.astype(np.int64) @ b.astype(np.int64)).astype(np.float64))


def test_sampled_matches_full():
    ab, bb = wl.make_inputs_custom(200, 300, 257, "normal", seed=14)
    C, S = oracle.gemm(ab, bb)
    r, c = wl.uniform_samples(200, 300, 500, seed=1)
    cs, ss = oracle.gemm_sampled(ab, bb, r, c)
    assert np.array_equal(cs, C[r, c]) and np.array_equal(ss, S[r, c])


def test_freivalds_identity_on_oracle_output():
    ab, bb = wl.make_inputs_custom(300, 280, 500, "normal", seed=15)
    a = oracle.bf16_decode(ab)
    b = oracle.bf16_decode(bb)
    C, S = oracle.gemm(ab, bb)
    r = np.random.default_rng(16).choice([-1.0, 1.0], size=280)
    assert np.all(np.abs(C @ r - a @ (b @ r)) <= 1e-10 * (S @ np.ones(280)))


# ---------------------------------------------------------------- degenerate
def test_degenerate_extents():
    z = np.zeros((0, 5), dtype=np.uint16)
    C, S = oracle.gemm(z, np.zeros((5, 4), dtype=np.uint16))
    assert C.shape == (0, 4)
    C, S = oracle.gemm(np.zeros((3, 0), dtype=np.uint16), np.zeros((0, 4), dtype=np.uint16))
    assert C.shape == (3, 4) and np.all(C == 0) and np.all(S == 0)   # K == 0 -> zeros (reading c8)


def test_cfg1_is_exact_and_bounded():
    ab, bb = wl.make_inputs(wl.CFG1)
    a = oracle.bf16_decode(ab)
    assert np.all(a == np.round(a)) and np.abs(a).max() <= 4
    C, S = oracle.gemm(ab, bb)
    assert np.all(C == np.round(C)) and np.abs(C).max() <= 16 * 256
    assert np.array_equal(C.astype(np.float32).astype(np.float64), C)  # exact in fp32 too
