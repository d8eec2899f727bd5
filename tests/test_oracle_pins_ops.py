"""Pins for the oracle functions behind the SURVEY.md section 8(f) rows: the element-wise add of
Listing 1, the binary16 codec and the f16-input GEMM (the paper's own
precision).  Same rule as test_oracle_pins.py: each pin fixes the oracle against
something other than itself -- the paper's printed example, IEEE-754 cases, closed forms,
numpy's own float32 add / float16 casts (library routines), a separately written loop.
All CPU; no CUDA code is touched.
"""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def golden_rows(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def f32(hexstr):
    return np.float32(float.fromhex(hexstr)) if hexstr not in ("inf", "-inf") else np.float32(hexstr)


# ---------------------------------------------------------------- element-wise add (Listing 1)
def test_add_paper_example_ones_plus_ones():
    (n, tile, x, y, z), = golden_rows("listing1_add.txt")
    n = int(n)
    out = oracle.add_f32(np.full(n, float(x), np.float32), np.full(n, float(y), np.float32))
    assert out.dtype == np.float32 and out.shape == (n,)
    assert np.all(out == np.float32(float(z)))


def test_add_ieee_rounding_cases():
    for xs, ys, zs in golden_rows("f32_add_rne.txt"):
        x, y, z = f32(xs), f32(ys), f32(zs)
        got = oracle.add_f32(np.array([x]), np.array([y]))[0]
        assert got.view(np.uint32) == z.view(np.uint32), (xs, ys, zs, float(got).hex())
        got = oracle.add_f32(np.array([y]), np.array([x]))[0]          # commutative
        assert got.view(np.uint32) == z.view(np.uint32)


def test_add_identities():
    rng = np.random.default_rng(5)
    x = (rng.standard_normal(4097) * np.exp(rng.uniform(-40, 40, 4097))).astype(np.float32)
    zero = np.zeros_like(x)
    assert np.array_equal(oracle.add_f32(x, zero).view(np.uint32), x.view(np.uint32))      # x + 0 = x
    assert np.all(oracle.add_f32(x, -x).view(np.uint32) == 0)                               # x + (-x) = +0
    assert np.array_equal(oracle.add_f32(x, x), np.float32(2) * x)                          # doubling is exact
    ints = rng.integers(-2 ** 22, 2 ** 22, size=(2, 5000))
    out = oracle.add_f32(ints[0].astype(np.float32), ints[1].astype(np.float32))
    assert np.array_equal(out.astype(np.int64), ints[0] + ints[1])                          # |sum| < 2^24: exact


def test_add_against_numpy_float32_add():
    rng = np.random.default_rng(6)
    n = 1_000_000
    x = (rng.standard_normal(n) * np.exp(rng.uniform(-30, 30, n))).astype(np.float32)
    y = (rng.standard_normal(n) * np.exp(rng.uniform(-30, 30, n))).astype(np.float32)
    # nearby magnitudes too, where the rounding actually bites
    y[::2] = (x[::2] * rng.uniform(-2, 2, (n + 1) // 2)).astype(np.float32)
    ours = oracle.add_f32(x, y)
    assert np.array_equal(ours.view(np.uint32), (x + y).view(np.uint32))


def test_add_against_a_separately_written_loop():
    rng = np.random.default_rng(7)
    x = rng.standard_normal(300).astype(np.float32)
    y = rng.standard_normal(300).astype(np.float32)
    ours = oracle.add_f32(x, y)
    for i in range(300):   # Python floats are binary64: exact sum, then one rounding
        assert ours[i] == np.float32(float(x[i]) + float(y[i]))


def test_add_empty():
    assert oracle.add_f32(np.zeros(0, np.float32), np.zeros(0, np.float32)).shape == (0,)


# ---------------------------------------------------------------- binary16 codec
def test_f16_decode_all_patterns_against_numpy():
    allbits = np.arange(65536, dtype=np.uint16)
    ours = oracle.f16_decode(allbits)
    ref = allbits.view(np.float16).astype(np.float64)
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(ours), nan)
    assert np.array_equal(ours[~nan], ref[~nan])
    assert np.array_equal(np.signbit(ours[~nan]), np.signbit(ref[~nan]))


def test_f16_decode_closed_forms():
    d = oracle.f16_decode(np.array([0x3C00, 0xC000, 0x0001, 0x0400, 0x7BFF, 0x3555], np.uint16))
    assert list(d[:5]) == [1.0, -2.0, 2.0 ** -24, 2.0 ** -14, 65504.0]
    assert d[5] == (1 + 0x155 / 1024) * 2.0 ** -2


def test_f16_encode_ieee_cases():
    for xs, hs in golden_rows("f16_rne.txt"):
        got = int(oracle.f16_encode(np.array([f32(xs)]))[0])
        assert got == int(hs, 16), (xs, hs, hex(got))


def test_f16_encode_round_trip_and_against_numpy():
    allbits = np.arange(65536, dtype=np.uint16)
    vals = allbits.view(np.float16)
    ok = ~np.isnan(vals)
    assert np.array_equal(oracle.f16_encode(vals.astype(np.float32))[ok], allbits[ok])
    rng = np.random.default_rng(8)
    x = (rng.standard_normal(1_000_000) * np.exp(rng.uniform(-20, 13, 1_000_000))).astype(np.float32)
    with np.errstate(over="ignore"):
        ref = x.astype(np.float16).view(np.uint16)
    assert np.array_equal(oracle.f16_encode(x), ref)
    # every midpoint between adjacent positive binary16 values (exact in binary32) and its neighbours
    lo = np.arange(0, 0x7BFF, dtype=np.uint16)
    a = lo.view(np.float16).astype(np.float64)
    b = (lo + 1).astype(np.uint16).view(np.float16).astype(np.float64)
    mid = ((a + b) / 2).astype(np.float32)
    assert np.array_equal(mid.astype(np.float64), (a + b) / 2)
    expect = np.where(lo & 1, lo + 1, lo).astype(np.uint16)
    assert np.array_equal(oracle.f16_encode(mid), expect)
    assert np.array_equal(oracle.f16_encode(np.nextafter(mid, np.float32(np.inf))), (lo + 1).astype(np.uint16))
    assert np.array_equal(oracle.f16_encode(np.nextafter(mid, np.float32(0))), lo)


# ---------------------------------------------------------------- GEMM with f16 inputs
def h(x):
    """values exactly representable in binary16 -> bit patterns (numpy's cast, not the oracle's)."""
    x = np.asarray(x, dtype=np.float32)
    b = x.astype(np.float16)
    assert np.array_equal(b.astype(np.float32), x), "test input not f16-exact"
    return b.view(np.uint16)


def test_f16_gemm_brute_force_8x8x8():
    rng = np.random.default_rng(9)
    a = rng.integers(-4, 5, (8, 8)).astype(np.float32)
    b = rng.integers(-4, 5, (8, 8)).astype(np.float32)
    C, S = oracle.gemm(h(a), h(b), in_dtype=oracle.IN_F16)
    for i in range(8):
        for j in range(8):
            acc, sacc = 0.0, 0.0
            for k in range(8):
                acc += float(a[i, k]) * float(b[k, j])
                sacc += abs(float(a[i, k])) * abs(float(b[k, j]))
            assert C[i, j] == acc and S[i, j] == sacc


def test_f16_gemm_identity_allones_onehot():
    rng = np.random.default_rng(10)
    bvals = rng.standard_normal((33, 47)).astype(np.float16)
    bb = bvals.view(np.uint16)
    C, S = oracle.gemm(h(np.eye(33)), bb, in_dtype=oracle.IN_F16)
    assert np.array_equal(C, bvals.astype(np.float64)) and np.array_equal(S, np.abs(bvals.astype(np.float64)))
    K = 769
    C, _ = oracle.gemm(h(np.ones((5, K))), h(np.ones((K, 7))), in_dtype=oracle.IN_F16)
    assert np.all(C == K)
    perm = rng.permutation(33)
    onehot = np.zeros((33, 33), np.float32)
    onehot[np.arange(33), perm] = 1
    C, _ = oracle.gemm(h(onehot), bb, in_dtype=oracle.IN_F16)
    assert np.array_equal(C, bvals.astype(np.float64)[perm])


def test_f16_gemm_against_numpy_fp64_and_sampled():
    rng = np.random.default_rng(11)
    a = rng.standard_normal((70, 300)).astype(np.float16)
    b = (rng.standard_normal((300, 90)) * 0.05).astype(np.float16)
    b[::7] = np.float16(2.0 ** -20)                      # subnormal binary16 inputs
    C, S = oracle.gemm(a.view(np.uint16), b.view(np.uint16), in_dtype=oracle.IN_F16)
    ref = a.astype(np.float64) @ b.astype(np.float64)
    sref = np.abs(a.astype(np.float64)) @ np.abs(b.astype(np.float64))
    assert np.all(np.abs(C - ref) <= 1e-12 * sref) and np.all(np.abs(S - sref) <= 1e-12 * sref)
    rows = rng.integers(0, 70, 50)
    cols = rng.integers(0, 90, 50)
    c, s = oracle.gemm_sampled(a.view(np.uint16), b.view(np.uint16), rows, cols, in_dtype=oracle.IN_F16)
    assert np.array_equal(c, C[rows, cols]) and np.array_equal(s, S[rows, cols])


def test_same_bits_mean_different_values_per_dtype():
    # 0x3C00 is 1.0 in binary16 and 0.0078125 in bf16: a swapped decode cannot pass both
    one = np.full((2, 2), 0x3C00, np.uint16)
    Ch, _ = oracle.gemm(one, one, in_dtype=oracle.IN_F16)
    Cb, _ = oracle.gemm(one, one, in_dtype=oracle.IN_BF16)
    assert np.all(Ch == 2.0) and np.all(Cb == 2 * 0.0078125 ** 2)


# ---------------------------------------------------------------- SwiGLU epilogue
def test_silu_closed_forms_and_identities():
    import math
    assert oracle.silu(0.0) == 0.0
    assert oracle.silu(1.0) == 1.0 / (1.0 + math.exp(-1.0))
    assert abs(oracle.silu(math.log(3.0)) - math.log(3.0) * 0.75) < 1e-15        # sigmoid(ln 3) = 3/4
    x = np.linspace(-30, 30, 2001)
    assert np.allclose(oracle.silu(x) - oracle.silu(-x), x, rtol=0, atol=1e-13)  # x*s(x) + x*s(-x) = x
    assert np.all(np.abs(oracle.silu(np.array([50.0, 700.0, 1e4])) - [50.0, 700.0, 1e4]) < 1e-12)
    assert np.all(np.abs(oracle.silu(np.array([-50.0, -700.0, -1e4]))) < 1e-19)  # no overflow to NaN on the left tail
    xm = -1.2784645427610738                                                    # argmin of silu: 1 + e^x (1 + x) = 0
    assert abs(oracle.silu(xm) - (-0.2784645427610738)) < 1e-12
    assert np.all(oracle.silu(x) >= -0.2784645427610739)


def test_silu_against_torch_float64():
    import torch
    rng = np.random.default_rng(12)
    x = rng.standard_normal(100_000) * 6
    ref = torch.nn.functional.silu(torch.from_numpy(x)).numpy()
    assert np.allclose(oracle.silu(x), ref, rtol=1e-14, atol=1e-300)


def test_swiglu_gemm_special_cases():
    from paper_2606_15991_b200 import workloads as wl
    rng = np.random.default_rng(13)
    M, K, inter = 9, 40, 24
    x = wl.f32_to_bf16_bits(rng.integers(-3, 4, (M, K)).astype(np.float32))
    wg = rng.integers(-2, 3, (K, inter)).astype(np.float32)
    wu = rng.integers(-2, 3, (K, inter)).astype(np.float32)
    W = wl.f32_to_bf16_bits(np.concatenate([wg, wu], axis=1))
    H, G, U, Sg, Su = oracle.swiglu_gemm(x, W)
    xd = oracle.bf16_decode(x)
    assert np.array_equal(G, xd @ wg) and np.array_equal(U, xd @ wu)              # the halves are [gate | up], in this order
    expect = np.where(G == 0, 0.0, G / (1 + np.exp(-G))) * U
    assert np.allclose(H, expect, rtol=1e-15, atol=0)
    # gate weights zero -> H = 0 exactly; up weights zero -> H = 0 exactly
    W0 = wl.f32_to_bf16_bits(np.concatenate([np.zeros_like(wg), wu], axis=1))
    assert np.all(oracle.swiglu_gemm(x, W0)[0] == 0)
    W1 = wl.f32_to_bf16_bits(np.concatenate([wg, np.zeros_like(wu)], axis=1))
    assert np.all(oracle.swiglu_gemm(x, W1)[0] == 0)
    # swapping the halves swaps the roles: silu(U) * G
    Ws = wl.f32_to_bf16_bits(np.concatenate([wu, wg], axis=1))
    assert np.allclose(oracle.swiglu_gemm(x, Ws)[0], oracle.silu(U) * G, rtol=1e-15, atol=0)
    # a large positive gate passes the up projection through: K ones times 64 = gate 2560 -> silu = identity to 1e-300
    xo = wl.f32_to_bf16_bits(np.ones((2, K), np.float32))
    Wb = wl.f32_to_bf16_bits(np.concatenate([np.full((K, 4), 64.0, np.float32), wu[:, :4]], axis=1))
    Hb, Gb, Ub, _, _ = oracle.swiglu_gemm(xo, Wb)
    assert np.array_equal(Hb, Gb * Ub)


def test_word_sum_against_python_integers():
    rng = np.random.default_rng(14)
    w = rng.integers(0, 2 ** 32, 5000, dtype=np.uint64).astype(np.uint32)
    assert oracle.word_sum_u32(w) == sum(int(v) for v in w) % 2 ** 64
    assert oracle.word_sum_u32(np.full(3, 0xFFFFFFFF, np.uint32)) == 3 * 0xFFFFFFFF
    assert oracle.word_sum_u32(np.zeros(0, np.uint32)) == 0
