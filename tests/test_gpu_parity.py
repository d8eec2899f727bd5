"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, on a B200.

Covers BASELINE.json's five configs at full size in the launch configuration bench.py times,
plus the extra cases SURVEY.md 8(c) asks for: one-hot inputs per tile configuration, integer
ragged / large-K shapes bit-exact, canary-filled C, owner map, force_path sweep, determinism,
degenerate extents and the host-buffer entry.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl
import parity
from parity import check_bit_exact, check_close, freivalds_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"
CANARY_F32 = 0x7FC0DEAD
CANARY_BF16 = 0x7FD5


@pytest.fixture(autouse=True)
def _reset_tuning():
    yield
    for key in range(tg.NUM_TUNE_KEYS):
        tg.tile_gemm_set_tuning(key, 0)
    torch.cuda.synchronize()


def device_operand(bits, pad_cols=0, misalign_elems=0):
    """bf16 operand on the device with `pad_cols` extra (NaN) columns per row and an optional
    element offset of the base pointer; returns a strided view."""
    r, c = bits.shape
    ld = c + pad_cols
    flat = torch.full((r * ld + misalign_elems + 8,), float("nan"), dtype=torch.bfloat16, device=DEV)
    view = flat[misalign_elems:misalign_elems + r * ld].view(r, ld)[:, :c]
    view.copy_(wl.bits_to_torch(bits, DEV))
    return view


class CanaryC:
    """C with guard rows above/below and padding columns, all canary filled."""

    def __init__(self, M, N, out, pad_cols=0, guard=8, misalign_elems=0):
        self.M, self.N, self.out, self.guard = M, N, out, guard
        self.ld = N + pad_cols
        rows = M + 2 * guard
        if out == "f32":
            self.raw = torch.full((rows * self.ld + misalign_elems + 4,), 0, dtype=torch.int32, device=DEV)
            self.raw.fill_(np.int32(CANARY_F32))
            self.dtype, self.canary = torch.float32, np.uint32(CANARY_F32)
        else:
            self.raw = torch.full((rows * self.ld + misalign_elems + 8,), 0, dtype=torch.int16, device=DEV)
            self.raw.fill_(np.int16(CANARY_BF16))
            self.dtype, self.canary = torch.bfloat16, np.uint16(CANARY_BF16)
        self.full = self.raw[misalign_elems:misalign_elems + rows * self.ld].view(rows, self.ld)
        self.C = self.full[guard:guard + M, :N].view(self.dtype)

    def check(self, what=""):
        """Guards untouched, every inside element overwritten.  Returns C as float64."""
        host = self.full.cpu().numpy()
        bits = host.view(np.uint32 if self.out == "f32" else np.uint16)
        g = self.guard
        outside = np.ones(bits.shape, dtype=bool)
        outside[g:g + self.M, :self.N] = False
        touched = outside & (bits != self.canary)
        assert not touched.any(), (f"{what}: {int(touched.sum())} elements written outside C[0:M,0:N], "
                                   f"first at (row-guard, col) {(np.argwhere(touched)[:5] - [g, 0]).tolist()}")
        inside = bits[g:g + self.M, :self.N]
        assert not (inside == self.canary).any(), f"{what}: some elements of C were never written"
        if self.out == "f32":
            return inside.view(np.float32).astype(np.float64)
        return oracle.bf16_decode(np.ascontiguousarray(inside))


def run_case(a_bits, b_bits, out="f32", pads=(0, 0, 0), force=tg.PATH_AUTO, misalign=(0, 0, 0), what="", static_b=False):
    M, K = a_bits.shape
    N = b_bits.shape[1]
    A = device_operand(a_bits, pads[0], misalign[0])
    B = device_operand(b_bits, pads[1], misalign[1])
    cc = CanaryC(M, N, out, pads[2], misalign_elems=misalign[2])
    tg.tile_gemm(A, B, cc.C, force_path=force, static_b=static_b)
    torch.cuda.synchronize()
    return cc.check(what)


def rne_bf16(x64):
    """Library RNE (torch) of fp32 values to bf16, back as float64."""
    t = torch.from_numpy(np.asarray(x64, dtype=np.float32)).to(torch.bfloat16)
    return t.to(torch.float64).numpy()


# ------------------------------------------------------------------ library actually loaded
def test_native_library_is_loaded_and_launches():
    tg.load_library()
    maps = open("/proc/self/maps").read()
    assert "libtilegemm.so" in maps
    before = tg.tile_gemm_launch_count()
    a, b = wl.make_inputs(wl.CFG1)
    run_case(a, b)
    assert tg.tile_gemm_launch_count() > before


# ------------------------------------------------------------------ config 1
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_cfg1_bit_exact(cfg):
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    a, b = wl.make_inputs(wl.CFG1)
    ref, _ = oracle.gemm(a, b)
    got = run_case(a, b, "f32", what=f"cfg1 config={cfg}")
    check_bit_exact(got, ref, f"cfg1 config={cfg}")
    got = run_case(a, b, "bf16", what=f"cfg1 bf16 config={cfg}")
    assert np.array_equal(got, rne_bf16(ref))


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_one_hot_rows_and_columns(cfg):
    """a_{i,pi(i)} = 1 gives C_i. = B_{pi(i)}. exactly: any k-pairing, transposition, swizzle or
    descriptor error in the tensor-core path shows up as a wrong row/column."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    rng = np.random.default_rng(cfg)
    M, N, K = 384, 640, 448
    pi = rng.integers(0, K, size=M)
    A = np.zeros((M, K), np.float32)
    A[np.arange(M), pi] = 1.0
    bb = wl.f32_to_bf16_bits(rng.standard_normal((K, N)).astype(np.float32))
    got = run_case(wl.f32_to_bf16_bits(A), bb, what="one-hot rows")
    assert np.array_equal(got, oracle.bf16_decode(bb)[pi])
    pj = rng.integers(0, K, size=N)
    Bm = np.zeros((K, N), np.float32)
    Bm[pj, np.arange(N)] = 1.0
    ab = wl.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    got = run_case(ab, wl.f32_to_bf16_bits(Bm), what="one-hot columns")
    assert np.array_equal(got, oracle.bf16_decode(ab)[:, pj])


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
@pytest.mark.parametrize("K", [1, 63, 64, 65, 257])
def test_all_ones_any_k(cfg, K):
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    M, N = 130, 264
    ones = lambda r, c: wl.f32_to_bf16_bits(np.ones((r, c), np.float32))
    got = run_case(ones(M, K), ones(K, N), "f32", what="all ones")
    assert np.all(got == K)
    got = run_case(ones(M, K), ones(K, N), "bf16", what="all ones bf16")
    assert np.all(got == rne_bf16(np.array([float(K)]))[0])


# ------------------------------------------------------------------ config 2 (ragged, canary)
LAYOUTS = {
    "packed": ((0, 0, 0), (0, 0, 0)),                       # lda=769, ldb=ldc=1537: repack + st.global
    "padded": ((776 - 769, 1544 - 1537, 1544 - 1537), (0, 0, 0)),   # TMA loads and TMA stores
    "offset": ((776 - 769, 1544 - 1537, 1544 - 1537), (1, 3, 1)),   # 16-byte multiples, odd bases
    "mixed": ((776 - 769, 0, 1544 - 1537), (0, 0, 0)),      # only B needs a repack
}


@pytest.mark.parametrize("layout", list(LAYOUTS))
@pytest.mark.parametrize("out", ["f32", "bf16"])
def test_cfg2_ragged_full_oracle_and_canary(layout, out):
    pads, mis = LAYOUTS[layout]
    a, b = wl.make_inputs(wl.CFG2)
    ref, S = oracle.gemm(a, b)
    got = run_case(a, b, out, pads=pads, misalign=mis, what=f"cfg2 {layout} {out}")
    check_close(got, ref, S, wl.CFG2.K, out, f"cfg2 {layout} {out}")


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
@pytest.mark.parametrize("layout", ["packed", "padded"])
def test_cfg2_shape_integer_inputs_bit_exact(cfg, layout):
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    pads, mis = LAYOUTS[layout]
    a, b = wl.make_inputs_custom(1023, 1537, 769, "int4", seed=21)
    ref, _ = oracle.gemm(a, b)
    got = run_case(a, b, "f32", pads=pads, misalign=mis, what=f"cfg2-int {layout} config={cfg}")
    check_bit_exact(got, ref, f"cfg2-int {layout} config={cfg}")


def test_force_path_sweep_agrees():
    a, b = wl.make_inputs_custom(300, 520, 200, "int4", seed=5)
    ref, _ = oracle.gemm(a, b)
    for force in (tg.PATH_GEMM_TMA, tg.PATH_GEMM_REPACK):
        got = run_case(a, b, "f32", force=force, what=f"force={force}")
        check_bit_exact(got, ref, f"force={force}")
    # M = 1 through the tensor-core path and through every GEMV variant
    a, b = wl.make_inputs_custom(1, 1032, 520, "int4", seed=6)
    ref, _ = oracle.gemm(a, b)
    for force in (tg.PATH_GEMM_TMA, tg.PATH_GEMM_REPACK, tg.PATH_GEMV):
        check_bit_exact(run_case(a, b, "f32", force=force), ref, f"M=1 force={force}")


def test_large_k_integer_bit_exact():
    a, b = wl.make_inputs_custom(512, 768, 8192, "int4", seed=8)
    ref, _ = oracle.gemm(a, b)
    check_bit_exact(run_case(a, b, "f32"), ref, "K=8192 ints")


# ------------------------------------------------------------------ GEMV variants
@pytest.mark.parametrize("variant", [2, 3, 4])
@pytest.mark.parametrize("split", [0, 1, 3, 8])
def test_gemv_variants_integer_bit_exact(variant, split):
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_VARIANT, variant)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, split)
    for (K, N, padb) in ((512, 1024, 0), (769, 1537, 7), (2000, 264, 0), (64, 8, 0), (1, 300, 4)):
        a, b = wl.make_inputs_custom(1, N, K, "int4", seed=K + N)
        ref, _ = oracle.gemm(a, b)
        got = run_case(a, b, "f32", pads=(0, padb, 0), what=f"gemv v{variant} s{split} K={K} N={N}")
        check_bit_exact(got, ref, f"gemv v{variant} s{split} K={K} N={N}")


@pytest.mark.parametrize("shape", [2, 4, 6])
@pytest.mark.parametrize("cap", [0, 1, 3, 7, 100])
@pytest.mark.parametrize("nopdl", [0, 1])
@pytest.mark.parametrize("fix", [0, 1])
def test_gemv_split_decompositions_integer_bit_exact(shape, cap, nopdl, fix):
    """The interleaved split-K kernel under every decomposition: one CTA looping over all column
    blocks (cap=1), fewer CTAs than column blocks (cap 3, 7), deep splits (cap 100 and the full
    budget); K and N tails; every ring shape; with and without programmatic dependent launch; with
    the automatic choice of fix-up protocol (cluster / tagged slots / tickets) and with tickets only."""
    occ = shape
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, fix)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_VARIANT, 4)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SHAPE, shape)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MAX_CTAS, cap)
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, nopdl)
    for (K, N, padb) in ((512, 1024, 0), (769, 1537, 7), (2000, 264, 0), (64, 8, 0), (1, 300, 4), (4100, 2056, 0)):
        a, b = wl.make_inputs_custom(1, N, K, "int4", seed=K + N)
        ref, _ = oracle.gemm(a, b)
        for rep in range(2):   # the second call finds the tickets re-armed by the first
            got = run_case(a, b, "f32", pads=(0, padb, 0), what=f"flat occ{occ} cap{cap} K={K} N={N}")
            check_bit_exact(got, ref, f"flat occ{occ} cap{cap} K={K} N={N} rep{rep}")


@pytest.mark.parametrize("split", [0, 2, 3, 5, 8, 11, 24])
@pytest.mark.parametrize("static_b", [False, True])
def test_gemv_fixup_protocols_give_the_same_bits(split, static_b):
    """The three split-K hand-over protocols of the M = 1 kernel (thread-block cluster + DSMEM, tagged
    slots with a designated combiner, tickets) add the S partial sums in the same slice order: on
    normal inputs they must agree bit for bit, call after call (slots and tickets re-armed), and each
    matches the oracle."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, split)
    for (K, N) in ((5120, 2048), (2560, 8200), (1999, 1000)):
        a, b = wl.make_inputs_custom(1, N, K, sigma_b=K ** -0.5, seed=K + N + split)
        ref, S = oracle.gemm(a, b)
        x, W = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
        outs = {}
        for fix in (1, 2, 3, 0):
            tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, fix)
            for rep in range(3):
                y = torch.full((1, N), float("nan"), dtype=torch.float32, device=DEV)
                tg.tile_gemm(x, W, y, static_b=static_b)
                torch.cuda.synchronize()
                outs[(fix, rep)] = y.cpu().numpy()
            check_close(outs[(fix, 0)].astype(np.float64), ref, S, K, "f32", f"fix-up {fix} K={K} N={N} S={split}")
        # with the automatic slice count the cluster protocol may pick another S (a cluster size that fits the
        # device), so only protocols that ran the same decomposition are comparable bit for bit
        same_cut = (1, 2) if split == 0 else (1, 2, 3, 0)
        first = outs[(1, 0)].view(np.uint32)
        for (fix, rep), v in outs.items():
            want = first if fix in same_cut else outs[(fix, 0)].view(np.uint32)
            assert np.array_equal(v.view(np.uint32), want), f"fix-up {fix} rep {rep}: bits differ (K={K} N={N} S={split})"


def test_gemv_completes_next_to_a_kernel_that_holds_sms():
    """Tagged slots and clusters assume the launch fits the device; with 100 SMs held by another kernel
    the CTAs arrive in waves instead.  The designated combiner is the LAST slice of its column block,
    so everything it waits for was dispatched before it: the launch still completes, with the same bits."""
    K, N = 5120, 8192
    a, b = wl.make_inputs_custom(1, N, K, "int4", seed=77)
    ref, _ = oracle.gemm(a, b)
    x, W = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    blocker, worker = torch.cuda.Stream(), torch.cuda.Stream()
    for fix in (0, 2, 3):
        tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, fix)
        y = torch.full((1, N), float("nan"), dtype=torch.float32, device=DEV)
        torch.cuda.synchronize()
        tg.tile_gemm_debug_occupy(100, 20_000_000, stream=blocker)
        for _ in range(3):
            tg.tile_gemm(x, W, y, stream=worker, static_b=True)
        worker.synchronize()
        blocker.synchronize()
        check_bit_exact(y.cpu().numpy(), ref, f"GEMV next to a blocker, fix-up {fix}")


@pytest.mark.parametrize("fix", [0, 1, 2])
@pytest.mark.parametrize("static_b", [False, True])
def test_gemv_chain_is_stream_ordered_under_pdl(static_b, fix):
    """y of one GEMV is x of the next, launched back to back with programmatic dependent launch:
    the bits must equal those of the same chain run with a synchronise after every launch, and every
    link must match the oracle on the bits it was given."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_FIXUP, fix)
    K = N = 2048
    depth = 6
    rng = np.random.default_rng(31)
    Ws = [wl.bits_to_torch(wl.f32_to_bf16_bits((rng.standard_normal((K, N)) * K ** -0.5).astype(np.float32)), DEV)
          for _ in range(depth)]
    x0 = wl.bits_to_torch(wl.f32_to_bf16_bits(rng.standard_normal((1, K)).astype(np.float32)), DEV)

    def chain(sync):
        xs = [x0] + [torch.empty((1, N), dtype=torch.bfloat16, device=DEV) for _ in range(depth)]
        for i in range(depth):
            tg.tile_gemm(xs[i], Ws[i], xs[i + 1], static_b=static_b)
            if sync:
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        return xs

    want = chain(True)
    for i in range(depth):
        ref, S = oracle.gemm(wl.torch_to_bits(want[i]), wl.torch_to_bits(Ws[i]))
        check_close(want[i + 1].float().cpu().numpy(), ref, S, K, "bf16", f"chain link {i}")
    for rep in range(10):
        got = chain(False)
        for i in range(depth + 1):
            assert torch.equal(got[i].view(torch.int16), want[i].view(torch.int16)), f"rep {rep} link {i}"


def test_gemv_unaligned_weights_take_scalar_path():
    a, b = wl.make_inputs_custom(1, 1537, 769, "normal", seed=3)
    ref, S = oracle.gemm(a, b)
    for out in ("f32", "bf16"):
        got = run_case(a, b, out, misalign=(1, 1, 1), what="gemv odd")
        check_close(got, ref, S, 769, out, "gemv odd ldb / odd base")


# ------------------------------------------------------------------ config 3 (headline)
def test_cfg3_8192_sampled_freivalds_and_rounding_chain():
    case = wl.CFG3
    a, b = wl.make_inputs(case)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    C32 = torch.empty((case.M, case.N), dtype=torch.float32, device=DEV)
    Cb = torch.empty((case.M, case.N), dtype=torch.bfloat16, device=DEV)
    Cb2 = torch.empty_like(Cb)
    tg.tile_gemm(A, B, C32)
    tg.tile_gemm(A, B, Cb)
    tg.tile_gemm(A, B, Cb2)
    torch.cuda.synchronize()
    assert torch.equal(Cb.view(torch.int16), Cb2.view(torch.int16)), "run-to-run bits differ"
    # (ii) the bf16 result is RNE of the fp32 result bit for bit (same main loop)
    assert torch.equal(C32.to(torch.bfloat16).view(torch.int16), Cb.view(torch.int16))
    rows, cols = wl.stratified_samples(case.M, case.N, 128, seed=2)
    assert rows.size == 4096
    c_ref, s_ref = oracle.gemm_sampled(a, b, rows, cols)
    got32 = C32[torch.from_numpy(rows).to(DEV), torch.from_numpy(cols).to(DEV)].cpu().numpy()
    gotb = Cb[torch.from_numpy(rows).to(DEV), torch.from_numpy(cols).to(DEV)].float().cpu().numpy()
    check_close(got32, c_ref, s_ref, case.K, "f32", "cfg3 fp32 samples")
    check_close(gotb, c_ref, s_ref, case.K, "bf16", "cfg3 bf16 samples")
    # (i) Freivalds on the full fp32 matrix
    freivalds_rows(C32.cpu().numpy().astype(np.float64), oracle.bf16_decode(a), oracle.bf16_decode(b), seed=2)


# ------------------------------------------------------------------ config 4 (prefill projections)
@pytest.mark.parametrize("proj", [0, 1, 2, 3])
def test_cfg4_prefill_sampled(proj):
    case = wl.CFG4[proj]
    a, b = wl.make_inputs(case)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    Cb = torch.empty((case.M, case.N), dtype=torch.bfloat16, device=DEV)
    C32 = torch.empty((case.M, case.N), dtype=torch.float32, device=DEV)
    tg.tile_gemm(A, B, Cb)
    tg.tile_gemm(A, B, C32)
    torch.cuda.synchronize()
    assert torch.equal(C32.to(torch.bfloat16).view(torch.int16), Cb.view(torch.int16))
    rows, cols = wl.uniform_samples(case.M, case.N, 4096, seed=proj)
    c_ref, s_ref = oracle.gemm_sampled(a, b, rows, cols)
    ri, ci = torch.from_numpy(rows).to(DEV), torch.from_numpy(cols).to(DEV)
    check_close(Cb[ri, ci].float().cpu().numpy(), c_ref, s_ref, case.K, "bf16", case.name)
    check_close(C32[ri, ci].cpu().numpy(), c_ref, s_ref, case.K, "f32", case.name + " fp32")
    # Freivalds on the FULL fp32 matrix (reading c13), rows and columns, in 1024-row bands:
    # |C r - A (B r)| per row and |c C - (c A) B| per column with r, c in {+-1}.  Tolerance 2^-14 plus the
    # K-dependent term of parity.check_close's rel_rms gate (the tensor core adds each K = 16 step into the fp32
    # accumulator with truncation), times the row's / column's 2-norm.
    rng = np.random.default_rng(proj)
    r = rng.choice([-1.0, 1.0], size=case.N)
    c = rng.choice([-1.0, 1.0], size=case.M)
    rel = 2.0 ** -14 + (case.K / 16.0) * 2.0 ** -24
    br = np.zeros(case.K)
    for k0 in range(0, case.K, 1024):
        br[k0:k0 + 1024] = oracle.bf16_decode(b[k0:k0 + 1024]) @ r
    ca = np.zeros(case.K)          # c A
    cC = np.zeros(case.N)          # c C
    col_sq = np.zeros(case.N)      # squared column norms of C
    for r0 in range(0, case.M, 1024):
        band = slice(r0, min(r0 + 1024, case.M))
        a64 = oracle.bf16_decode(a[band])
        Cband = C32[band].cpu().numpy().astype(np.float64)
        tol = rel * np.linalg.norm(Cband, axis=1) + 1e-30
        bad = np.abs(Cband @ r - a64 @ br) > tol
        assert not bad.any(), f"{case.name}: Freivalds row test failed in rows {(r0 + np.where(bad)[0][:8]).tolist()}"
        ca += c[band] @ a64
        cC += c[band] @ Cband
        col_sq += (Cband * Cband).sum(axis=0)
    cab = np.zeros(case.N)         # (c A) B
    for k0 in range(0, case.K, 1024):
        cab += ca[k0:k0 + 1024] @ oracle.bf16_decode(b[k0:k0 + 1024])
    bad = np.abs(cC - cab) > rel * np.sqrt(col_sq) + 1e-30
    assert not bad.any(), f"{case.name}: Freivalds column test failed for columns {np.where(bad)[0][:8].tolist()}"


# ------------------------------------------------------------------ the accumulator's arithmetic
@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_tcgen05_accumulator_model_predicts_every_bit(cfg):
    """DESIGN.md 7 / tests/parity.py widen the fp32 gates by (K/16) * 2^-24 because "the tensor core
    adds each K = 16 step with truncation".  This pins that claim: parity.tcgen05_accumulate_model
    (align 16 products + accumulator to the largest exponent, truncate each toward zero with two guard
    bits, add exactly, truncate to fp32) predicts the kernel's fp32 output BIT FOR BIT -- on inputs
    constructed so that round-to-nearest and truncation differ, and on random normal inputs -- for the
    1-CTA and the 2-CTA tile configurations alike."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    M = N = 256
    for groups, exact, nearest, want in parity.TRUNCATION_CASES:
        v = []
        for g in groups:
            v += list(g) + [0.0] * (16 - len(g))
        K = max(64, len(v))
        a32 = np.zeros((M, K), dtype=np.float32)
        a32[:, :len(v)] = np.asarray(v, dtype=np.float32)
        a = wl.f32_to_bf16_bits(a32)
        a64 = oracle.bf16_decode(a)
        assert np.array_equal(a64, a32.astype(np.float64)), "the constructed values must be exact in bf16"
        b = wl.f32_to_bf16_bits(np.ones((K, N), dtype=np.float32))
        ref, S = oracle.gemm(a, b)
        assert ref[0, 0] == exact                                     # the oracle states the exact sum
        got = run_case(a, b, "f32", what=f"constructed {groups}")
        assert np.all(got == want), f"{groups}: kernel {got[0, 0]}, truncation model says {want}, round-to-nearest {nearest}"
        model = parity.tcgen05_accumulate_model(a64, oracle.bf16_decode(b))
        assert np.all(model == want), f"{groups}: the model itself gives {model[0, 0]}, expected {want}"
        assert np.all(np.abs(got - ref) <= 2.0 * K * 2.0 ** -24 * S)    # and all of it is inside the tight gate
    rng = np.random.default_rng([77, cfg])
    for K in (16, 80, 256, 1024):
        a = wl.f32_to_bf16_bits(rng.standard_normal((M, K), dtype=np.float32))
        b = wl.f32_to_bf16_bits(rng.standard_normal((K, N), dtype=np.float32) * np.float32(K ** -0.5))
        got = run_case(a, b, "f32", what=f"random K={K}")
        model = parity.tcgen05_accumulate_model(oracle.bf16_decode(a), oracle.bf16_decode(b))
        bad = got != model
        assert not bad.any(), f"K={K}: {int(bad.sum())} of {bad.size} elements differ from the truncation model"
        ref, S = oracle.gemm(a, b)
        signed = (got - ref) * np.sign(ref)
        assert signed.mean() < 0, "truncation toward zero must show as a bias toward zero against the exact sums"


# ------------------------------------------------------------------ config 5 (decode GEMV)
def _cfg5_layers():
    """All 64 layers by default (BASELINE.json config 5: "full oracle comparison");
    TILEGEMM_CFG5_LAYERS=n restricts a quick local run to layers {0, ..., n-2, 63}."""
    n = int(os.environ.get("TILEGEMM_CFG5_LAYERS", wl.DECODE_LAYERS))
    if n >= wl.DECODE_LAYERS:
        return list(range(wl.DECODE_LAYERS))
    return sorted(set(list(range(max(n - 1, 1))) + [wl.DECODE_LAYERS - 1]))


def test_cfg5_decode_full_oracle():
    """Every output of all 256 GEMVs of config 5 (64 layers x 4 projections, 62.4 GB of weights, each
    generated in its own buffer) against the oracle, in the auto launch configuration; odd layers go
    through tile_gemm_static_b (the entry bench.py times), even layers through tile_gemm.  The four
    oracle calls of a layer (M = 1: one thread each) run side by side on the host."""
    from concurrent.futures import ThreadPoolExecutor
    checked = 0
    with ThreadPoolExecutor(max_workers=4) as pool:
        for layer in _cfg5_layers():
            jobs = []
            for proj in range(4):
                case = wl.cfg5_case(layer, proj)
                x, W = wl.make_inputs_device(case, DEV)
                y = torch.empty((1, case.N), dtype=torch.bfloat16, device=DEV)
                assert tg.tile_gemm_select(1, case.N, case.K, case.K, case.N, case.N) == tg.PATH_GEMV
                tg.tile_gemm(x, W, y, static_b=(layer % 2 == 1))
                torch.cuda.synchronize()
                xb, Wb, got = wl.torch_to_bits(x), wl.torch_to_bits(W), y.float().cpu().numpy()
                del W
                jobs.append((case, got, pool.submit(oracle.gemm, xb, Wb)))
            for case, got, fut in jobs:
                ref, S = fut.result()
                check_close(got, ref, S, case.K, "bf16", case.name)
                checked += 1
    assert checked == 4 * len(_cfg5_layers())


# ------------------------------------------------------------------ column shards
@pytest.mark.parametrize("G", [2, 8])
def test_column_shards_equal_the_unsharded_result(G):
    """SURVEY 8(e) / DESIGN.md 9: a caller that shards N over G devices calls tile_gemm on
    B[:, n_g] (ldb = N) and C[:, n_g] (ldc = N).  Every output element is the same K-ordered sum
    whatever tile it falls in, so as long as neither launch cuts K the shards reproduce the
    unsharded bits exactly (normal inputs); M = 1 shards change the K slicing, so there the check is
    bit-exact on integer-valued inputs and within tolerance on normal ones."""
    M, N, K = 384, 4096, 768
    a, b = wl.make_inputs_custom(M, N, K, sigma_b=K ** -0.5, seed=90 + G)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    assert tg.tile_gemm_query_plan(M, N, K)["split"] == 0 and tg.tile_gemm_query_plan(M, N // G, K)["split"] == 0
    for out_dt in (torch.float32, torch.bfloat16):
        whole = torch.empty((M, N), dtype=out_dt, device=DEV)
        tg.tile_gemm(A, B, whole)
        shards = torch.full((M, N), float("nan"), dtype=out_dt, device=DEV)
        w = N // G
        for g in range(G):
            tg.tile_gemm(A, B[:, g * w:(g + 1) * w], shards[:, g * w:(g + 1) * w])
        torch.cuda.synchronize()
        assert torch.equal(whole, shards), f"G={G} {out_dt}: column shards differ from the unsharded result"
    ref, S = oracle.gemm(a, b)
    check_close(whole.float().cpu().numpy(), ref, S, K, "bf16", f"unsharded G={G}")
    # M = 1 (decode): integer-valued inputs, bit-exact against the oracle shard by shard
    N1, K1 = 8192, 2560
    x, Wt = wl.make_inputs_custom(1, N1, K1, "int4", seed=95 + G)
    ref1, _ = oracle.gemm(x, Wt)
    xd, Wd = wl.bits_to_torch(x, DEV), wl.bits_to_torch(Wt, DEV)
    y = torch.full((1, N1), float("nan"), dtype=torch.float32, device=DEV)
    w = N1 // G
    for g in range(G):
        tg.tile_gemm(xd, Wd[:, g * w:(g + 1) * w], y[:, g * w:(g + 1) * w], static_b=True)
    torch.cuda.synchronize()
    check_bit_exact(y.cpu().numpy(), ref1, f"M=1 column shards G={G}")


# ------------------------------------------------------------------ ownership
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 6])
@pytest.mark.parametrize("shape", [(1023, 1537), (256, 256), (4096, 5120), (130, 70), (1300, 520)])
def test_owner_map_is_the_documented_function(cfg, shape):
    """Each output element is written by exactly one CTA, the one tile_coords assigns
    (PAPER.md:163 'each sub-tensor has exactly one owner').  cfg 6 = config 4 with two CTA pairs per
    cluster (B multicast): a work unit is two tile rows, one per pair."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, min(cfg, 4))
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MULTICAST, 2 if cfg == 6 else 1)
    M, N = shape
    conf = tg.tile_gemm_query_config(M, N, 64)
    assert conf["config"] == (4 if cfg == 6 and M <= 256 else cfg)     # one tile row: nothing to pair up
    for ld in (N, N + 3):
        owner = tg.tile_gemm_debug_owner_map(M, N, 64, ld_owner=ld)
        torch.cuda.synchronize()
        host = owner.cpu().numpy()
        assert np.all(host[:, N:] == -1), "padding columns were written"
        want = parity.expected_owner_map(M, N, conf)
        assert np.array_equal(host[:, :N].astype(np.int64), want)
        ctas = np.unique(host[:, :N] & 0xFF)
        assert ctas.max() < conf["ctas"]


# ------------------------------------------------------------------ degenerate + errors
def test_k_zero_writes_zeros_and_empty_is_noop():
    for out in ("f32", "bf16"):
        a = np.zeros((37, 0), np.uint16)
        b = np.zeros((0, 53), np.uint16)
        got = run_case(a, b, out, pads=(4, 3, 5), what="K=0")
        assert np.all(got == 0)
    C = torch.full((4, 4), 7.0, device=DEV)
    A = torch.zeros((0, 4), dtype=torch.bfloat16, device=DEV)
    B = torch.zeros((4, 4), dtype=torch.bfloat16, device=DEV)
    assert tg.tile_gemm_raw(A.data_ptr(), B.data_ptr(), C.data_ptr(), 0, 4, 4, 4, 4, 4, 0) == 0
    assert tg.tile_gemm_raw(A.data_ptr(), B.data_ptr(), C.data_ptr(), 4, 0, 4, 4, 4, 4, 0) == 0
    torch.cuda.synchronize()
    assert torch.all(C == 7.0)


def test_precondition_failures_enqueue_nothing():
    C = torch.full((8, 8), 3.0, device=DEV)
    A = torch.ones((8, 8), dtype=torch.bfloat16, device=DEV)
    B = torch.ones((8, 8), dtype=torch.bfloat16, device=DEV)
    before = tg.tile_gemm_launch_count()
    p = (A.data_ptr(), B.data_ptr(), C.data_ptr())
    assert tg.tile_gemm_raw(*p, 8, 8, 8, 7, 8, 8, 0) == tg.E_LDA
    assert tg.tile_gemm_raw(*p, 8, 8, 8, 8, 7, 8, 0) == tg.E_LDB
    assert tg.tile_gemm_raw(*p, 8, 8, 8, 8, 8, 7, 0) == tg.E_LDC
    assert tg.tile_gemm_raw(*p, 8, 8, 8, 8, 8, 8, 3) == tg.E_DTYPE   # 2 is TILE_GEMM_OUT_F16 since the 8(f)1 rows
    assert tg.tile_gemm_raw(A.data_ptr(), B.data_ptr(), A.data_ptr(), 8, 8, 8, 8, 8, 8, 1) == tg.E_ALIAS
    assert tg.tile_gemm_raw(0, B.data_ptr(), C.data_ptr(), 8, 8, 8, 8, 8, 8, 0) == tg.E_NULL
    assert tg.tile_gemm_raw(*p, 8, 8, 8, 8, 8, 8, 0, 0, tg.PATH_GEMV) == tg.E_PATH
    torch.cuda.synchronize()
    assert tg.tile_gemm_launch_count() == before
    assert torch.all(C == 3.0)


# ------------------------------------------------------------------ host-buffer entry (e2e)
def test_host_entry_matches_oracle():
    a, b = wl.make_inputs_custom(333, 520, 129, "normal", seed=12)
    ref, S = oracle.gemm(a, b)
    C = np.full((333, 528), np.float32(-77.0))
    tg.tile_gemm_host(a, b, C[:, :520])
    check_close(C[:, :520], ref, S, 129, "f32", "host entry")
    assert np.all(C[:, 520:] == -77.0)
    x, W = wl.make_inputs_custom(1, 2048, 1024, "normal", seed=13)
    ref, S = oracle.gemm(x, W)
    y = np.zeros((1, 2048), np.uint16)
    tg.tile_gemm_host(x, W, y)
    check_close(oracle.bf16_decode(y), ref, S, 1024, "bf16", "host entry gemv")


@pytest.mark.parametrize("out", ["f32", "bf16"])
def test_host_entry_pipelined_chunks(out):
    """M >= 2048 goes up in 1024-row chunks with copy-in, GEMM and copy-out overlapped: same bits as one
    device call (integers: exact against the oracle), padded lda / ldc honoured, host padding untouched."""
    M, N, K = 2304 + 77, 520, 300                      # three chunks, the last one ragged
    a, b = wl.make_inputs_custom(M, N, K, "int4", seed=14)
    ref, _ = oracle.gemm(a, b)
    apad = np.full((M, K + 4), 0x7FC0, np.uint16)       # NaN padding columns in A
    apad[:, :K] = a
    if out == "f32":
        C = np.full((M, N + 8), np.float32(-77.0))
        tg.tile_gemm_host(apad[:, :K], b, C[:, :N])
        check_bit_exact(C[:, :N], ref, "pipelined host entry")
        assert np.all(C[:, N:] == -77.0)
    else:
        C = np.full((M, N + 8), 0x7FD5, np.uint16)
        tg.tile_gemm_host(apad[:, :K], b, C[:, :N])
        assert np.array_equal(oracle.bf16_decode(C[:, :N]), oracle.bf16_decode(oracle.bf16_encode(ref.astype(np.float32))))
        assert np.all(C[:, N:] == 0x7FD5)
    # and the one-shot path gives the same bits
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, 64)
    C2 = np.zeros_like(C)
    tg.tile_gemm_host(apad[:, :K], b, C2[:, :N])
    assert np.array_equal(C2[:, :N], C[:, :N])


# ------------------------------------------------------------------ split-K of the last wave
@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
@pytest.mark.parametrize("split", [2, 3, 5, 16])
def test_gemm_split_k_integer_bit_exact_and_canary(cfg, split):
    """Forced K slices (tuning key 3) on the ragged cfg2 shape and on a long-K shape: integer inputs
    are exact whatever the slicing, nothing outside C is written, every element is written."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMV_SPLIT, split)
    for (M, N, K), pads in (((1023, 1537, 769), (0, 0, 0)), ((300, 700, 4100), (8, 8, 8)), ((130, 520, 1030), (0, 0, 3))):
        a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=31 + split)
        ref, _ = oracle.gemm(a, b)
        got = run_case(a, b, "f32", pads=pads, what=f"split {split} cfg {cfg}")
        check_bit_exact(got.astype(np.float32), ref, f"split-K ints cfg{cfg} split{split} {M}x{N}x{K}")


@pytest.mark.parametrize("out", ["f32", "bf16"])
def test_gemm_split_k_auto_normal_inputs_and_determinism(out):
    """Shapes on which the selector itself slices K (a long-K last wave, skinny M): full oracle, and
    two runs give identical bits (slices are added in slice order, not arrival order)."""
    for (M, N, K) in ((8, 5120, 6400), (64, 1024, 8192), (2304, 2560, 6400)):
        a, b = wl.make_inputs_custom(M, N, K, sigma_b=K ** -0.5, seed=41)
        ref, S = oracle.gemm(a, b)
        got1 = run_case(a, b, out, what="split auto")
        got2 = run_case(a, b, out, what="split auto")
        check_close(got1, ref, S, K, out, f"split-K auto {M}x{N}x{K} {out}")
        assert np.array_equal(got1, got2), "split-K result depends on arrival order"


# ------------------------------------------------------------------ B multicast across two CTA pairs (tuning key 12)
@pytest.mark.parametrize("cap", [0, 8, 20])
def test_gemm_multicast_pairs_integer_bit_exact_and_canary(cap):
    """Config 4 with clusters of two CTA pairs that share every B stage through TMA multicast: ragged shapes, an odd
    number of tile rows (one pair of the last unit owns rows past M), few clusters walking many units; integer inputs
    are exact, nothing outside C is written, every element is written; lockstep producers on top stay exact."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, 4)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MULTICAST, 2)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MAX_CTAS, cap)
    for (M, N, K), pads in (((1023, 1537, 769), (0, 0, 0)), ((300, 700, 4100), (8, 8, 8)), ((1300, 520, 1030), (0, 0, 3)),
                            ((2304, 2560, 512), (0, 8, 0))):
        assert tg.tile_gemm_query_config(M, N, K)["config"] == 6
        a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=51 + cap)
        ref, _ = oracle.gemm(a, b)
        for out in ("f32", "bf16"):
            got = run_case(a, b, out, pads=pads, what=f"multicast pairs cap {cap}")
            if out == "f32":
                check_bit_exact(got.astype(np.float32), ref, f"multicast pairs {M}x{N}x{K} cap {cap}")
            else:
                assert np.array_equal(got, rne_bf16(ref))
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, 4 | (2 << 8))                  # lockstep forced on, window 2
    a, b = wl.make_inputs_custom(1023, 1537, 769, dist="int4", seed=59)
    ref, _ = oracle.gemm(a, b)
    check_bit_exact(run_case(a, b, "f32", what="multicast + lockstep").astype(np.float32), ref, "multicast + lockstep")


def test_gemm_multicast_pairs_give_the_bits_of_the_plain_config():
    """The MMA order per tile does not depend on how the operands reached shared memory."""
    M, N, K = 2304, 2560, 2048
    a, b = wl.make_inputs_custom(M, N, K, sigma_b=K ** -0.5, seed=58)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, 4)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MULTICAST, 1)
    plain = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MULTICAST, 2)
    mc = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32)
    torch.cuda.synchronize()
    assert torch.equal(plain, mc)
    rows, cols = wl.uniform_samples(M, N, 2048, seed=58)
    c, s = oracle.gemm_sampled(a, b, rows, cols)
    check_close(mc.cpu().numpy()[rows, cols], c, s, K, "f32", "multicast pairs sampled")


# ------------------------------------------------------------------ lockstep producers (long launches)
@pytest.mark.parametrize("window", [0, 1, 8, 200])
@pytest.mark.parametrize("cfg", [1, 3, 4])
def test_gemm_lockstep_forced_small_windows_bit_exact(cfg, window):
    """Lockstep forced on (tuning key 6 bit 2) with few CTAs so that every cluster walks many rounds
    and many windows: integer inputs stay exact, nothing hangs, nothing outside C is written."""
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_MAX_CTAS, 12)
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, 4 | (window << 8))
    a, b = wl.make_inputs_custom(1023, 1537, 769, dist="int4", seed=61)
    ref, _ = oracle.gemm(a, b)
    got = run_case(a, b, "f32", what=f"lockstep cfg{cfg} window{window}")
    check_bit_exact(got.astype(np.float32), ref, f"lockstep cfg{cfg} window{window}")


def test_gemm_long_k_auto_lockstep_and_split_sampled():
    """K = 16384 with 160 tiles on 74 clusters: the selector turns on lockstep producers (two whole
    rounds) AND slices the 12 left-over tiles along K.  Integer inputs: sampled elements exact; normal
    inputs: sampled oracle + Freivalds on the fp32 result + bf16 == RNE(fp32) bit for bit."""
    M, N, K = 4096, 5120, 16384
    a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=62)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    C = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32).cpu().numpy()
    rows, cols = wl.uniform_samples(M, N, 4096, seed=62)
    c, _ = oracle.gemm_sampled(a, b, rows, cols)
    check_bit_exact(C[rows, cols], c, "long-K ints sampled")
    a, b = wl.make_inputs_custom(M, N, K, sigma_b=K ** -0.5, seed=63)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    C32 = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32)
    C16 = tg.tile_gemm(A, B, out_dtype=tg.OUT_BF16)
    c, s = oracle.gemm_sampled(a, b, rows, cols)
    h32 = C32.cpu().numpy()
    check_close(h32[rows, cols], c, s, K, "f32", "long-K sampled")
    freivalds_rows(h32.astype(np.float64), oracle.bf16_decode(a), oracle.bf16_decode(b), seed=63)
    assert torch.equal(C16, C32.to(torch.bfloat16)), "bf16 output is not RNE of the fp32 output"
    C32b = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32)
    assert torch.equal(C32, C32b), "long-K result is not reproducible"


def test_selector_plans_for_the_benchmarked_shapes():
    """a2, extended: what the selector decides beyond the tile shape.  The tile counts and K-slice
    figures below are those of the 148-SM B200 the constants were measured on; CTA counts that are "one per
    column block" or "one per SM" are derived from the shape and the queried SM count."""
    plan = tg.tile_gemm_query_plan
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    blocks_51200 = -(-51200 // 128)       # the weight-streaming kernel: one CTA per 128-column block when unsliced
    p = plan(8192, 8192, 8192)            # cfg 3: whole tiles only (68 of 74 left over: cutting does not pay), K too short for lockstep
    assert p["config"] == 4 and p["split"] == 0 and p["full_units"] == 512 and p["lockstep_rounds"] == 0
    p = plan(4096, 5120, 25600)           # cfg 4 down: 12 of 160 tiles left over -> 6 K slices each, two lockstep rounds
    assert p["config"] == 4 and p["full_units"] == 148 and p["split"] == 6 and p["lockstep_rounds"] == 2
    assert p["split"] * p["k_tiles_per_slice"] >= 400 > (p["split"] - 1) * p["k_tiles_per_slice"]
    p = plan(32768, 32768, 32768)
    assert p["lockstep_rounds"] >= 100 and p["lockstep_window"] == 32
    assert plan(2048, 2048, 2048)["config"] == 3      # 64 pair tiles on 74 pairs: 256x256 pair tiles, not 128x256 single-CTA ones
    assert plan(1536, 1536, 2048)["config"] == 1      # 36 pair tiles or 72 of 128x256: too few, 144 single-CTA tiles of 128x128
    p = plan(1024, 1024, 1024)            # below one wave but a short K loop: not cut
    assert p["split"] == 0 and p["a_box_rows"] == 128
    for M in (2, 8, 16):                  # skinny M: the weight-streaming kernel, K-sliced over clusters; A box only as tall as M needs
        p = plan(M, 5120, 25600)
        assert p["config"] == 5 and p["full_units"] == 0 and p["split"] >= 4 and p["a_box_rows"] == 16 and sms <= p["ctas"] <= 2 * sms
    p = plan(24, 10240, 5120)
    assert p["config"] == 5 and p["a_box_rows"] == 32 and p["split"] >= 2
    for M in (8, 16):                     # column blocks that fill the CTA slots run unsliced
        p = plan(M, 51200, 5120)
        assert p["config"] == 5 and p["split"] == 0 and p["ctas"] == blocks_51200
    p = plan(32, 51200, 5120)             # 17..32 rows unsliced: a three-stage ring, three CTAs per SM, one wave
    assert p["config"] == 5 and p["split"] == 0 and p["ctas"] == blocks_51200 and p["a_box_rows"] == 32
    p = plan(40, 5120, 25600)             # 33..48 rows: still the weight-streaming kernel (three-stage ring, 64-row box)
    assert p["config"] == 5 and p["split"] >= 4 and p["a_box_rows"] == 64
    p = plan(64, 5120, 25600)             # 49..64 rows on weights that must be sliced: the tiled kernel, K-sliced below one wave
    assert p["config"] == 1 and p["full_units"] == 0 and p["split"] >= 2 and p["a_box_rows"] == 64 and p["ctas"] >= 100
    p = plan(64, 51200, 5120)             # ... on weights that run unsliced: the weight-streaming kernel
    assert p["config"] == 5 and p["split"] == 0 and p["ctas"] == blocks_51200
    p = plan(128, 51200, 5120)            # one row of 128-tall tiles: never a CTA pair, 128x128 tiles on every SM
    assert p["config"] == 1 and p["ctas"] == sms
    assert plan(129, 51200, 5120)["config"] in (3, 4)


# ------------------------------------------------------------------ 2 <= M <= 64: the weight-streaming tensor-core kernel
SKINNY_SHAPES = (((776, 1537), (0, 7, 3)), ((5120, 10240), (0, 0, 0)), ((64, 8), (8, 8, 0)), ((4104, 520), (8, 0, 8)),
                 ((1030, 130), (0, 6, 1)))


def _skinny_tune(mode=0, split=0, rows=0):
    tg.tile_gemm_set_tuning(tg.TUNE_SKINNY, mode | (split << 8) | (rows << 16))


@pytest.mark.parametrize("M", [2, 3, 4, 5, 8, 13, 16, 17, 31, 32, 33, 48, 57, 64])
@pytest.mark.parametrize("split", [0, 1, 2, 3, 4, 5, 6, 7, 8])
def test_skinny_integer_bit_exact_and_canary(M, split):
    """Every cluster size of the split-K reduce-scatter (1 = no cluster; 3, 5, 7: groups unevenly owned; 5..8: slices
    that own nothing) on ragged N, K and padded strides: integer inputs are exact whatever the slicing, nothing
    outside C is written, every element is written."""
    _skinny_tune(2, split)
    for (K, N), pads in SKINNY_SHAPES:
        a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=71 + M)
        ref, _ = oracle.gemm(a, b)
        pads_ok = (pads[0], pads[1] + (-(N + pads[1])) % 8, pads[2])          # ldb stays a multiple of 8: operands TMA-addressable
        assert tg.tile_gemm_query_plan(M, N, K)["config"] == 5
        got = run_case(a, b, "f32", pads=pads_ok, what=f"skinny M={M}")
        check_bit_exact(got.astype(np.float32), ref, f"skinny M={M} K={K} N={N} split={split}")


@pytest.mark.parametrize("M", [2, 8, 24, 32, 48])
@pytest.mark.parametrize("out", ["f32", "bf16"])
def test_skinny_normal_inputs_reproducible_and_agrees_with_the_tiled_gemm(M, out):
    K, N = 5120, 8192
    a, b = wl.make_inputs_custom(M, N, K, sigma_b=0.02, seed=73)
    ref, S = oracle.gemm(a, b)
    assert tg.tile_gemm_query_plan(M, N, K)["config"] == 5 and tg.tile_gemm_query_plan(M, N, K)["split"] >= 2
    got = run_case(a, b, out, what="skinny")
    check_close(got, ref, S, K, out, f"skinny M={M} {out}")
    again = run_case(a, b, out, what="skinny")
    assert np.array_equal(got, again), "the skinny-M kernel is not reproducible"
    static = run_case(a, b, out, what="skinny static_b", static_b=True)
    assert np.array_equal(got, static), "weights prefetched ahead of the dependency wait change the result"
    _skinny_tune(1)                                                         # the tiled kernel on the same problem
    assert tg.tile_gemm_query_plan(M, N, K)["config"] == 1
    tiled = run_case(a, b, out, what="tiled")
    check_close(tiled, ref, S, K, out, f"tiled M={M} {out}")


@pytest.mark.parametrize("M", [3, 8, 24, 40])
@pytest.mark.parametrize("static_b", [False, True])
def test_skinny_chain_is_stream_ordered_under_pdl(M, static_b):
    """C of one skinny-M GEMM is A of the next, launched back to back with programmatic dependent launch (weights
    prefetched ahead of the dependency wait when they are immutable, activations behind it): the bits must equal
    those of the same chain run with a synchronise after every launch, and every link must match the oracle on
    the bits it was given.  Shapes alternate so that consecutive launches differ in cluster size."""
    dims = [2048, 4096, 1024, 2048, 8192, 2048]
    rng = np.random.default_rng(33 + M)
    Ws = [wl.bits_to_torch(wl.f32_to_bf16_bits((rng.standard_normal((dims[i], dims[i + 1])) * dims[i] ** -0.5).astype(np.float32)), DEV)
          for i in range(len(dims) - 1)]
    x0 = wl.bits_to_torch(wl.f32_to_bf16_bits(rng.standard_normal((M, dims[0])).astype(np.float32)), DEV)
    for i in range(len(Ws)):
        assert tg.tile_gemm_query_plan(M, dims[i + 1], dims[i])["config"] == 5

    def chain(sync):
        xs = [x0] + [torch.empty((M, dims[i + 1]), dtype=torch.bfloat16, device=DEV) for i in range(len(Ws))]
        for i in range(len(Ws)):
            tg.tile_gemm(xs[i], Ws[i], xs[i + 1], static_b=static_b)
            if sync:
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        return xs

    want = chain(True)
    for i in range(len(Ws)):
        ref, S = oracle.gemm(wl.torch_to_bits(want[i]), wl.torch_to_bits(Ws[i]))
        check_close(want[i + 1].float().cpu().numpy(), ref, S, dims[i], "bf16", f"skinny chain link {i}")
    for rep in range(10):
        got = chain(False)
        for i in range(len(Ws) + 1):
            assert torch.equal(got[i].view(torch.int16), want[i].view(torch.int16)), f"rep {rep} link {i}"


def test_skinny_completes_next_to_a_kernel_that_holds_sms():
    """The plan sizes the clusters for an empty device; with 100 SMs held by another kernel they arrive in waves
    instead.  A slice only ever waits for the CTAs of its own cluster (which start together), so the launch still
    completes, with the same bits."""
    M, K, N = 8, 5120, 8192
    a, b = wl.make_inputs_custom(M, N, K, "int4", seed=78)
    ref, _ = oracle.gemm(a, b)
    A, W = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    assert tg.tile_gemm_query_plan(M, N, K)["split"] >= 2
    blocker, worker = torch.cuda.Stream(), torch.cuda.Stream()
    C = torch.full((M, N), float("nan"), dtype=torch.float32, device=DEV)
    torch.cuda.synchronize()
    tg.tile_gemm_debug_occupy(100, 20_000_000, stream=blocker)
    for _ in range(3):
        tg.tile_gemm(A, W, C, stream=worker, static_b=True)
    worker.synchronize()
    blocker.synchronize()
    check_bit_exact(C.cpu().numpy(), ref, "skinny M next to a blocker")


@pytest.mark.parametrize("M", [8, 24, 32, 64])
def test_skinny_unsliced_wide_weights(M):
    """Column blocks that fill the CTA slots run unsliced, in several waves or (17..32 rows: three-stage ring) three
    CTAs per SM: a ragged N just above 36864, integer inputs exact, canary intact."""
    N, K = 36864 + 72, 328
    p = tg.tile_gemm_query_plan(M, N, K)
    assert p["config"] == 5 and p["split"] == 0 and p["ctas"] == -(-N // 128)      # one CTA per 128-column block
    a, b = wl.make_inputs_custom(M, N, K, dist="int4", seed=79 + M)
    ref, _ = oracle.gemm(a, b)
    for out in ("f32", "bf16"):
        got = run_case(a, b, out, pads=(0, 8, 8), what=f"skinny unsliced M={M}", static_b=True)
        if out == "f32":
            check_bit_exact(got.astype(np.float32), ref, f"skinny unsliced M={M}")
        else:
            assert np.array_equal(got, rne_bf16(ref))


def test_skinny_32_row_box_for_few_rows_gives_the_same_bits():
    """The rows past M are TMA zero fill: a 32-row activation box (N = 32 of the MMA) on M = 8 changes nothing."""
    a, b = wl.make_inputs_custom(8, 1537 + 7, 2048, sigma_b=0.02, seed=76)
    got16 = run_case(a, b, "f32", what="skinny 16-row box")
    _skinny_tune(0, 0, 32)
    assert tg.tile_gemm_query_plan(8, 1544, 2048)["a_box_rows"] == 32
    got32 = run_case(a, b, "f32", what="skinny 32-row box")
    assert np.array_equal(got16, got32)


def test_skinny_f16_and_unaligned_falls_back_to_the_tiled_gemm():
    a, b = wl.make_inputs_f16(3, 2048, 1024, sigma_b=0.05, seed=74)
    ref, S = oracle.gemm(a, b, in_dtype=oracle.IN_F16)
    A, B = wl.bits_to_torch(a, DEV, torch.float16), wl.bits_to_torch(b, DEV, torch.float16)
    C = tg.tile_gemm(A, B, out_dtype=tg.OUT_F16)
    check_close(oracle.f16_decode(C.cpu().view(torch.int16).numpy().view(np.uint16)), ref, S, 1024, "f16", "skinny f16")
    ai, bi = wl.make_inputs_f16(20, 1000, 520, dist="int4", seed=77)           # f16 integers through the f16 decode: exact
    refi, _ = oracle.gemm(ai, bi, in_dtype=oracle.IN_F16)
    Ci = tg.tile_gemm(wl.bits_to_torch(ai, DEV, torch.float16), wl.bits_to_torch(bi, DEV, torch.float16), out_dtype=tg.OUT_F32)
    check_bit_exact(Ci.cpu().numpy(), refi, "skinny f16 ints")
    # lda not a multiple of 8: A is not TMA-addressable, the selector goes to the (repacking) tiled GEMM
    assert tg.tile_gemm_select(3, 2048, 1023, 1023, 2048, 2048) == tg.PATH_GEMM_REPACK
    ai, bi = wl.make_inputs_custom(3, 2048, 1023, dist="int4", seed=75)
    refi, _ = oracle.gemm(ai, bi)
    check_bit_exact(run_case(ai, bi, "f32").astype(np.float32), refi, "M=3 unaligned")
