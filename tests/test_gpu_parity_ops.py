"""Parity of the SURVEY.md 8(f) rows (through the C ABI) against the oracle, on a B200:
element-wise add (Listing 1; bit-exact, the paper fixes f32) and the GEMM with
f16 inputs / f16 output (the paper's sweep is in f16; same gates as bf16)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15991_b200 import binding as tg
from paper_2606_15991_b200 import workloads as wl
from parity import check_bit_exact, check_close, freivalds_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"
CANARY = 0x7FC0DEAD


@pytest.fixture(autouse=True)
def _reset_tuning():
    yield
    for key in range(tg.NUM_TUNE_KEYS):
        tg.tile_gemm_set_tuning(key, 0)
    torch.cuda.synchronize()


# ------------------------------------------------------------------ element-wise add
def run_add(x, y, offset=(0, 0, 0)):
    """x, y: host float32.  Buffers sit `offset` elements past a 256-byte aligned base, z between
    canary guards.  Returns z (host) after checking the guards."""
    n = x.size
    G = 64

    def dev(v, off):
        buf = torch.zeros(n + off + 8, dtype=torch.float32, device=DEV)
        view = buf[off:off + n]
        view.copy_(torch.from_numpy(v))
        return view

    xd, yd = dev(x, offset[0]), dev(y, offset[1])
    zraw = torch.empty(n + 2 * G + offset[2] + 8, dtype=torch.int32, device=DEV)
    zraw.fill_(np.int32(CANARY))
    zd = zraw[G + offset[2]:G + offset[2] + n].view(torch.float32)
    tg.tile_add_f32(xd, yd, zd)
    torch.cuda.synchronize()
    bits = zraw.cpu().numpy().view(np.uint32)
    lo = G + offset[2]
    assert np.all(bits[:lo] == CANARY) and np.all(bits[lo + n:] == CANARY), "written outside z[0:n)"
    return bits[lo:lo + n].view(np.float32).copy()


def test_add_paper_example():
    x = np.ones(1024, np.float32)
    z = run_add(x, x.copy())
    assert np.all(z == 2.0)


@pytest.mark.parametrize("n", [1, 3, 4, 5, 1023, 1024, 4095, 4096, 4097, 100_003, 148 * 8 * 4096 + 4099, 1 << 22])
@pytest.mark.parametrize("shape", [0, 8 * 16 + 1, 4 * 16 + 8, 16 * 16 + 2])
def test_add_bit_exact_ragged_sizes(n, shape):
    tg.tile_gemm_set_tuning(tg.TUNE_ADD_SHAPE, shape)
    x, y = wl.make_add_inputs(n, seed=n)
    z = run_add(x, y)
    ref = oracle.add_f32(x, y)
    assert np.array_equal(z.view(np.uint32), ref.view(np.uint32))


@pytest.mark.parametrize("offset", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (1, 1, 1), (4, 4, 4)])
def test_add_unaligned_buffers(offset):
    n = 70_001
    x, y = wl.make_add_inputs(n, seed=11)
    z = run_add(x, y, offset)
    assert np.array_equal(z.view(np.uint32), oracle.add_f32(x, y).view(np.uint32))


def test_add_ieee_cases_and_specials():
    vals = np.array([1.0, 2.0 ** -24, 1.5 * 2.0 ** -23, 3.0, -3.0, 3.4028235e38, 2.0 ** 103, 1e-45, -1e-45,
                     2.0 ** -126, 0.0, -0.0], np.float32)
    x = np.repeat(vals, vals.size)
    y = np.tile(vals, vals.size)
    z = run_add(x, y)
    ref = oracle.add_f32(x, y)
    assert np.array_equal(z.view(np.uint32), ref.view(np.uint32))


def test_add_full_size_sampled():
    """n = 2^28, device-generated; the oracle checks 2^20 strided elements and a
    checksum identity covers the rest: sum(z) over int32-valued inputs is exact."""
    n = 1 << 28
    g = torch.Generator(device=DEV)
    g.manual_seed(28)
    x = torch.empty(n, dtype=torch.float32, device=DEV).normal_(0, 1, generator=g)
    y = torch.empty(n, dtype=torch.float32, device=DEV).normal_(0, 1, generator=g)
    z = tg.tile_add_f32(x, y)
    idx = torch.arange(0, n, 256, device=DEV) + torch.randint(0, 256, (n // 256,), device=DEV, generator=g)
    xs, ys, zs = x[idx].cpu().numpy(), y[idx].cpu().numpy(), z[idx].cpu().numpy()
    assert np.array_equal(zs.view(np.uint32), oracle.add_f32(xs, ys).view(np.uint32))
    # small integers: every element and every partial sum exact, so sum(z) = sum(x) + sum(y) holds exactly
    xi = torch.randint(-8, 9, (n,), device=DEV, generator=g).float()
    yi = torch.randint(-8, 9, (n,), device=DEV, generator=g).float()
    zi = tg.tile_add_f32(xi, yi)
    assert int(zi.double().sum().item()) == int(xi.double().sum().item()) + int(yi.double().sum().item())
    assert float(zi.abs().max().item()) <= 16.0


def test_add_preconditions():
    x = torch.zeros(64, dtype=torch.float32, device=DEV)
    z = torch.full((64,), 7.0, dtype=torch.float32, device=DEV)
    p, q = x.data_ptr(), z.data_ptr()
    assert tg.tile_add_f32_raw(p, p, q, -1) == tg.E_EXTENT
    assert tg.tile_add_f32_raw(p, 0, q, 8) == tg.E_NULL
    assert tg.tile_add_f32_raw(p + 2, p, q, 8) == tg.E_ALIGN
    assert tg.tile_add_f32_raw(p, p, p + 16, 8) == tg.E_ALIAS
    assert tg.tile_add_f32_raw(p, p, q, 0) == tg.E_OK
    assert tg.tile_add_f32_raw(p, p, q, 8) == tg.E_OK          # x and y may be the same buffer (shared reads)
    torch.cuda.synchronize()
    assert torch.all(z[:8] == 0) and torch.all(z[8:] == 7.0)


# ------------------------------------------------------------------ f16 GEMM
def run_f16(a_bits, b_bits, out, in_f16=True, pad=0):
    M, K = a_bits.shape
    N = b_bits.shape[1]
    dt = torch.float16 if in_f16 else torch.bfloat16
    A = torch.zeros((M, K + pad), dtype=dt, device=DEV)[:, :K]
    B = torch.zeros((K, N + pad), dtype=dt, device=DEV)[:, :N]
    A.copy_(wl.bits_to_torch(a_bits, DEV, dt))
    B.copy_(wl.bits_to_torch(b_bits, DEV, dt))
    odt = {"f32": torch.float32, "bf16": torch.bfloat16, "f16": torch.float16}[out]
    Cfull = torch.full((M + 2, N + pad + 8), float("nan"), dtype=odt, device=DEV)
    C = Cfull[1:M + 1, :N]
    tg.tile_gemm(A, B, C)
    torch.cuda.synchronize()
    host = Cfull.cpu()
    assert torch.isnan(host[0]).all() and torch.isnan(host[-1]).all() and torch.isnan(host[:, N:]).all(), \
        "written outside C"
    c = host[1:M + 1, :N].contiguous()
    if out == "f32":
        return c.numpy().astype(np.float64)
    if out == "f16":
        return oracle.f16_decode(c.view(torch.int16).numpy().view(np.uint16))
    return oracle.bf16_decode(c.view(torch.int16).numpy().view(np.uint16))


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_f16_integer_inputs_bit_exact(cfg):
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, cfg)
    a, b = wl.make_inputs_f16(1023, 1537, 769, dist="int4", seed=21)
    ref, _ = oracle.gemm(a, b, in_dtype=oracle.IN_F16)
    got = run_f16(a, b, "f32")
    check_bit_exact(got.astype(np.float32), ref, f"f16 ints cfg{cfg}")


def test_f16_bits_are_not_read_as_bf16():
    # 0x3C00 is 1.0 in f16 and 2^-7 in bf16; all-ones f16 inputs give C = K exactly
    K = 2049
    a = np.full((130, K), 0x3C00, np.uint16)
    b = np.full((K, 70), 0x3C00, np.uint16)
    assert np.all(run_f16(a, b, "f32") == K)
    # binary16 spacing in [2048, 4096) is 2: 2049 is the tie between 2048 and 2050 -> even -> 2048
    assert np.all(run_f16(a, b, "f16") == 2048)


@pytest.mark.parametrize("out", ["f32", "f16", "bf16"])
@pytest.mark.parametrize("pad", [0, 8, 3])
def test_f16_ragged_full_oracle(out, pad):
    a, b = wl.make_inputs_f16(1023, 1537, 769, seed=22)
    b[5::97] = wl.f32_to_f16_bits(np.full(b[5::97].shape, 3e-6, np.float32))     # subnormal f16 inputs
    ref, S = oracle.gemm(a, b, in_dtype=oracle.IN_F16)
    got = run_f16(a, b, out, pad=pad)
    check_close(got, ref, S, 769, out, f"f16 ragged out={out} pad={pad}")


def test_bf16_inputs_with_f16_output():
    a, b = wl.make_inputs_custom(300, 520, 1000, sigma_b=1000 ** -0.5, seed=23)
    ref, S = oracle.gemm(a, b)
    got = run_f16(a, b, "f16", in_f16=False)
    check_close(got, ref, S, 1000, "f16", "bf16 in, f16 out")


def test_f16_output_is_rne_of_the_fp32_result():
    a, b = wl.make_inputs_f16(512, 768, 2048, sigma_b=2048 ** -0.5, seed=24)
    b[:, ::5] = wl.f32_to_f16_bits(np.float32(1e-3) * wl.bits_to_torch(b[:, ::5], dtype=torch.float16).float().numpy())
    c32 = run_f16(a, b, "f32").astype(np.float32)
    dt = torch.float16
    A, B = wl.bits_to_torch(a, DEV, dt), wl.bits_to_torch(b, DEV, dt)
    C16 = tg.tile_gemm(A, B, out_dtype=tg.OUT_F16)
    got = C16.cpu().view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(got, oracle.f16_encode(c32))


@pytest.mark.parametrize("K,N", [(5120, 10240), (769, 1537), (64, 8)])
@pytest.mark.parametrize("out", ["f32", "f16"])
def test_f16_gemv(K, N, out):
    a, b = wl.make_inputs_f16(1, N, K, sigma_b=0.02, seed=25)
    ref, S = oracle.gemm(a, b, in_dtype=oracle.IN_F16)
    got = run_f16(a, b, out)
    check_close(got, ref, S, K, out, f"f16 gemv K={K} N={N} out={out}")
    ai, bi = wl.make_inputs_f16(1, N, K, dist="int4", seed=26)
    refi, _ = oracle.gemm(ai, bi, in_dtype=oracle.IN_F16)
    check_bit_exact(run_f16(ai, bi, "f32").astype(np.float32), refi, "f16 gemv ints")


def test_f16_4096_sampled_and_freivalds():
    M = N = K = 4096
    a, b = wl.make_inputs_f16(M, N, K, sigma_b=K ** -0.5, seed=27)
    dt = torch.float16
    A, B = wl.bits_to_torch(a, DEV, dt), wl.bits_to_torch(b, DEV, dt)
    C32 = tg.tile_gemm(A, B, out_dtype=tg.OUT_F32).cpu().numpy()
    rows, cols = wl.stratified_samples(M, N, 128, seed=27)
    c, s = oracle.gemm_sampled(a, b, rows, cols, in_dtype=oracle.IN_F16)
    check_close(C32[rows, cols], c, s, K, "f32", "f16 4096 sampled")
    freivalds_rows(C32.astype(np.float64), oracle.f16_decode(a), oracle.f16_decode(b), seed=27)
    C16 = tg.tile_gemm(A, B, out_dtype=tg.OUT_F16).cpu().view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(C16, oracle.f16_encode(C32))


def test_typed_preconditions():
    x = torch.zeros((8, 8), dtype=torch.float16, device=DEV)
    c = torch.full((8, 8), 5.0, dtype=torch.float32, device=DEV)
    assert tg.tile_gemm_typed_raw(x.data_ptr(), x.data_ptr(), c.data_ptr(), 8, 8, 8, 8, 8, 8, 5, tg.OUT_F32) == tg.E_IN_DTYPE
    assert tg.tile_gemm_typed_raw(x.data_ptr(), x.data_ptr(), c.data_ptr(), 8, 8, 8, 8, 8, 8, tg.IN_F16, 3) == tg.E_DTYPE
    torch.cuda.synchronize()
    assert torch.all(c == 5.0)


# ------------------------------------------------------------------ recorded steps
def test_recorded_step_replays_bit_identically_and_follows_new_inputs():
    """A decode-like chain (4 GEMVs on the Qwen3 shapes scaled down, a GEMM and an add) recorded once
    and replayed: same bits as the direct calls, and a replay after rewriting the inputs in place
    matches the oracle on the new data (nodes keep addresses, not contents)."""
    s = torch.cuda.Stream()
    shapes = [(640, 1280), (640, 1024), (640, 6400), (3200, 640)]
    xs = [torch.empty((1, K), dtype=torch.bfloat16, device=DEV) for K, N in shapes]
    Ws = [torch.empty((K, N), dtype=torch.bfloat16, device=DEV) for K, N in shapes]
    ys = [torch.empty((1, N), dtype=torch.float32, device=DEV) for K, N in shapes]
    A = torch.empty((300, 640), dtype=torch.bfloat16, device=DEV)
    C = torch.empty((300, 1280), dtype=torch.float32, device=DEV)
    u = torch.empty(5000, dtype=torch.float32, device=DEV)
    v = torch.empty(5000, dtype=torch.float32, device=DEV)
    w = torch.empty(5000, dtype=torch.float32, device=DEV)

    def fill(seed):
        host = []
        for i, (K, N) in enumerate(shapes):
            a, b = wl.make_inputs_custom(1, N, K, sigma_b=0.05, seed=seed * 10 + i)
            xs[i].copy_(wl.bits_to_torch(a, DEV))
            Ws[i].copy_(wl.bits_to_torch(b, DEV))
            host.append((a, b))
        a, _ = wl.make_inputs_custom(300, 8, 640, seed=seed * 10 + 9)
        A.copy_(wl.bits_to_torch(a, DEV))
        hu, hv = wl.make_add_inputs(5000, seed=seed)
        u.copy_(torch.from_numpy(hu))
        v.copy_(torch.from_numpy(hv))
        return host, a, hu, hv

    def chain(stream):
        for i in range(4):
            tg.tile_gemm(xs[i], Ws[i], ys[i], stream=stream, static_b=True)
        tg.tile_gemm(A, Ws[0], C, stream=stream)
        tg.tile_add_f32(u, v, w, stream=stream)

    fill(1)
    chain(s)                                    # warm-up on the stream: workspaces exist before recording
    s.synchronize()
    direct = [y.clone() for y in ys] + [C.clone(), w.clone()]
    before = tg.tile_gemm_launch_count()
    tg.tile_gemm_record_begin(s)
    chain(s)
    step = tg.tile_gemm_record_end(s)
    s.synchronize()
    assert tg.tile_gemm_launch_count() - before == 6, "recording counts the recorded kernels once"
    assert step.nodes >= 6
    for t in ys + [C, w]:
        t.fill_(float("nan"))                   # recording executed nothing
    step.replay(s)
    s.synchronize()
    for got, want in zip(ys + [C, w], direct):
        assert torch.equal(got, want)
    host, a_host, hu, hv = fill(2)              # new contents, same addresses
    step.replay(s)
    step.replay(s)
    s.synchronize()
    for i, (K, N) in enumerate(shapes):
        ref, S = oracle.gemm(*host[i])
        check_close(ys[i].cpu().numpy().astype(np.float64), ref, S, K, "f32", f"replayed gemv {i}")
    ref, S = oracle.gemm(a_host, host[0][1])
    check_close(C.cpu().numpy().astype(np.float64), ref, S, 640, "f32", "replayed gemm")
    assert np.array_equal(w.cpu().numpy().view(np.uint32), oracle.add_f32(hu, hv).view(np.uint32))
    step.free()
    assert step.nodes == -1


def test_record_preconditions():
    lib = tg.load_library()
    assert lib.tile_gemm_record_begin(None) == tg.E_PATH
    assert lib.tile_gemm_replay(None, None) == tg.E_NULL
    assert lib.tile_gemm_record_free(None) == tg.E_OK


# ------------------------------------------------------------------ SwiGLU epilogue
def swiglu_gate(got, H, G, U, Sg, Su, K, out, what):
    """|err| <= output rounding + the two accumulation errors pushed through h = silu(g) * u
    (|silu'| <= 1.1) + 2^-18 |H| for the fast exp / divide."""
    eg = 2.0 * K * 2.0 ** -24 * Sg
    eu = 2.0 * K * 2.0 ** -24 * Su
    rnd = {"f32": 2.0 ** -23 * np.abs(H), "bf16": 2.0 ** -8 * np.abs(H), "f16": 2.0 ** -11 * np.abs(H) + 2.0 ** -24}[out]
    tol = rnd + 1.1 * np.abs(U) * eg + np.abs(oracle.silu(G)) * eu + 2.0 ** -18 * np.abs(H) + 1e-30
    err = np.abs(got - H)
    assert not np.isnan(got).any(), f"{what}: NaN"
    bad = err > tol
    assert not bad.any(), f"{what}: {int(bad.sum())} elements out of tolerance, first {np.argwhere(bad)[:4].tolist()}, max ratio {np.max(err / tol):.3g}"


def run_swiglu(x_bits, w_bits, out, pad=0):
    M, K = x_bits.shape
    inter = w_bits.shape[1] // 2
    ldw = (2 * inter + 7) // 8 * 8 + pad
    ldx = (K + 7) // 8 * 8
    X = torch.zeros((M, ldx), dtype=torch.bfloat16, device=DEV)[:, :K]
    W = torch.full((K, ldw), float("nan"), dtype=torch.bfloat16, device=DEV)[:, :2 * inter]
    X.copy_(wl.bits_to_torch(x_bits, DEV))
    W.copy_(wl.bits_to_torch(w_bits, DEV))
    odt = {"f32": torch.float32, "bf16": torch.bfloat16, "f16": torch.float16}[out]
    Hfull = torch.full((M + 2, inter + 8 + pad), float("nan"), dtype=odt, device=DEV)
    H = Hfull[1:M + 1, :inter]
    tg.tile_gemm_swiglu(X, W, H)
    torch.cuda.synchronize()
    host = Hfull.cpu()
    assert torch.isnan(host[0]).all() and torch.isnan(host[-1]).all() and torch.isnan(host[:, inter:]).all(), "written outside H"
    h = host[1:M + 1, :inter].contiguous()
    if out == "f32":
        return h.numpy().astype(np.float64)
    bits = h.view(torch.int16).numpy().view(np.uint16)
    return oracle.f16_decode(bits) if out == "f16" else oracle.bf16_decode(bits)


@pytest.mark.parametrize("out", ["f32", "bf16", "f16"])
@pytest.mark.parametrize("shape", [(1023, 1544, 769), (300, 256, 64), (8, 1000, 4100), (513, 520, 1030)])
def test_swiglu_full_oracle_ragged(out, shape):
    M, inter, K = shape
    x, w = wl.make_inputs_custom(M, 2 * inter, K, sigma_b=2.0 * K ** -0.5, seed=51)
    H, G, U, Sg, Su = oracle.swiglu_gemm(x, w)
    got = run_swiglu(x, w, out, pad=8 if M == 513 else 0)
    swiglu_gate(got, H, G, U, Sg, Su, K, out, f"swiglu {shape} {out}")


def test_swiglu_integer_inputs_and_special_halves():
    M, inter, K = 260, 296, 200
    x, w = wl.make_inputs_custom(M, 2 * inter, K, dist="int4", seed=52)
    H, G, U, Sg, Su = oracle.swiglu_gemm(x, w)                       # G, U exact integers up to 3200
    got = run_swiglu(x, w, "f32")
    assert np.all(np.abs(got - H) <= 2.0 ** -18 * np.abs(H) + 1e-30)
    assert np.all(got[(G == 0) | (U == 0)] == 0)                      # silu(0) * u = 0 and g * 0 = 0, exactly
    assert np.all(got[G < -110] == 0) and not np.isnan(got).any()     # e^110 overflows fp32: the left tail is a clean zero
    wz = w.copy()
    wz[:, :inter] = 0                                                 # gate weights zero -> H = 0 everywhere
    assert np.all(run_swiglu(x, wz, "bf16") == 0)
    ws = np.concatenate([w[:, inter:], w[:, :inter]], axis=1)         # swapped halves: silu(U) * G, not silu(G) * U
    Hs = oracle.swiglu_gemm(x, ws)[0]
    gots = run_swiglu(x, ws, "f32")
    assert np.all(np.abs(gots - Hs) <= 2.0 ** -18 * np.abs(Hs) + 1e-30)
    assert not np.allclose(Hs, H)


def test_swiglu_matches_two_gemms_of_the_same_library():
    """The fused kernel's accumulators are the ones tile_gemm produces for the two halves: H must
    equal silu(G32) * U32 evaluated on those fp32 results to fast-math accuracy."""
    M, inter, K = 512, 768, 2048
    x, w = wl.make_inputs_custom(M, 2 * inter, K, sigma_b=2.0 * K ** -0.5, seed=53)
    X, W = wl.bits_to_torch(x, DEV), wl.bits_to_torch(w, DEV)
    tg.tile_gemm_set_tuning(tg.TUNE_GEMM_CONFIG, 4)
    G32 = tg.tile_gemm(X, W[:, :inter], out_dtype=tg.OUT_F32).double()
    U32 = tg.tile_gemm(X, W[:, inter:], out_dtype=tg.OUT_F32).double()
    H = tg.tile_gemm_swiglu(X, W, out_dtype=tg.OUT_F32).double()
    ref = G32 / (1 + torch.exp(-G32)) * U32
    assert torch.all((H - ref).abs() <= 2.0 ** -18 * ref.abs() + 1e-30)


def test_swiglu_gate_up_shape_sampled():
    """BASELINE.json's fused gate/up projection (M=4096, K=5120, 2I=51200), sampled against the oracle."""
    M, K, inter = 4096, 5120, 25600
    g = torch.Generator(device=DEV)
    g.manual_seed(54)
    X = torch.empty((M, K), dtype=torch.bfloat16, device=DEV).normal_(0, 1, generator=g)
    W = torch.empty((K, 2 * inter), dtype=torch.bfloat16, device=DEV).normal_(0, 0.02, generator=g)
    H = tg.tile_gemm_swiglu(X, W, out_dtype=tg.OUT_BF16)
    rows, cols = wl.uniform_samples(M, inter, 2048, seed=54)
    xb, wb = wl.torch_to_bits(X), wl.torch_to_bits(W)
    Gs, Sg = oracle.gemm_sampled(xb, wb, rows, cols)
    Us, Su = oracle.gemm_sampled(xb, wb, rows, cols + inter)
    got = oracle.bf16_decode(wl.torch_to_bits(H)[rows, cols])
    swiglu_gate(got, oracle.silu(Gs) * Us, Gs, Us, Sg, Su, K, "bf16", "swiglu gate_up sampled")
    assert torch.isfinite(H.float()).all()


def test_swiglu_preconditions():
    X = torch.zeros((8, 64), dtype=torch.bfloat16, device=DEV)
    W = torch.zeros((64, 32), dtype=torch.bfloat16, device=DEV)
    H = torch.full((8, 16), 3.0, dtype=torch.float32, device=DEV)
    a = (X.data_ptr(), W.data_ptr(), H.data_ptr())
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 31, 16, tg.OUT_F32) == tg.E_LDB         # ldw < 2I
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 63, 32, 16, tg.OUT_F32) == tg.E_LDA
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 32, 15, tg.OUT_F32) == tg.E_LDC
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 64, 64, 32, 16, 5) == tg.E_DTYPE
    assert tg.tile_gemm_swiglu_raw(X.data_ptr() + 2, W.data_ptr(), H.data_ptr(), 8, 16, 56, 64, 32, 16, tg.OUT_F32) == tg.E_PATH
    assert tg.tile_gemm_swiglu_raw(X.data_ptr(), W.data_ptr(), W.data_ptr() + 32, 8, 8, 64, 64, 32, 16, tg.OUT_BF16) == tg.E_ALIAS
    assert tg.tile_gemm_swiglu_raw(*a, 8, 12, 64, 64, 32, 16, tg.OUT_F32) == tg.E_PATH        # I not a multiple of 8
    torch.cuda.synchronize()
    assert torch.all(H == 3.0)
    assert tg.tile_gemm_swiglu_raw(*a, 8, 16, 0, 64, 32, 16, tg.OUT_F32) == tg.E_OK            # K == 0 -> zeros
    torch.cuda.synchronize()
    assert torch.all(H == 0.0)


def test_recorded_step_with_lockstep_and_split_gemm():
    """A long-K GEMM (lockstep counters zeroed by a memset node, K-cut last wave with workspace and
    tickets) inside a recorded step: two replays give the bits of the direct call."""
    M, N, K = 2048, 5120, 16384
    a, b = wl.make_inputs_custom(M, N, K, sigma_b=K ** -0.5, seed=81)
    A, B = wl.bits_to_torch(a, DEV), wl.bits_to_torch(b, DEV)
    s = torch.cuda.Stream()
    tg.tile_gemm_set_tuning(tg.TUNE_FLAGS, 4)            # lockstep on even with one whole round
    C = torch.empty((M, N), dtype=torch.bfloat16, device=DEV)
    tg.tile_gemm(A, B, C, stream=s)
    s.synchronize()
    want = C.clone()
    tg.tile_gemm_record_begin(s)
    tg.tile_gemm(A, B, C, stream=s)
    step = tg.tile_gemm_record_end(s)
    assert step.nodes >= 2                               # the kernel and its memset
    for _ in range(2):
        C.zero_()
        step.replay(s)
        s.synchronize()
        assert torch.equal(C, want)
    step.free()
    rows, cols = wl.uniform_samples(M, N, 1024, seed=81)
    c, sc = oracle.gemm_sampled(a, b, rows, cols)
    check_close(oracle.bf16_decode(wl.torch_to_bits(want)[rows, cols]), c, sc, K, "bf16", "recorded long-K GEMM")


# ------------------------------------------------------------------ read-bandwidth probe
@pytest.mark.parametrize("n", [0, 1, 3, 4, 1023, 1024, 1025, 1027, 100_003, (1 << 24) + 5])
def test_read_probe_is_the_word_sum(n):
    g = torch.Generator(device=DEV)
    g.manual_seed(90 + n % 97)
    buf = torch.randint(-2 ** 31, 2 ** 31 - 1, (n + 4,), dtype=torch.int32, device=DEV, generator=g)[:n]
    out = torch.full((1,), 5, dtype=torch.int64, device=DEV)          # accumulates on top of what is there
    lib = tg.load_library()
    import ctypes
    rc = lib.tile_read_probe_u32(ctypes.c_void_p(buf.data_ptr()), n, ctypes.c_void_p(out.data_ptr()), None)
    assert rc == tg.E_OK
    torch.cuda.synchronize()
    want = (oracle.word_sum_u32(buf.cpu().numpy()) + 5) % 2 ** 64
    assert int(out.item()) % 2 ** 64 == want


def test_read_probe_preconditions():
    import ctypes
    lib = tg.load_library()
    buf = torch.zeros(64, dtype=torch.int32, device=DEV)
    out = torch.zeros(1, dtype=torch.int64, device=DEV)
    vp = ctypes.c_void_p
    assert lib.tile_read_probe_u32(vp(buf.data_ptr()), -1, vp(out.data_ptr()), None) == tg.E_EXTENT
    assert lib.tile_read_probe_u32(vp(buf.data_ptr() + 4), 8, vp(out.data_ptr()), None) == tg.E_ALIGN
    assert lib.tile_read_probe_u32(vp(buf.data_ptr()), 8, None, None) == tg.E_NULL
    assert lib.tile_read_probe_u32(vp(buf.data_ptr()), 64, vp(buf.data_ptr() + 8), None) == tg.E_ALIAS
