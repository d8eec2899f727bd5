"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end to ``gemm_oracle.c``: the plain fp64 CPU statement of
``C = A @ B`` (Listing 2) used to judge the CUDA path, and to
``ops_oracle.c``: the element-wise add of Listing 1 and the
binary16 encoder.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_2606_15991_b200`` and that package imports
nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gemm_oracle.c")
_SRC_OPS = os.path.join(_HERE, "ops_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_gemm.so")
_lib = None

_i64 = ctypes.c_int64
_u16p = ctypes.POINTER(ctypes.c_uint16)
_f64p = ctypes.POINTER(ctypes.c_double)
_f32p = ctypes.POINTER(ctypes.c_float)
_i64p = ctypes.POINTER(ctypes.c_int64)


def build(force: bool = False) -> str:
    """Compile gemm_oracle.c and ops_oracle.c with gcc (x86-64-v3: runs on any AVX2 host)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_OPS))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O3", "-march=x86-64-v3", "-std=c11", "-fPIC", "-shared",
               "-pthread", "-o", _LIB, _SRC, _SRC_OPS, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_gemm.restype = ctypes.c_int
        lib.oracle_gemm.argtypes = [_u16p, _u16p, _f64p, _f64p, _i64, _i64, _i64, _i64, _i64,
                                    _i64, ctypes.c_int, _i64, _i64, _i64]
        lib.oracle_gemm_sampled.restype = ctypes.c_int
        lib.oracle_gemm_sampled.argtypes = [_u16p, _u16p, _i64p, _i64p, _i64, _f64p, _f64p,
                                            _i64, _i64, _i64, _i64, _i64]
        lib.oracle_gemm_typed.restype = ctypes.c_int
        lib.oracle_gemm_typed.argtypes = lib.oracle_gemm.argtypes + [ctypes.c_int]
        lib.oracle_gemm_sampled_typed.restype = ctypes.c_int
        lib.oracle_gemm_sampled_typed.argtypes = lib.oracle_gemm_sampled.argtypes + [ctypes.c_int]
        lib.oracle_f16_decode_array.restype = None
        lib.oracle_f16_decode_array.argtypes = [_u16p, _f64p, _i64]
        lib.oracle_f16_encode_array.restype = None
        lib.oracle_f16_encode_array.argtypes = [_f32p, _u16p, _i64]
        lib.oracle_add_f32.restype = None
        lib.oracle_add_f32.argtypes = [_f32p, _f32p, _f32p, _i64]
        lib.oracle_bf16_decode_array.restype = None
        lib.oracle_bf16_decode_array.argtypes = [_u16p, _f64p, _i64]
        lib.oracle_bf16_encode_array.restype = None
        lib.oracle_bf16_encode_array.argtypes = [_f32p, _u16p, _i64]
        _lib = lib
    return _lib


def default_threads() -> int:
    return max(1, len(os.sched_getaffinity(0)))


def _as_u16_2d(x, name):
    x = np.asarray(x)
    if x.dtype != np.uint16 or x.ndim != 2:
        raise TypeError(f"{name} must be a 2-D uint16 array of bf16 bit patterns")
    if x.strides[1] != 2 or x.strides[0] % 2 or x.strides[0] < 2 * x.shape[1]:
        x = np.ascontiguousarray(x)
    return x


IN_BF16, IN_F16 = 0, 1


def gemm(A, B, threads: int | None = None, blocks=(0, 0, 0), in_dtype: int = IN_BF16):
    """Full fp64 GEMM.  A: (M,K) uint16 bit patterns (bf16, or binary16 when
    in_dtype == IN_F16), B: (K,N).  Row strides are taken from the arrays
    (padded leading dimensions are honoured).
    Returns (C, S) float64 (M,N): C = A@B and S = |A|@|B|."""
    A = _as_u16_2d(A, "A")
    B = _as_u16_2d(B, "B")
    M, K = A.shape
    K2, N = B.shape
    if K != K2:
        raise ValueError("inner dimensions differ")
    C = np.empty((M, N), dtype=np.float64)
    S = np.empty((M, N), dtype=np.float64)
    lda = A.strides[0] // 2 if M > 1 else max(K, 1)
    ldb = B.strides[0] // 2 if K > 1 else max(N, 1)
    lda, ldb = max(lda, K), max(ldb, N)
    rc = _load().oracle_gemm_typed(A.ctypes.data_as(_u16p), B.ctypes.data_as(_u16p),
                                   C.ctypes.data_as(_f64p), S.ctypes.data_as(_f64p),
                                   M, N, K, lda, ldb, max(N, 1),
                                   default_threads() if threads is None else int(threads),
                                   int(blocks[0]), int(blocks[1]), int(blocks[2]), int(in_dtype))
    if rc != 0:
        raise RuntimeError(f"oracle_gemm failed ({rc})")
    return C, S


def gemm_sampled(A, B, rows, cols, in_dtype: int = IN_BF16):
    """Dot products for the listed output elements: returns (c, s) float64."""
    A = _as_u16_2d(A, "A")
    B = _as_u16_2d(B, "B")
    M, K = A.shape
    _, N = B.shape
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    cols = np.ascontiguousarray(cols, dtype=np.int64)
    n = rows.shape[0]
    c = np.empty(n, dtype=np.float64)
    s = np.empty(n, dtype=np.float64)
    lda = max(A.strides[0] // 2 if M > 1 else K, K)
    ldb = max(B.strides[0] // 2 if K > 1 else N, N)
    rc = _load().oracle_gemm_sampled_typed(A.ctypes.data_as(_u16p), B.ctypes.data_as(_u16p),
                                           rows.ctypes.data_as(_i64p), cols.ctypes.data_as(_i64p), n,
                                           c.ctypes.data_as(_f64p), s.ctypes.data_as(_f64p),
                                           M, N, K, lda, ldb, int(in_dtype))
    if rc != 0:
        raise RuntimeError(f"oracle_gemm_sampled failed ({rc})")
    return c, s


def bf16_decode(bits):
    """uint16 bf16 bit patterns -> float64 values (exact)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    out = np.empty(bits.shape, dtype=np.float64)
    _load().oracle_bf16_decode_array(bits.ctypes.data_as(_u16p), out.ctypes.data_as(_f64p), bits.size)
    return out


def bf16_encode(x):
    """float32 -> uint16 bf16 bit patterns, round to nearest even."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, dtype=np.uint16)
    _load().oracle_bf16_encode_array(x.ctypes.data_as(_f32p), out.ctypes.data_as(_u16p), x.size)
    return out


def f16_decode(bits):
    """uint16 IEEE binary16 bit patterns -> float64 values (exact)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    out = np.empty(bits.shape, dtype=np.float64)
    _load().oracle_f16_decode_array(bits.ctypes.data_as(_u16p), out.ctypes.data_as(_f64p), bits.size)
    return out


def f16_encode(x):
    """float32 -> uint16 binary16 bit patterns, round to nearest even."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, dtype=np.uint16)
    _load().oracle_f16_encode_array(x.ctypes.data_as(_f32p), out.ctypes.data_as(_u16p), x.size)
    return out


def add_f32(x, y):
    """Listing 1: z_i = fl32(x_i + y_i) for two equal-length float32 vectors."""
    x = np.ascontiguousarray(x, dtype=np.float32).ravel()
    y = np.ascontiguousarray(y, dtype=np.float32).ravel()
    if x.shape != y.shape:
        raise ValueError("x and y differ in length")
    z = np.empty_like(x)
    _load().oracle_add_f32(x.ctypes.data_as(_f32p), y.ctypes.data_as(_f32p), z.ctypes.data_as(_f32p), x.size)
    return z


def silu(g):
    """silu(g) = g * sigmoid(g) = g / (1 + exp(-g)) in float64 (the SwiGLU gate activation of the
    Qwen3 MLP; the paper names the fused kernels around the projections,
    PAPER.md:343, without printing the formula -- DESIGN.md reading c21)."""
    g = np.asarray(g, dtype=np.float64)
    with np.errstate(over="ignore"):
        return g / (1.0 + np.exp(-g))


def swiglu_gemm(X, Wgu, threads: int | None = None):
    """Fused gate/up projection with the SwiGLU epilogue, stated step by step in float64:
        G = X @ Wgu[:, :I],  U = X @ Wgu[:, I:],  H = silu(G) * U,   I = Wgu.shape[1] // 2
    X: (M,K), Wgu: (K,2I) uint16 bf16 bit patterns ([gate | up] concatenated along N).
    Returns (H, G, U, Sg, Su): the result, both projections and their tolerance scales."""
    X = _as_u16_2d(X, "X")
    Wgu = _as_u16_2d(Wgu, "Wgu")
    if Wgu.shape[1] % 2:
        raise ValueError("the fused gate/up weight needs an even number of columns")
    inter = Wgu.shape[1] // 2
    G, Sg = gemm(X, Wgu[:, :inter], threads=threads)
    U, Su = gemm(X, Wgu[:, inter:], threads=threads)
    return silu(G) * U, G, U, Sg, Su


def word_sum_u32(buf) -> int:
    """Sum of a buffer's 32-bit words as an integer modulo 2^64 (what the read-bandwidth probe of
    the harness returns): the definition, through numpy's uint64 accumulation."""
    w = np.ascontiguousarray(buf).view(np.uint32).ravel()
    return int(np.sum(w, dtype=np.uint64))
