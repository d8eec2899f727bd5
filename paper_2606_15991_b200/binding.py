"""ctypes binding of libtilegemm.so (include/tile_gemm.h, include/tile_gemm_debug.h) -- argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  There is no CPU
fallback: if the shared library cannot be found or built, ``load_library``
raises, and on a machine without an sm_100 device every compute entry returns
``TILE_GEMM_E_DEVICE`` which is raised as ``TileGemmError``.
"""
from __future__ import annotations

import contextlib
import ctypes
import os

import torch

from . import build as _build

OUT_F32 = 0
OUT_BF16 = 1
OUT_F16 = 2
IN_BF16 = 0
IN_F16 = 1

PATH_AUTO, PATH_GEMM_TMA, PATH_GEMM_REPACK, PATH_GEMV, PATH_ZERO, PATH_NOOP = range(6)
PATH_NAMES = {PATH_AUTO: "auto", PATH_GEMM_TMA: "gemm_tma", PATH_GEMM_REPACK: "gemm_repack",
              PATH_GEMV: "gemv", PATH_ZERO: "zero", PATH_NOOP: "noop"}

(E_OK, E_NULL, E_EXTENT, E_LDA, E_LDB, E_LDC, E_DTYPE, E_ALIGN, E_ALIAS, E_OVERFLOW, E_DEVICE,
 E_CUDA, E_PATH, E_INTERNAL, E_IN_DTYPE, E_LIMIT) = range(16)

(TUNE_GEMM_CONFIG, TUNE_GEMM_GROUP_M, TUNE_GEMM_MAX_CTAS, TUNE_GEMV_SPLIT, TUNE_GEMV_VARIANT, TUNE_GEMV_SHAPE, TUNE_FLAGS,
 TUNE_ADD_SHAPE, TUNE_GEMV_FIXUP, TUNE_GEMV_L2_POST, TUNE_GEMV_CLUSTER_MARGIN, TUNE_SKINNY, TUNE_GEMM_MULTICAST) = range(13)
NUM_TUNE_KEYS = 16

NO_ALLOC_MAX_N = 262144           # TILE_GEMV_NO_ALLOC_MAX_N
NO_ALLOC_MAX_TILES = 1024         # TILE_GEMV_NO_ALLOC_MAX_TILES
NO_ALLOC_SCRATCH_BYTES = 1052672  # TILE_GEMV_NO_ALLOC_SCRATCH_BYTES

EXPORTS = ("tile_gemm", "tile_gemm_ex", "tile_gemm_static_b", "tile_gemm_typed", "tile_gemm_swiglu", "tile_add_f32", "tile_read_probe_u32",
           "tile_gemv_no_alloc",
           "tile_gemm_record_begin", "tile_gemm_record_end", "tile_gemm_replay", "tile_gemm_recorded_nodes",
           "tile_gemm_record_free", "tile_gemm_select", "tile_gemm_host",
           "tile_gemm_debug_owner_map", "tile_gemm_debug_trace", "tile_gemm_debug_occupy", "tile_gemm_query_config", "tile_gemm_query_plan", "tile_gemm_set_tuning",
           "tile_gemm_launch_count", "tile_gemm_status_string", "tile_gemm_last_error",
           "tile_gemm_shutdown")

_lib = None
_NULL_CTX = contextlib.nullcontext()
_i64 = ctypes.c_int64
_vp = ctypes.c_void_p
_int = ctypes.c_int


class TileGemmError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"tile_gemm status {status}: {message}")
        self.status = status
        self.message = message


def library_path() -> str:
    return _build.LIB


def load_library():
    """Loads csrc/libtilegemm.so, building it first when it is missing or older than its sources.
    A rebuild that is needed and fails raises: a stale library is never loaded silently
    (TILEGEMM_NO_REBUILD=1 skips the staleness check for a deployed, prebuilt library)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    stale_check = os.environ.get("TILEGEMM_NO_REBUILD", "0") != "1"
    if not os.path.exists(path) or (stale_check and _build.needs_build()):
        why = "is missing" if not os.path.exists(path) else "is older than its sources"
        try:
            _build.build()
        except Exception as exc:
            raise RuntimeError(f"libtilegemm.so {why} and could not be built ({exc}); "
                               "the CUDA path has no fallback") from exc
    lib = ctypes.CDLL(path)
    g = [_vp, _vp, _vp, _i64, _i64, _i64, _i64, _i64, _i64, _int]
    lib.tile_gemm.argtypes = g + [_vp]
    lib.tile_gemm.restype = _int
    lib.tile_gemm_ex.argtypes = g + [_vp, _int]
    lib.tile_gemm_ex.restype = _int
    lib.tile_gemm_static_b.argtypes = g + [_vp]
    lib.tile_gemm_static_b.restype = _int
    lib.tile_gemm_typed.argtypes = g[:-1] + [_int, _int, _vp]
    lib.tile_gemm_typed.restype = _int
    lib.tile_gemm_swiglu.argtypes = g + [_vp]
    lib.tile_gemm_swiglu.restype = _int
    lib.tile_gemv_no_alloc.argtypes = [_vp, _vp, _vp, _i64, _i64, _i64, _int, _int, _int, _vp]
    lib.tile_gemv_no_alloc.restype = _int
    lib.tile_read_probe_u32.argtypes = [_vp, _i64, _vp, _vp]
    lib.tile_read_probe_u32.restype = _int
    lib.tile_add_f32.argtypes = [_vp, _vp, _vp, _i64, _vp]
    lib.tile_add_f32.restype = _int
    lib.tile_gemm_record_begin.argtypes = [_vp]
    lib.tile_gemm_record_begin.restype = _int
    lib.tile_gemm_record_end.argtypes = [_vp, ctypes.POINTER(_vp)]
    lib.tile_gemm_record_end.restype = _int
    lib.tile_gemm_replay.argtypes = [_vp, _vp]
    lib.tile_gemm_replay.restype = _int
    lib.tile_gemm_recorded_nodes.argtypes = [_vp]
    lib.tile_gemm_recorded_nodes.restype = _i64
    lib.tile_gemm_record_free.argtypes = [_vp]
    lib.tile_gemm_record_free.restype = _int
    lib.tile_gemm_select.argtypes = [_i64] * 6 + [_vp, _vp, _vp, _int]
    lib.tile_gemm_select.restype = _int
    lib.tile_gemm_host.argtypes = g
    lib.tile_gemm_host.restype = _int
    lib.tile_gemm_debug_owner_map.argtypes = [_vp, _i64, _i64, _i64, _i64, _int, _vp]
    lib.tile_gemm_debug_owner_map.restype = _int
    lib.tile_gemm_debug_occupy.argtypes = [_int, _i64, _vp]
    lib.tile_gemm_debug_occupy.restype = _int
    lib.tile_gemm_debug_trace.argtypes = [_vp, _i64]
    lib.tile_gemm_debug_trace.restype = _int
    lib.tile_gemm_query_config.argtypes = [_i64, _i64, _i64, _int, ctypes.POINTER(ctypes.c_int32)]
    lib.tile_gemm_query_config.restype = _int
    lib.tile_gemm_query_plan.argtypes = [_i64, _i64, _i64, ctypes.POINTER(ctypes.c_int32)]
    lib.tile_gemm_query_plan.restype = _int
    lib.tile_gemm_set_tuning.argtypes = [_int, _int]
    lib.tile_gemm_set_tuning.restype = _int
    lib.tile_gemm_launch_count.argtypes = []
    lib.tile_gemm_launch_count.restype = _i64
    lib.tile_gemm_status_string.argtypes = [_int]
    lib.tile_gemm_status_string.restype = ctypes.c_char_p
    lib.tile_gemm_last_error.argtypes = []
    lib.tile_gemm_last_error.restype = ctypes.c_char_p
    lib.tile_gemm_shutdown.argtypes = []
    lib.tile_gemm_shutdown.restype = _int
    _lib = lib
    return lib


def _check(status: int):
    if status != 0:
        raise TileGemmError(status, tile_gemm_last_error())


def _stream_handle(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _on_device(*tensors):
    """All tensors must live on one CUDA device; the call then runs with that device current
    (the library launches on the current device and dereferences raw pointers)."""
    dev = tensors[0].device
    for t in tensors:
        if not t.is_cuda:
            raise TypeError("expected CUDA tensors (tile_gemm_host takes host buffers)")
        if t.device != dev:
            raise ValueError(f"operands live on different devices: {dev} and {t.device}")
    if dev.index is None or dev.index == torch.cuda.current_device():
        return _NULL_CTX
    return torch.cuda.device(dev)


def _ld(t: torch.Tensor) -> int:
    if t.dim() != 2 or (t.shape[1] > 1 and t.stride(1) != 1):
        raise ValueError("expected a 2-D row-major tensor (unit column stride)")
    return int(t.stride(0)) if t.shape[0] > 1 else max(int(t.stride(0)), int(t.shape[1]), 1)


def tile_gemm_status_string(status: int) -> str:
    return load_library().tile_gemm_status_string(int(status)).decode()


def tile_gemm_last_error() -> str:
    return load_library().tile_gemm_last_error().decode()


def tile_gemm_launch_count() -> int:
    return int(load_library().tile_gemm_launch_count())


def tile_gemm_set_tuning(key: int, value: int) -> None:
    _check(load_library().tile_gemm_set_tuning(int(key), int(value)))


def tile_gemm_shutdown() -> None:
    _check(load_library().tile_gemm_shutdown())


def tile_gemm_raw(A: int, B: int, C: int, M, N, K, lda, ldb, ldc, out_dtype, stream: int = 0,
                  force_path: int = PATH_AUTO) -> int:
    """Raw pointer form; returns the status code instead of raising."""
    return int(load_library().tile_gemm_ex(_vp(A), _vp(B), _vp(C), M, N, K, lda, ldb, ldc,
                                           int(out_dtype), _vp(stream), int(force_path)))


def tile_gemm_select(M, N, K, lda, ldb, ldc, A: int = 256, B: int = 1 << 40, C: int = 1 << 41,
                     out_dtype: int = OUT_F32) -> int:
    """Pure host: path id (> 0) or the negated status of the failing precondition."""
    return int(load_library().tile_gemm_select(M, N, K, lda, ldb, ldc, _vp(A), _vp(B), _vp(C), int(out_dtype)))


def tile_gemm(A: torch.Tensor, B: torch.Tensor, C: torch.Tensor | None = None, out_dtype=None,
              stream=None, force_path: int = PATH_AUTO, static_b: bool = False) -> torch.Tensor:
    """C = A @ B on the current CUDA device.  A: (M,K), B: (K,N), both bf16 or both f16, row-major
    (any row stride); C: (M,N) fp32, bf16 or f16, allocated if None.  Asynchronous on `stream`.
    bf16 inputs with fp32/bf16 output go through tile_gemm_ex / tile_gemm_static_b, anything
    involving f16 through tile_gemm_typed.
    static_b=True calls tile_gemm_static_b (B holds weights nobody in flight writes)."""
    if A.dtype != B.dtype or A.dtype not in (torch.bfloat16, torch.float16):
        raise TypeError("A and B must both be torch.bfloat16 or both torch.float16")
    M, K = A.shape
    K2, N = B.shape
    if K != K2:
        raise ValueError("inner dimensions differ")
    if C is None:
        dt = (torch.float32 if out_dtype in (None, OUT_F32, torch.float32)
              else torch.float16 if out_dtype in (OUT_F16, torch.float16) else torch.bfloat16)
        C = torch.empty((M, N), dtype=dt, device=A.device)
    if C.dtype not in (torch.float32, torch.bfloat16, torch.float16) or tuple(C.shape) != (M, N):
        raise TypeError("C must be an (M,N) float32, bfloat16 or float16 tensor")
    od = {torch.float32: OUT_F32, torch.bfloat16: OUT_BF16, torch.float16: OUT_F16}[C.dtype]
    with _on_device(A, B, C):
        st = _tile_gemm_call(A, B, C, M, N, K, od, stream, force_path, static_b)
    _check(st)
    return C


def _tile_gemm_call(A, B, C, M, N, K, od, stream, force_path, static_b) -> int:
    if A.dtype == torch.float16 or od == OUT_F16:
        if static_b or force_path != PATH_AUTO:
            raise ValueError("static_b / force_path apply to the bf16 entries only")
        st = load_library().tile_gemm_typed(_vp(A.data_ptr()), _vp(B.data_ptr()), _vp(C.data_ptr()), M, N, K,
                                            _ld(A), _ld(B), _ld(C), IN_F16 if A.dtype == torch.float16 else IN_BF16,
                                            od, _vp(_stream_handle(stream)))
    elif static_b:
        if force_path != PATH_AUTO:
            raise ValueError("static_b cannot be combined with force_path")
        st = load_library().tile_gemm_static_b(_vp(A.data_ptr()), _vp(B.data_ptr()), _vp(C.data_ptr()), M, N, K,
                                               _ld(A), _ld(B), _ld(C), od, _vp(_stream_handle(stream)))
    else:
        st = load_library().tile_gemm_ex(_vp(A.data_ptr()), _vp(B.data_ptr()), _vp(C.data_ptr()), M, N, K,
                                         _ld(A), _ld(B), _ld(C), od, _vp(_stream_handle(stream)),
                                         int(force_path))
    return int(st)


def tile_gemm_typed_raw(A: int, B: int, C: int, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, stream: int = 0) -> int:
    """Raw pointer form of tile_gemm_typed; returns the status code instead of raising."""
    return int(load_library().tile_gemm_typed(_vp(A), _vp(B), _vp(C), M, N, K, lda, ldb, ldc, int(in_dtype),
                                              int(out_dtype), _vp(stream)))


def tile_gemm_swiglu_raw(X: int, W: int, H: int, M, I, K, ldx, ldw, ldh, out_dtype, stream: int = 0) -> int:
    return int(load_library().tile_gemm_swiglu(_vp(X), _vp(W), _vp(H), M, I, K, ldx, ldw, ldh, int(out_dtype), _vp(stream)))


def tile_gemm_swiglu(X: torch.Tensor, Wgu: torch.Tensor, H: torch.Tensor | None = None, out_dtype=None,
                     stream=None) -> torch.Tensor:
    """H = silu(X @ Wgu[:, :I]) * (X @ Wgu[:, I:]) with I = Wgu.shape[1] // 2; X, Wgu bf16; H fp32, bf16 or f16."""
    if X.dtype != torch.bfloat16 or Wgu.dtype != torch.bfloat16:
        raise TypeError("X and Wgu must be torch.bfloat16")
    M, K = X.shape
    K2, N2 = Wgu.shape
    if K != K2 or N2 % 2:
        raise ValueError("Wgu must be (K, 2*I)")
    inter = N2 // 2
    if H is None:
        dt = (torch.float32 if out_dtype in (OUT_F32, torch.float32)
              else torch.float16 if out_dtype in (OUT_F16, torch.float16) else torch.bfloat16)
        H = torch.empty((M, inter), dtype=dt, device=X.device)
    if tuple(H.shape) != (M, inter):
        raise TypeError("H must be (M, I)")
    if H.dtype not in (torch.float32, torch.bfloat16, torch.float16):
        raise TypeError("H must be float32, bfloat16 or float16")
    od = {torch.float32: OUT_F32, torch.bfloat16: OUT_BF16, torch.float16: OUT_F16}[H.dtype]
    with _on_device(X, Wgu, H):
        st = load_library().tile_gemm_swiglu(_vp(X.data_ptr()), _vp(Wgu.data_ptr()), _vp(H.data_ptr()), M, inter, K,
                                             _ld(X), _ld(Wgu), _ld(H), od, _vp(_stream_handle(stream)))
    _check(st)
    return H


def tile_gemv_no_alloc_raw(x: int, B: int, y: int, N, K, ldb, in_dtype, out_dtype, split: int = 0, stream: int = 0) -> int:
    """Raw pointer form of tile_gemv_no_alloc; returns the status code instead of raising."""
    return int(load_library().tile_gemv_no_alloc(_vp(x), _vp(B), _vp(y), N, K, ldb, int(in_dtype), int(out_dtype),
                                                 int(split), _vp(stream)))


def tile_gemv_no_alloc(x: torch.Tensor, B: torch.Tensor, y: torch.Tensor, split: int = 0, stream=None) -> torch.Tensor:
    """y = x @ B for one activation row, through the entry point that allocates no device memory.

    For programs that cannot call cudaMalloc once they are running -- a server whose own pool already
    holds all of HBM, a host that forbids allocations after start-up, a decode loop that cannot absorb
    cudaMalloc's device-wide synchronisation.  The kernel's split-K scratch is a fixed array inside the
    library (NO_ALLOC_SCRATCH_BYTES per GPU, shared by every call on that GPU), so the caller supplies
    all three tensors, `y` included: this wrapper creates none.

    x: (K,) or (1, K); B: (K, N) row-major with a 16-byte aligned base and a row stride that is a
    multiple of 8 elements; x and B both bf16 or both f16; y: (N,) or (1, N) float32, bfloat16 or
    float16.  split = 0 lets the library choose the number of K slices.  Raises TileGemmError with
    status E_LIMIT when N > NO_ALLOC_MAX_N or ceil(N / 256) * slices > NO_ALLOC_MAX_TILES.
    Calls on one stream may follow each other freely; calls that could run at the same time on one GPU
    (unordered streams) race on the shared scratch.  The first call on a device does the one-time
    set-up and should come before any stream capture."""
    if x.dtype != B.dtype or x.dtype not in (torch.bfloat16, torch.float16):
        raise TypeError("x and B must both be torch.bfloat16 or both torch.float16")
    if B.dim() != 2 or x.numel() != B.shape[0] or x.dim() > 2 or (x.dim() == 2 and x.shape[0] != 1):
        raise ValueError("x must hold K elements ((K,) or (1, K)) for B of shape (K, N)")
    K, N = B.shape
    if y.dtype not in (torch.float32, torch.bfloat16, torch.float16) or y.numel() != N or y.dim() > 2 \
            or (y.dim() == 2 and y.shape[0] != 1):
        raise TypeError("y must be an (N,) or (1, N) float32, bfloat16 or float16 tensor")
    if (x.numel() > 1 and x.stride(-1) != 1) or (y.numel() > 1 and y.stride(-1) != 1):
        raise ValueError("x and y must have unit element stride")
    od = {torch.float32: OUT_F32, torch.bfloat16: OUT_BF16, torch.float16: OUT_F16}[y.dtype]
    with _on_device(x, B, y):
        st = load_library().tile_gemv_no_alloc(_vp(x.data_ptr()), _vp(B.data_ptr()), _vp(y.data_ptr()), N, K, _ld(B),
                                               IN_F16 if x.dtype == torch.float16 else IN_BF16, od, int(split),
                                               _vp(_stream_handle(stream)))
    _check(int(st))
    return y


def tile_read_probe_u32(buf: torch.Tensor, out_sum: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """Adds the sum of buf's 32-bit words (mod 2^64) to out_sum (a 1-element int64 tensor, created zeroed if None)."""
    if buf.element_size() * buf.numel() % 4 or not buf.is_contiguous():
        raise ValueError("buf must be contiguous and a whole number of 32-bit words")
    if out_sum is None:
        out_sum = torch.zeros(1, dtype=torch.int64, device=buf.device)
    with _on_device(buf, out_sum):
        st = load_library().tile_read_probe_u32(_vp(buf.data_ptr()), buf.element_size() * buf.numel() // 4,
                                                _vp(out_sum.data_ptr()), _vp(_stream_handle(stream)))
    _check(st)
    return out_sum


def tile_add_f32_raw(x: int, y: int, z: int, n: int, stream: int = 0) -> int:
    return int(load_library().tile_add_f32(_vp(x), _vp(y), _vp(z), int(n), _vp(stream)))


def tile_add_f32(x: torch.Tensor, y: torch.Tensor, z: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """z = x + y over contiguous float32 vectors on the current CUDA device (Listing 1)."""
    if x.dtype != torch.float32 or y.dtype != torch.float32 or x.numel() != y.numel():
        raise TypeError("x and y must be float32 tensors of equal length")
    if not (x.is_contiguous() and y.is_contiguous()):
        raise ValueError("x and y must be contiguous")
    if z is None:
        z = torch.empty_like(x)
    if z.dtype != torch.float32 or z.numel() != x.numel() or not z.is_contiguous():
        raise TypeError("z must be a contiguous float32 tensor of the same length")
    with _on_device(x, y, z):
        st = load_library().tile_add_f32(_vp(x.data_ptr()), _vp(y.data_ptr()), _vp(z.data_ptr()), x.numel(),
                                         _vp(_stream_handle(stream)))
    _check(st)
    return z


class RecordedStep:
    """A recorded sequence of library calls (tile_gemm_record_begin/_end), replayed with one driver call."""

    def __init__(self, handle: int):
        self.handle = handle

    @property
    def nodes(self) -> int:
        return int(load_library().tile_gemm_recorded_nodes(_vp(self.handle)))

    def replay(self, stream=None) -> None:
        _check(load_library().tile_gemm_replay(_vp(self.handle), _vp(_stream_handle(stream))))

    def free(self) -> None:
        if self.handle:
            _check(load_library().tile_gemm_record_free(_vp(self.handle)))
            self.handle = 0


def tile_gemm_record_begin(stream) -> None:
    _check(load_library().tile_gemm_record_begin(_vp(_stream_handle(stream))))


def tile_gemm_record_end(stream) -> RecordedStep:
    out = _vp()
    _check(load_library().tile_gemm_record_end(_vp(_stream_handle(stream)), ctypes.byref(out)))
    return RecordedStep(int(out.value))


def tile_gemm_host(A_bits, B_bits, C_out, lda=None, ldb=None, ldc=None):
    """End-to-end on HOST numpy arrays: A_bits (M,K) uint16, B_bits (K,N) uint16 bf16 patterns,
    C_out (M,N) float32 or uint16 (bf16 patterns), all C-contiguous rows."""
    import numpy as np
    if A_bits.dtype != np.uint16 or B_bits.dtype != np.uint16:
        raise TypeError("A_bits and B_bits must be uint16 arrays of bf16 bit patterns")
    if C_out.dtype not in (np.float32, np.uint16):
        raise TypeError("C_out must be float32 or uint16 (bf16 bit patterns)")
    for arr in (A_bits, B_bits, C_out):
        if arr.ndim != 2 or (arr.shape[1] > 1 and arr.strides[1] != arr.itemsize):
            raise ValueError("expected 2-D arrays with contiguous rows")
    M, K = A_bits.shape
    K2, N = B_bits.shape
    if K2 != K or C_out.shape != (M, N):
        raise ValueError("shapes do not form C (M,N) = A (M,K) @ B (K,N)")
    od = OUT_F32 if C_out.dtype == np.float32 else OUT_BF16
    lda = lda or max(A_bits.strides[0] // 2, K, 1)
    ldb = ldb or max(B_bits.strides[0] // 2, N, 1)
    ldc = ldc or max(C_out.strides[0] // C_out.itemsize, N, 1)
    st = load_library().tile_gemm_host(_vp(A_bits.ctypes.data), _vp(B_bits.ctypes.data), _vp(C_out.ctypes.data),
                                       M, N, K, lda, ldb, ldc, od)
    _check(st)
    return C_out


def tile_gemm_host_raw(A: int, B: int, C: int, M, N, K, lda, ldb, ldc, out_dtype) -> int:
    return int(load_library().tile_gemm_host(_vp(A), _vp(B), _vp(C), M, N, K, lda, ldb, ldc, int(out_dtype)))


def tile_gemm_query_config(M, N, K, out_dtype=OUT_F32) -> dict:
    out = (ctypes.c_int32 * 8)()
    _check(load_library().tile_gemm_query_config(M, N, K, int(out_dtype), out))
    return {"BM": out[0], "BN": out[1], "cta_group": out[2], "ctas": out[3], "group_m": out[4],
            "stages": out[5], "BK": out[6], "config": out[7]}


def tile_gemm_query_plan(M, N, K) -> dict:
    out = (ctypes.c_int32 * 8)()
    _check(load_library().tile_gemm_query_plan(M, N, K, out))
    return {"config": out[0], "ctas": out[1], "full_units": out[2], "split": out[3], "k_tiles_per_slice": out[4],
            "lockstep_rounds": out[5], "lockstep_window": out[6], "a_box_rows": out[7]}


def tile_gemm_debug_occupy(ctas: int, ns: int, stream=None) -> None:
    """`ctas` CTAs holding one SM each for `ns` nanoseconds on `stream` (test helper)."""
    _check(load_library().tile_gemm_debug_occupy(int(ctas), int(ns), _vp(_stream_handle(stream))))


_trace_ref = None   # the tensor the library currently holds a raw pointer to (tile_gemm_debug_trace)


def tile_gemm_debug_trace(records: torch.Tensor | None) -> None:
    """records: int64 CUDA tensor of shape (capacity, 8) that the following M = 1 and tiled-GEMM launches fill,
    or None to stop.  The library keeps only the raw device pointer, so this module keeps the tensor alive
    until tracing is switched off (or another buffer is set); launches made while a stream is recording or
    capturing get no trace pointer."""
    global _trace_ref
    if records is None:
        _check(load_library().tile_gemm_debug_trace(_vp(0), 0))
        _trace_ref = None
        return
    if records.dtype != torch.int64 or records.dim() != 2 or records.shape[1] != 8 or not records.is_contiguous():
        raise TypeError("records must be a contiguous int64 tensor of shape (capacity, 8)")
    _check(load_library().tile_gemm_debug_trace(_vp(records.data_ptr()), records.shape[0]))
    _trace_ref = records


def tile_gemm_debug_owner_map(M, N, K, out_dtype=OUT_F32, ld_owner=None, stream=None, device="cuda"):
    ld = int(ld_owner or N)
    owner = torch.full((M, ld), -1, dtype=torch.int32, device=device)
    _check(load_library().tile_gemm_debug_owner_map(_vp(owner.data_ptr()), M, N, K, ld, int(out_dtype),
                                                    _vp(_stream_handle(stream))))
    return owner
