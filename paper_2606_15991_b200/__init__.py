"""paper_2606_15991_b200 -- B200-native BF16 GEMM / decode-GEMV hot path.

``tile_gemm`` and friends are thin ctypes bindings over the C-ABI library
``csrc/libtilegemm.so`` (declared in ``include/tile_gemm.h``).  Every step of
the path runs in hand-written sm_100a kernels; there is no CPU fallback and the
binding raises if the library is missing.  ``workloads`` holds the seeded
synthetic input generators (no method arithmetic).
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    # The binding is imported lazily so that `workloads` stays importable where
    # the CUDA library has not been built (e.g. the oracle's CPU tests).
    if name == "binding" or name.startswith("tile_gemm") or name in (
        "TileGemmError", "load_library", "PATH_NAMES", "OUT_F32", "OUT_BF16"):
        import importlib
        _b = importlib.import_module(__name__ + ".binding")
        return _b if name == "binding" else getattr(_b, name)
    raise AttributeError(name)
