"""Builds csrc/libtilegemm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libtilegemm.so")
SOURCES = ["tile_gemm.cu"]
HEADERS = ["ptx.cuh", "gemm_kernel.cuh", "gemv_kernel.cuh", "skinny_kernel.cuh", "aux_kernels.cuh", "add_kernel.cuh",
           os.path.join("..", "..", "include", "tile_gemm.h"), os.path.join("..", "..", "include", "tile_gemm_debug.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",           # the .so must load where libcuda / libcudart are absent
    "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _defines() -> list:
    """TILEGEMM_WATCHDOG=0 in the environment builds without the bounded-wait watchdog (csrc/ptx.cuh: every
    mbarrier wait then spins without the %globaltimer check, printf and trap).  The default build keeps it:
    measured cost on B200 see DESIGN.md "Watchdog"."""
    wd = os.environ.get("TILEGEMM_WATCHDOG")
    return [f"-DTILEGEMM_WATCHDOG={int(wd)}"] if wd not in (None, "") else []


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + _defines() + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libtilegemm.so")
    with open(os.path.join(CSRC, "ptxas_report.txt"), "w") as f:
        f.write("$ " + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
