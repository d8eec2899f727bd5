"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the CUDA path's tests/bench and by the oracle's tests.
It holds none of the method's arithmetic: it only draws random numbers, rounds
them to bf16 with torch's own cast (a library routine) and hands out bit
patterns.  The recipe:

  cfg 1  M=N=K=256, uniform integers in [-4,4], seed 0                (exact)
  cfg 2  M=1023 N=1537 K=769, A,B ~ N(0,1), seed 1                    (ragged)
  cfg 3  M=N=K=8192, A ~ N(0,1), B ~ N(0,1/K), seed 2                 (headline)
  cfg 4  M=4096, X ~ N(0,1), W ~ N(0,0.02^2), (K,N) in QWEN3_32B, seed 3
  cfg 5  M=1, same four (K,N), x ~ N(0,1), W ~ N(0,0.02^2), 64 layers, seed 4

The paper measures square f16 GEMMs and Qwen3-32B
inference; the Qwen3-32B projection *shapes* come from BASELINE.json and stand
in for Grout's linear layers with random weights (no checkpoint exists here).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

# (K, N) of the four Qwen3-32B projections, in BASELINE.json's order:
# fused QKV, attention output, fused gate/up, down.
QWEN3_32B = ((5120, 10240), (5120, 8192), (5120, 51200), (25600, 5120))
QWEN3_32B_NAMES = ("qkv", "attn_out", "gate_up", "down")
DECODE_LAYERS = 64


@dataclass(frozen=True)
class GemmCase:
    name: str
    M: int
    N: int
    K: int
    dist_a: str          # "int4" (uniform ints in [-4,4]) or "normal"
    sigma_a: float
    dist_b: str
    sigma_b: float
    out_dtype: str       # "f32" or "bf16"
    seed: tuple


CFG1 = GemmCase("cfg1_256_int", 256, 256, 256, "int4", 1.0, "int4", 1.0, "f32", (0,))
CFG2 = GemmCase("cfg2_ragged", 1023, 1537, 769, "normal", 1.0, "normal", 1.0, "f32", (1,))
CFG3 = GemmCase("cfg3_8192", 8192, 8192, 8192, "normal", 1.0, "normal", 8192 ** -0.5, "bf16", (2,))
CFG4 = tuple(
    GemmCase(f"cfg4_prefill_{nm}", 4096, n, k, "normal", 1.0, "normal", 0.02, "bf16", (3, p))
    for p, ((k, n), nm) in enumerate(zip(QWEN3_32B, QWEN3_32B_NAMES))
)


def cfg5_case(layer: int, proj: int) -> GemmCase:
    k, n = QWEN3_32B[proj]
    return GemmCase(f"cfg5_decode_l{layer}_{QWEN3_32B_NAMES[proj]}", 1, n, k,
                    "normal", 1.0, "normal", 0.02, "bf16", (4, layer, proj))


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 array -> uint16 bf16 bit patterns via torch's RNE cast."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16)


def bits_to_torch(bits: np.ndarray, device="cpu", dtype=torch.bfloat16) -> torch.Tensor:
    """uint16 bit patterns -> torch.bfloat16 (or torch.float16) tensor of the same shape."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(dtype)
    return t.to(device)


def f32_to_f16_bits(x: np.ndarray) -> np.ndarray:
    """float32 array -> uint16 IEEE binary16 bit patterns via numpy's RNE cast."""
    return np.ascontiguousarray(x, dtype=np.float32).astype(np.float16).view(np.uint16)


def make_inputs_f16(M, N, K, dist="normal", sigma_a=1.0, sigma_b=1.0, seed=0):
    """f16 twin of make_inputs_custom (the paper's GEMM sweep is in f16)."""
    rng = np.random.default_rng([int(seed), 7927])
    a = f32_to_f16_bits(_draw(rng, (M, K), dist, sigma_a))
    b = f32_to_f16_bits(_draw(rng, (K, N), dist, sigma_b))
    return a, b


def make_add_inputs(n: int, seed=0):
    """Element-wise add (Listing 1; the paper fills x and y with ones and measures at n = 2^28):
    seeded N(0,1) float32 vectors with every 16th element scaled by 2^+-20, so that sums round,
    cancel and absorb."""
    rng = np.random.default_rng([int(seed), 7933])
    x = rng.standard_normal(n, dtype=np.float32)
    y = rng.standard_normal(n, dtype=np.float32)
    x[::16] *= np.float32(2.0 ** 20)
    y[8::16] *= np.float32(2.0 ** -20)
    return x, y


def torch_to_bits(t: torch.Tensor) -> np.ndarray:
    """torch.bfloat16 tensor (any device) -> uint16 bit patterns on the host."""
    return t.detach().contiguous().cpu().view(torch.int16).numpy().view(np.uint16)


def _draw(rng: np.random.Generator, shape, dist: str, sigma: float) -> np.ndarray:
    if dist == "int4":
        return rng.integers(-4, 5, size=shape).astype(np.float32)
    if dist == "normal":
        return (rng.standard_normal(size=shape, dtype=np.float32) * np.float32(sigma))
    raise ValueError(dist)


def make_inputs(case: GemmCase):
    """Host-generated bf16 bit patterns (A: MxK, B: KxN) for a case."""
    rng = np.random.default_rng(list(case.seed))
    a = f32_to_bf16_bits(_draw(rng, (case.M, case.K), case.dist_a, case.sigma_a))
    b = f32_to_bf16_bits(_draw(rng, (case.K, case.N), case.dist_b, case.sigma_b))
    return a, b


def make_inputs_custom(M, N, K, dist="normal", sigma_a=1.0, sigma_b=1.0, seed=0):
    case = GemmCase("custom", M, N, K, dist, sigma_a, dist, sigma_b, "f32", (int(seed), 7919))
    return make_inputs(case)


def make_inputs_device(case: GemmCase, device="cuda"):
    """Device-generated inputs for shapes too large for a host RNG pass
    (cfg 5: 31.2 G weights).  Same seeded torch generator for both the CUDA
    path and, after a read-back, the oracle: inputs are shared, code is not."""
    g = torch.Generator(device=device)
    g.manual_seed(int(np.random.SeedSequence(list(case.seed)).generate_state(1)[0]))
    a = torch.empty((case.M, case.K), dtype=torch.bfloat16, device=device)
    b = torch.empty((case.K, case.N), dtype=torch.bfloat16, device=device)
    if case.dist_a != "normal" or case.dist_b != "normal":
        raise ValueError("device generation is only used for the normal cases")
    a.normal_(0.0, case.sigma_a, generator=g)
    b.normal_(0.0, case.sigma_b, generator=g)
    return a, b


def make_int_inputs_device(M, N, K, seed=0, device="cuda", dtype=torch.bfloat16):
    """Device-generated integer-valued inputs, uniform in [-4, 4] like "int4", for shapes whose host
    generation would take longer than the test (weights of the decode shapes, the 32768^3 sweep point)."""
    g = torch.Generator(device=device)
    g.manual_seed(int(np.random.SeedSequence([int(seed), 7933]).generate_state(1)[0]))
    a = torch.randint(-4, 5, (M, K), generator=g, device=device, dtype=torch.int8).to(dtype)
    b = torch.randint(-4, 5, (K, N), generator=g, device=device, dtype=torch.int8).to(dtype)
    return a, b


def stratified_samples(M: int, N: int, block=128, seed: int = 0):
    """One seeded-uniform element inside every block x block cell of the output
    (SURVEY.md 8(c) c13): every output tile is touched.  `block` may be a
    (rows, columns) pair for rectangular cells.  Returns (rows, cols)."""
    rng = np.random.default_rng([int(seed), 104729])
    block_m, block_n = (block, block) if isinstance(block, int) else block
    bi = np.arange(0, M, block_m)
    bj = np.arange(0, N, block_n)
    ii, jj = np.meshgrid(bi, bj, indexing="ij")
    hi_i = np.minimum(ii + block_m, M) - ii
    hi_j = np.minimum(jj + block_n, N) - jj
    rows = ii + (rng.random(ii.shape) * hi_i).astype(np.int64)
    cols = jj + (rng.random(jj.shape) * hi_j).astype(np.int64)
    return rows.ravel().astype(np.int64), cols.ravel().astype(np.int64)


def uniform_samples(M: int, N: int, n: int, seed: int = 0):
    """n seeded-uniform output elements plus the four corners and a run along
    the last row / last column (edge tiles)."""
    rng = np.random.default_rng([int(seed), 1299709])
    rows = rng.integers(0, M, size=n)
    cols = rng.integers(0, N, size=n)
    er = np.array([0, 0, M - 1, M - 1] + [M - 1] * 8 + list(rng.integers(0, M, size=8)))
    ec = np.array([0, N - 1, 0, N - 1] + list(rng.integers(0, N, size=8)) + [N - 1] * 8)
    return (np.concatenate([rows, er]).astype(np.int64),
            np.concatenate([cols, ec]).astype(np.int64))
