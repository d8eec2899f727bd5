// Small helper kernels of the GEMM path: operand repack (rows that TMA cannot address are
// copied into 16-byte aligned rows) and the K == 0 zero fill.
#pragma once
#include <stdint.h>

namespace tg {

// dst[r][c] = src[r][c] for c < cols, 0 for cols <= c < ld_dst.  ld_dst is a multiple of 8 and
// dst is 16-byte aligned, so every thread writes one 16-byte chunk; src has no alignment beyond 2.
__global__ void __launch_bounds__(256)
repack_rows_kernel(const uint16_t* __restrict__ src, int64_t ld_src, uint16_t* __restrict__ dst, int64_t ld_dst,
                   int64_t rows, int64_t cols) {
    const int64_t chunks_per_row = ld_dst >> 3;
    const int64_t total = rows * chunks_per_row;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / chunks_per_row;
        const int64_t c0 = (i - r * chunks_per_row) << 3;
        const uint16_t* s = src + r * ld_src + c0;
        uint32_t h[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) h[e] = (c0 + e < cols) ? (uint32_t)__ldg(s + e) : 0u;
        uint4 w;
        w.x = h[0] | (h[1] << 16);
        w.y = h[2] | (h[3] << 16);
        w.z = h[4] | (h[5] << 16);
        w.w = h[6] | (h[7] << 16);
        *reinterpret_cast<uint4*>(dst + r * ld_dst + c0) = w;
    }
}

// C[0..M) x [0..N) <- 0 (K == 0, reading c8).  esize is 2 or 4; C is element aligned only.
__global__ void __launch_bounds__(256)
zero_fill_kernel(void* C, int64_t M, int64_t N, int64_t ldc, int esize) {
    const int64_t total = M * N;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / N, c = i - r * N;
        if (esize == 2) reinterpret_cast<uint16_t*>(C)[r * ldc + c] = 0;
        else reinterpret_cast<uint32_t*>(C)[r * ldc + c] = 0u;
    }
}

}  // namespace tg
