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

// Read-bandwidth probe ("a read-only streaming probe kernel ... to establish this
// box's achievable read bandwidth"): *out += sum of n 32-bit words as a 64-bit integer (exact, order
// independent).  One 32 KB tile per CTA, eight 16-byte loads in flight per thread (the shape of the
// fastest stand-alone probe: 7.5 TB/s on B200), one atomic per CTA; the words past the last full
// vector are added by the last CTA.
constexpr int PROBE_THREADS = 256, PROBE_UNROLL = 8;
__global__ void __launch_bounds__(PROBE_THREADS)
read_probe_kernel(const uint32_t* __restrict__ buf, int64_t n, unsigned long long* out) {
    __shared__ unsigned long long warp_sums[PROBE_THREADS / 32];
    const int64_t nvec = n >> 2;
    const uint4* v4 = reinterpret_cast<const uint4*>(buf);
    const int64_t base = (int64_t)blockIdx.x * (PROBE_THREADS * PROBE_UNROLL) + threadIdx.x;
    uint4 a[PROBE_UNROLL];
#pragma unroll
    for (int u = 0; u < PROBE_UNROLL; ++u) {
        a[u] = make_uint4(0, 0, 0, 0);
        if (base + u * PROBE_THREADS < nvec)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(a[u].x), "=r"(a[u].y), "=r"(a[u].z), "=r"(a[u].w)
                         : "l"(v4 + base + u * PROBE_THREADS));
    }
    unsigned long long s = 0;
#pragma unroll
    for (int u = 0; u < PROBE_UNROLL; ++u) s += (unsigned long long)a[u].x + a[u].y + a[u].z + a[u].w;
    if (blockIdx.x == gridDim.x - 1) {
        const int64_t e = (nvec << 2) + threadIdx.x;
        if (e < n) s += __ldg(buf + e);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
#pragma unroll
        for (int w = 0; w < PROBE_THREADS / 32; ++w) t += warp_sums[w];
        if (t) atomicAdd(out, t);
    }
}

// tile_gemm_debug_occupy: each CTA holds one SM (the launch asks for most of its shared memory) until
// `ns` nanoseconds have passed.  It waits for nothing but the clock.
__global__ void __launch_bounds__(128)
occupy_kernel(unsigned long long ns) {
    const unsigned long long t0 = global_timer_ns();
    while (global_timer_ns() - t0 < ns) __nanosleep(1000);
}

}  // namespace tg
