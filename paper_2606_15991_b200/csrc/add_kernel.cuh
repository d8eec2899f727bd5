// Element-wise add for sm_100a:  z_i = fl32(x_i + y_i)  over f32 vectors.
//
// What it computes: Listing 1 of the paper -- every tile program loads the
// tiles of x and y that line up with its exclusively owned sub-tensor of z, adds them and
// stores the sum; the paper measures it at n = 2^28 (6.97 TB/s on its B200,
// PAPER.md:306).  12 bytes of HBM traffic per element and one FADD: purely bandwidth bound, so
// the only jobs are to keep enough bytes in flight per SM and to waste none.
//
//   * a "tile" here is ADD_THREADS * UNROLL 16-byte vectors (e.g. 256 * 4 * 4 = 4096 elements);
//     tile t is owned by exactly one CTA (t = blockIdx.x, + gridDim.x, ...), the same
//     one-owner-per-sub-tensor contract as Listing 1's `.partition([128])`;
//   * every thread issues all 2 * UNROLL 16-byte loads of its tile before the first add
//     (2 * UNROLL * 16 B in flight per thread), streaming hints on loads and stores;
//   * bounds: full tiles run with no predicate at all; the single ragged tile and the < 4
//     element tail are handled once, after the loop (the paper's "masked stores" for the edge
//     tile, with the check hoisted out of the hot loop).
#pragma once
#include <stdint.h>

namespace tg {

constexpr int ADD_THREADS = 256;

__device__ __forceinline__ float4 ld_stream_f4(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream_f4(float4* p, const float4& v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
                 : "memory");
}

// x, y, z 16-byte aligned.  nvec = n / 4 full vectors; the n % 4 tail elements follow them.
template <int UNROLL>
__global__ void __launch_bounds__(ADD_THREADS)
add_f32_vec_kernel(const float* __restrict__ x, const float* __restrict__ y, float* __restrict__ z, int64_t n) {
    constexpr int64_t TILE_VECS = (int64_t)ADD_THREADS * UNROLL;
    const float4* x4 = reinterpret_cast<const float4*>(x);
    const float4* y4 = reinterpret_cast<const float4*>(y);
    float4* z4 = reinterpret_cast<float4*>(z);
    const int64_t nvec = n >> 2;
    const int64_t full_tiles = nvec / TILE_VECS;
    for (int64_t t = blockIdx.x; t < full_tiles; t += gridDim.x) {
        const int64_t base = t * TILE_VECS + threadIdx.x;
        float4 a[UNROLL], b[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) a[u] = ld_stream_f4(x4 + base + u * ADD_THREADS);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) b[u] = ld_stream_f4(y4 + base + u * ADD_THREADS);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            float4 c;
            c.x = __fadd_rn(a[u].x, b[u].x);
            c.y = __fadd_rn(a[u].y, b[u].y);
            c.z = __fadd_rn(a[u].z, b[u].z);
            c.w = __fadd_rn(a[u].w, b[u].w);
            st_stream_f4(z4 + base + u * ADD_THREADS, c);
        }
    }
    // the ragged tile (owner: the CTA next in the round robin) and the scalar tail
    if ((int64_t)blockIdx.x == full_tiles % gridDim.x) {
        for (int64_t v = full_tiles * TILE_VECS + threadIdx.x; v < nvec; v += ADD_THREADS) {
            const float4 a = ld_stream_f4(x4 + v), b = ld_stream_f4(y4 + v);
            float4 c;
            c.x = __fadd_rn(a.x, b.x);
            c.y = __fadd_rn(a.y, b.y);
            c.z = __fadd_rn(a.z, b.z);
            c.w = __fadd_rn(a.w, b.w);
            st_stream_f4(z4 + v, c);
        }
        const int64_t e = (nvec << 2) + threadIdx.x;
        if (e < n) z[e] = __fadd_rn(__ldg(x + e), __ldg(y + e));
    }
}

// Any 4-byte alignment: element-wise, still coalesced (a warp touches 128 contiguous bytes).
__global__ void __launch_bounds__(ADD_THREADS)
add_f32_scalar_kernel(const float* __restrict__ x, const float* __restrict__ y, float* __restrict__ z, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * ADD_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * ADD_THREADS)
        z[i] = __fadd_rn(__ldg(x + i), __ldg(y + i));
}

}  // namespace tg
