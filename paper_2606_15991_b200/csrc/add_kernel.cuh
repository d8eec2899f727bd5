// Element-wise add for sm_100a:  z_i = fl32(x_i + y_i)  over f32 vectors.
//
// What it computes: Listing 1 of the paper -- every tile program loads the
// tiles of x and y that line up with its exclusively owned sub-tensor of z, adds them and
// stores the sum; the paper measures it at n = 2^28 (6.97 TB/s on its B200,
// PAPER.md:306).  12 bytes of HBM traffic per element and one FADD: purely bandwidth bound, so
// the only jobs are to keep enough bytes in flight per SM and to waste none.
//
//   * a "tile" here is ADD_THREADS * UNROLL vectors (e.g. 256 * 4 * 4 = 4096 elements);
//     tile t is owned by exactly one CTA (t = blockIdx.x, + gridDim.x, ...), the same
//     one-owner-per-sub-tensor contract as Listing 1's `.partition([128])`;
//   * every thread issues all 2 * UNROLL vector loads (16 or 32 bytes each) of its tile before
//     the first add, streaming hints on loads and stores;
//   * bounds: full tiles run with no predicate at all; the single ragged tile and the < 4
//     element tail are handled once, after the loop (the paper's "masked stores" for the edge
//     tile, with the check hoisted out of the hot loop).
#pragma once
#include <stdint.h>

#include "ptx.cuh"

namespace tg {

constexpr int ADD_THREADS = 256;

// One vector of VW floats (VW = 4: 128-bit, VW = 8: 256-bit accesses, sm_100+).  HINT: streaming
// cache hints (read-only path without L1 allocation, evict-first stores) or plain ld/st.
template <int VW>
struct AddVec {
    float v[VW];
};

template <int VW, bool HINT>
__device__ __forceinline__ AddVec<VW> add_ld(const float* p) {
    AddVec<VW> r;
    if constexpr (VW == 8) {
        if constexpr (HINT)
            asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                         : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]), "=f"(r.v[4]), "=f"(r.v[5]),
                           "=f"(r.v[6]), "=f"(r.v[7])
                         : "l"(p));
        else
            asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                         : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]), "=f"(r.v[4]), "=f"(r.v[5]),
                           "=f"(r.v[6]), "=f"(r.v[7])
                         : "l"(p));
    } else {
        if constexpr (HINT)
            asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3])
                         : "l"(p));
        else
            asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3])
                         : "l"(p));
    }
    return r;
}

template <int VW, bool HINT>
__device__ __forceinline__ void add_st(float* p, const AddVec<VW>& r) {
    if constexpr (VW == 8) {
        asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "f"(r.v[0]), "f"(r.v[1]),
                     "f"(r.v[2]), "f"(r.v[3]), "f"(r.v[4]), "f"(r.v[5]), "f"(r.v[6]), "f"(r.v[7])
                     : "memory");
    } else {
        if constexpr (HINT)
            asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(r.v[0]), "f"(r.v[1]), "f"(r.v[2]),
                         "f"(r.v[3])
                         : "memory");
        else
            asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(r.v[0]), "f"(r.v[1]), "f"(r.v[2]),
                         "f"(r.v[3])
                         : "memory");
    }
}

// x, y, z aligned to VW * 4 bytes.  n / VW full vectors; the n % VW tail elements follow them.
template <int UNROLL, int VW, bool HINT>
__global__ void __launch_bounds__(ADD_THREADS)
add_f32_vec_kernel(const float* __restrict__ x, const float* __restrict__ y, float* __restrict__ z, int64_t n) {
    constexpr int64_t TILE_VECS = (int64_t)ADD_THREADS * UNROLL;
    // programmatic dependent launch: the next kernel of the stream may be scheduled now; x and y may be
    // the previous kernel's output, so nothing is read before the wait (a no-op without the attribute)
    griddep_launch_dependents();
    griddep_wait();
    const int64_t nvec = n / VW;
    const int64_t full_tiles = nvec / TILE_VECS;
    for (int64_t t = blockIdx.x; t < full_tiles; t += gridDim.x) {
        const int64_t base = (t * TILE_VECS + threadIdx.x) * VW;
        AddVec<VW> a[UNROLL], b[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) a[u] = add_ld<VW, HINT>(x + base + (int64_t)u * ADD_THREADS * VW);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) b[u] = add_ld<VW, HINT>(y + base + (int64_t)u * ADD_THREADS * VW);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
            for (int e = 0; e < VW; ++e) a[u].v[e] = __fadd_rn(a[u].v[e], b[u].v[e]);
            add_st<VW, HINT>(z + base + (int64_t)u * ADD_THREADS * VW, a[u]);
        }
    }
    // the ragged tile (owner: the CTA next in the round robin) and the scalar tail
    if ((int64_t)blockIdx.x == full_tiles % gridDim.x) {
        for (int64_t v = full_tiles * TILE_VECS + threadIdx.x; v < nvec; v += ADD_THREADS) {
            AddVec<VW> a = add_ld<VW, HINT>(x + v * VW);
            const AddVec<VW> b = add_ld<VW, HINT>(y + v * VW);
#pragma unroll
            for (int e = 0; e < VW; ++e) a.v[e] = __fadd_rn(a.v[e], b.v[e]);
            add_st<VW, HINT>(z + v * VW, a);
        }
        const int64_t e = nvec * VW + threadIdx.x;
        if (e < n) z[e] = __fadd_rn(__ldg(x + e), __ldg(y + e));
    }
}

// Any 4-byte alignment: element-wise, still coalesced (a warp touches 128 contiguous bytes).
__global__ void __launch_bounds__(ADD_THREADS)
add_f32_scalar_kernel(const float* __restrict__ x, const float* __restrict__ y, float* __restrict__ z, int64_t n) {
    griddep_launch_dependents();
    griddep_wait();
    for (int64_t i = (int64_t)blockIdx.x * ADD_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * ADD_THREADS)
        z[i] = __fadd_rn(__ldg(x + i), __ldg(y + i));
}

}  // namespace tg
