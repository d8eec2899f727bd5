// M = 1 decode GEMV for sm_100a:  y_j = sum_k x_k * B[k][j], bf16 in, fp32 accumulate.
//
// The same definition as the GEMM at M = 1, where the work is HBM-bound
// (decode roofline R = beta / (W + Kbar)): every weight is read exactly once, so
// the kernels only have to keep enough bytes in flight and waste none.  No tensor cores.
//
//   gemv_split_kernel : B rows are 16-byte addressable (the default, described at its definition below).  One
//                     producer warp streams weight tiles through a shared-memory ring with TMA + mbarriers; TMA
//                     zero fill handles the K and N tails.  Eight consumer warps each own rows of a tile,
//                     lanes own 8 consecutive columns (one conflict-free 16-byte LDS per row).
//   gemv_ldg_kernel : generic fallback (any alignment): direct global loads, 16-byte when VEC.
//
// Split-K of the fallback: gridDim.y CTAs (one thread-block cluster along y) share a column block; partial
// sums are combined through distributed shared memory in a fixed order (thread -> warp -> cluster
// rank), so results are bitwise reproducible and need no global workspace or atomics.  (Round 3 removed
// gemv_tma_kernel, the round-1 TMA kernel with that same cluster reduction: the automatic path never
// launched it once gemv_split_kernel existed.)
#pragma once
#include <cuda_fp16.h>

#include "ptx.cuh"

namespace tg {

constexpr int GEMV_COLS = 256;          // columns per CTA (32 lanes x 8)
constexpr int GEMV_TILE_K = 64;         // rows per TMA tile
constexpr int GEMV_CONSUMER_WARPS = 8;
constexpr int GEMV_TMA_THREADS = (GEMV_CONSUMER_WARPS + 1) * 32;
constexpr uint32_t GEMV_TILE_BYTES = GEMV_TILE_K * GEMV_COLS * 2;   // 32 KB

struct GemvParams {
    const uint16_t* x;
    const uint16_t* B;
    void* y;
    int32_t N, K;
    int64_t ldb;
    int32_t k_per_cta;   // rows per split-K slice (multiple of GEMV_TILE_K)
    int32_t out_kind;    // 0: fp32 y, 1: bf16 y, 2: f16 y
};

// 16-bit input element -> fp32 (exact).  F16 = false: bf16 is the upper half of a binary32;
// F16 = true: IEEE binary16 (the paper's precision), one cvt per element.
template <bool F16>
__device__ __forceinline__ float in_bits_to_f32(uint16_t h) {
    if constexpr (F16) return __half2float(__ushort_as_half(h));
    else return __uint_as_float(((uint32_t)h) << 16);
}

template <bool F16>
__device__ __forceinline__ void fma8(float (&acc)[8], const uint4& w, float xr) {
    if constexpr (F16) {
        const uint32_t u[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&u[i]));
            acc[2 * i] = fmaf(f.x, xr, acc[2 * i]);
            acc[2 * i + 1] = fmaf(f.y, xr, acc[2 * i + 1]);
        }
        return;
    }
    acc[0] = fmaf(__uint_as_float(w.x << 16), xr, acc[0]);
    acc[1] = fmaf(__uint_as_float(w.x & 0xffff0000u), xr, acc[1]);
    acc[2] = fmaf(__uint_as_float(w.y << 16), xr, acc[2]);
    acc[3] = fmaf(__uint_as_float(w.y & 0xffff0000u), xr, acc[3]);
    acc[4] = fmaf(__uint_as_float(w.z << 16), xr, acc[4]);
    acc[5] = fmaf(__uint_as_float(w.z & 0xffff0000u), xr, acc[5]);
    acc[6] = fmaf(__uint_as_float(w.w << 16), xr, acc[6]);
    acc[7] = fmaf(__uint_as_float(w.w & 0xffff0000u), xr, acc[7]);
}

__device__ __forceinline__ uint16_t f32_to_bf16_rne(float f) {
    uint16_t r;
    asm("cvt.rn.bf16.f32 %0, %1;" : "=h"(r) : "f"(f));
    return r;
}

// y[col] = round_out(s): out_kind 0 fp32, 1 bf16 (RNE), 2 f16 (RNE)
__device__ __forceinline__ void gemv_store(void* y, int col, float s, int out_kind) {
    if (out_kind == 0) reinterpret_cast<float*>(y)[col] = s;
    else if (out_kind == 1) reinterpret_cast<uint16_t*>(y)[col] = f32_to_bf16_rne(s);
    else reinterpret_cast<uint16_t*>(y)[col] = __half_as_ushort(__float2half_rn(s));
}

// Combine the per-thread partial sums of one CTA (warps ordered along K) and of the split-K
// cluster, then write this CTA's share of the 256 output columns.
//   red  : smem [nwarps][256] floats, part : smem [256] floats
template <int NWARPS>
__device__ __forceinline__ void gemv_reduce_and_store(const float (&acc)[8], float* red, float* part,
                                                      uint32_t cwarp, uint32_t lane, bool is_consumer,
                                                      const GemvParams& p, int n0) {
    if (is_consumer) {
#pragma unroll
        for (int e = 0; e < 8; ++e) red[cwarp * GEMV_COLS + lane * 8 + e] = acc[e];
    }
    __syncthreads();
    const uint32_t tid = threadIdx.x;
    if (tid < GEMV_COLS) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < NWARPS; ++w) s += red[w * GEMV_COLS + tid];   // fixed order
        part[tid] = s;
    }
    const uint32_t nsplit = gridDim.y;
    if (nsplit > 1) cluster_sync(); else __syncthreads();
    const uint32_t rank = blockIdx.y;   // cluster spans the whole y extent
    if (tid < GEMV_COLS && (tid % nsplit) == rank) {
        float s = 0.f;
        if (nsplit > 1) {
            const uint32_t a = smem_u32(&part[tid]);
            for (uint32_t q = 0; q < nsplit; ++q) s += ld_dsmem_f32(map_to_cta(a, q));   // fixed order
        } else {
            s = part[tid];
        }
        const int col = n0 + (int)tid;
        if (col < p.N) gemv_store(p.y, col, s, p.out_kind);
    }
    if (nsplit > 1) cluster_sync();   // peers may still be reading this CTA's `part`
}

// ---------------------------------------------------------------------------------------------
// gemv_split_kernel: the default M = 1 kernel.  Grid (x, S): CTA (bx, s) owns column blocks
// cb = bx, bx + gridDim.x, ... (256 columns each) and, inside each, the k-tiles kt = s, s + S,
// s + 2S, ... (TILE_K rows each): *interleaved* split-K, so at any moment the S x gridDim.x CTAs
// read one dense band of consecutive weight rows over the full row width -- the access pattern
// HBM likes best (measured: equal contiguous runs per CTA scattered over the matrix lose 4-18 %).
// All CTAs are co-resident and HBM-bound CTAs progress at equal rates, so equal tile counts per
// CTA (+-1) finish together whatever the SM count.
//
// Split-K fix-up: a CTA with S > 1 hands its 256 fp32 partial sums to one CTA of its column block,
// which adds the S partials in slice order (fixed order: bitwise reproducible, and the same bits
// whichever of the three protocols carries them) and stores y.  The hand-over is what ends a launch:
// it starts when the last tile has been consumed and nothing overlaps it, so its length in global
// round trips is what the short decode launches pay (measured with tile_gemm_debug_trace on
// K = 5120, N = 8192: 5 us of a 15 us launch with tickets, profiles/r02_gemv_trace.md).
//   * GEMV_FLAG_CLUSTER (S <= 8, one column block per CTA): the S slices are one thread-block
//     cluster.  Slice r > 0 pushes its partials into slice 0's shared memory with st.async, each
//     store counting its bytes on slice 0's mbarrier; slice 0 waits on that barrier.  No global
//     memory, no polling: ~1 us from last tile to y.
//   * GEMV_FLAG_PACKED (every CTA of the launch resident at once): a slice's thread writes
//     {partial, tag 1} as ONE 64-bit store into its slot and is done -- no fence, no ticket.  The CTA
//     of the LAST slice polls the S-1 other slots of its column block, sixteen loads in flight per
//     round, and writes them back to zero for the next launch.  One round trip + polling jitter.
//   * tickets (any launch, any S): partials to the workspace, __threadfence, a ticket on the column
//     block; the CTA that draws the last ticket re-reads all S partials.  Three dependent round trips.
//
// Programmatic dependent launch: every CTA signals launch_dependents at once, so the next kernel
// of the stream is scheduled while this one runs; everything that touches x, y or the workspace
// sits behind griddepcontrol.wait.  With GEMV_FLAG_B_IMMUTABLE (the caller promises that no work
// still in flight writes B: decode weights) the producer fills its ring with weight tiles ahead of
// that wait and, right after it, sends `l2_post` more units as far as L2 while the ring's
// activations are still on their way, so HBM stays busy across the kernel boundary.  (Measured and
// not kept: L2 prefetch ahead of the wait or all through the launch costs 1-15 %, it competes with
// the loads that are on the critical path; an evict-first policy on the weight stream and an L2
// prefetch of x change nothing.)
constexpr int GEMV_FLAG_B_IMMUTABLE = 1;
constexpr int GEMV_FLAG_X_TMA = 2;       // x is 16-byte aligned: its TILE_K-element slices ride the ring with the weight tiles
constexpr int GEMV_FLAG_PACKED = 8;
constexpr int GEMV_FLAG_CLUSTER = 32;
constexpr int GEMV_MAX_CLUSTER = 8;      // portable cluster size

struct GemvSplitParams {
    const uint16_t* x;
    void* y;
    float* partials;      // tickets: [col_blocks][split][COLS]
    uint32_t* tickets;    // tickets: [col_blocks], zero between launches
    unsigned long long* packed;   // GEMV_FLAG_PACKED: [col_blocks][split][COLS] slots {fp32 partial, tag}, all zero between launches
    int32_t N, K;
    int32_t k_tiles;      // ceil(K / TILE_K), >= split
    int32_t col_blocks;
    int32_t out_kind;     // 0: fp32 y, 1: bf16 y, 2: f16 y
    int32_t flags;
    int32_t l2_post;      // B_IMMUTABLE: units brought into L2 right after the dependency wait
    // tile_gemm_debug_trace: CTA (bx, by) writes its record of GEMV_TRACE_WORDS 64-bit words at
    // trace + (by * gridDim.x + bx) * GEMV_TRACE_WORDS when that index is below trace_cap
    unsigned long long* trace;
    int32_t trace_cap;
};
// trace record: [0] smid | bx << 16 | by << 32, then %globaltimer (ns) at [1] kernel entry, [2] release of
// griddepcontrol.wait, [3] first tile in shared memory, [4] last tile consumed, [5] CTA done; [6] tiles
// consumed; [7] ns: partial sums handed over (S > 1)
constexpr int GEMV_TRACE_WORDS = 8;
__device__ __forceinline__ uint32_t sm_id() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(r));
    return r;
}

__device__ __forceinline__ void consumer_bar_sync() {
    asm volatile("bar.sync 1, %0;" ::"n"(GEMV_CONSUMER_WARPS * 32) : "memory");
}
__device__ __forceinline__ float ld_cg_f32(const float* p) {
    float v;
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_cg_f32(float* p, float v) {
    asm volatile("st.global.cg.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}
// one naturally aligned 64-bit access: the fp32 partial and its tag become visible together
__device__ __forceinline__ void st_relaxed_gpu_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_gpu_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
template <int COLS, int TILE_K, int STAGES>
struct GemvSplitSmem {
    static constexpr uint32_t BOX_BYTES = TILE_K * GEMV_COLS * 2;          // one TMA box: TILE_K rows x 256 columns
    static constexpr uint32_t TILE_BYTES = (COLS / GEMV_COLS) * BOX_BYTES;
    static constexpr uint32_t X_OFF = STAGES * TILE_BYTES;                 // per stage: TILE_K activations (128 B slots)
    static constexpr uint32_t RED_OFF = X_OFF + STAGES * 128;
    // cluster fix-up (default ring shape only: the other shapes have no shared memory to spare at their
    // occupancy): the combiner receives the partial sums of the other <= 7 slices here
    static constexpr uint32_t RECV_BYTES = (COLS == GEMV_COLS && TILE_K == 64 && STAGES == 3) ? (GEMV_MAX_CLUSTER - 1) * COLS * 4 : 0;
    static constexpr uint32_t RECV_OFF = RED_OFF + GEMV_CONSUMER_WARPS * COLS * 4;
    static constexpr uint32_t FLAG_OFF = RECV_OFF + RECV_BYTES;
    static constexpr uint32_t BAR_OFF = FLAG_OFF + 16;
    static constexpr uint32_t TOTAL = BAR_OFF + (2 * STAGES + 1) * 8 + 128;   // + slack for 128 B alignment
};

// COLS columns per CTA (NV = COLS / 256 TMA boxes side by side: a row segment of COLS * 2
// contiguous bytes), TILE_K rows per ring stage.
template <int COLS, int TILE_K, int STAGES, int MIN_CTAS, bool F16>
__global__ void __launch_bounds__(GEMV_TMA_THREADS, MIN_CTAS)
gemv_split_kernel(const __grid_constant__ CUtensorMap tmap_b, const __grid_constant__ CUtensorMap tmap_x,
                  const GemvSplitParams p) {
    using L = GemvSplitSmem<COLS, TILE_K, STAGES>;
    constexpr int NV = COLS / GEMV_COLS;                 // 16-byte vectors per lane per row
    constexpr int RPW = TILE_K / GEMV_CONSUMER_WARPS;   // rows of a tile per consumer warp
    static_assert(NV >= 1 && NV <= 4 && COLS % GEMV_COLS == 0, "COLS is 256, 512, 768 or 1024");
    static_assert(RPW == 2 || RPW == 4 || RPW == 8, "TILE_K is 16, 32 or 64");
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    float* red = reinterpret_cast<float*>(smem_gen + L::RED_OFF);
    volatile uint32_t* s_last = reinterpret_cast<volatile uint32_t*>(smem_gen + L::FLAG_OFF);
    auto full_bar = [&](uint32_t s) { return smem_base + L::BAR_OFF + s * 8u; };
    auto empty_bar = [&](uint32_t s) { return smem_base + L::BAR_OFF + (STAGES + s) * 8u; };
    const uint32_t recv_bar = smem_base + L::BAR_OFF + 2 * STAGES * 8u;

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const int S = (int)gridDim.y, slice = (int)blockIdx.y;
    const int KT = p.k_tiles;
    // cluster mode: gridDim.y == cluster size, so %cluster_ctarank == slice
    const bool clus = L::RECV_BYTES > 0 && (p.flags & GEMV_FLAG_CLUSTER) != 0;

    const bool x_tma = (p.flags & GEMV_FLAG_X_TMA) != 0;
    // at entry (round 2: it used to follow the barrier set-up; +1.5-1.8 % on the two small decode shapes): the next
    // kernel of the stream is scheduled as soon as slots free up, everything it could disturb sits behind its own wait
    griddep_launch_dependents();
    unsigned long long* trace = nullptr;   // thread 0 only
    if (threadIdx.x == 0) {
        const int idx = (int)(blockIdx.y * gridDim.x + blockIdx.x);
        if (p.trace != nullptr && idx < p.trace_cap) {
            trace = p.trace + (size_t)idx * GEMV_TRACE_WORDS;
            trace[0] = (unsigned long long)sm_id() | ((unsigned long long)blockIdx.x << 16) | ((unsigned long long)blockIdx.y << 32);
            trace[1] = global_timer_ns();
        }
        prefetch_tmap(&tmap_b);
        if (x_tma) prefetch_tmap(&tmap_x);
        for (uint32_t s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), GEMV_CONSUMER_WARPS);
        }
        if (clus) mbar_init(recv_bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (clus) cluster_arrive();   // "my barriers exist"; the matching wait sits in front of the first remote access, at the very end

    if (warp == GEMV_CONSUMER_WARPS) {
        // ===== producer: one (column block, k-tile) unit per ring stage.  With x_tma the unit's
        //       TILE_K activations land in the same stage on the same barrier, so the consumers
        //       never wait on a global load of x =====
        if (elect_one()) {
            const uint32_t tx_bytes = L::TILE_BYTES + (x_tma ? (uint32_t)TILE_K * 2u : 0u);   // full boxes, even when clipped
            auto issue_b = [&](uint32_t stage, int cb, int kt) {
                mbar_arrive_expect_tx(full_bar(stage), tx_bytes);
#pragma unroll
                for (int v = 0; v < NV; ++v)
                    tma_load_2d(smem_base + stage * L::TILE_BYTES + v * L::BOX_BYTES, &tmap_b, full_bar(stage),
                                cb * COLS + v * GEMV_COLS, kt * TILE_K);
            };
            auto issue_x = [&](uint32_t stage, int kt) {
                if (x_tma) tma_load_2d(smem_base + L::X_OFF + stage * 128u, &tmap_x, full_bar(stage), kt * TILE_K, 0);
            };
            auto next_unit = [&](int& cb, int& kt) {
                kt += S;
                if (kt >= KT) { kt = slice; cb += (int)gridDim.x; }
            };
            int cb = (int)blockIdx.x, kt = slice;
            uint32_t stage = 0, phase = 0;
            const bool have_work = cb < p.col_blocks && kt < KT;
            if ((p.flags & GEMV_FLAG_B_IMMUTABLE) && have_work) {
                // weights first: the ring fills while the previous kernel of the stream drains; x (which
                // that kernel may have written) follows the dependency wait
                int cb2 = cb, kt2 = kt;
                uint32_t n_pre = 0;
                for (; n_pre < (uint32_t)STAGES && cb2 < p.col_blocks; ++n_pre) {
                    issue_b(n_pre, cb2, kt2);
                    next_unit(cb2, kt2);
                }
                griddep_wait();
                for (uint32_t i = 0; i < n_pre; ++i) {
                    issue_x(i, kt);
                    next_unit(cb, kt);
                }
                stage = n_pre % STAGES;
                phase = n_pre / STAGES;
                // the ring is full and its activations are on their way: meanwhile the next units go as far as L2
                cb2 = cb; kt2 = kt;
                for (int i = 0; i < p.l2_post && cb2 < p.col_blocks; ++i) {
#pragma unroll
                    for (int v = 0; v < NV; ++v) tma_prefetch_l2_2d(&tmap_b, cb2 * COLS + v * GEMV_COLS, kt2 * TILE_K);
                    next_unit(cb2, kt2);
                }
            } else {
                griddep_wait();
            }
            for (; cb < p.col_blocks; next_unit(cb, kt)) {
                mbar_wait(empty_bar(stage), phase ^ 1u);
                issue_b(stage, cb, kt);
                issue_x(stage, kt);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        __syncwarp();
        return;
    }

    // ===== consumers: warp w owns rows RPW*w .. RPW*w+RPW-1 of every tile; lane l owns columns
    //       256 v + 8 l .. + 7 of every box v =====
    griddep_wait();   // x may be the previous kernel's output; y and the workspace may still be in its use
    if (trace) trace[2] = global_timer_ns();
    int traced_tiles = 0;
    const uint32_t tid = threadIdx.x;   // 0..255
    auto load_x = [&](int kt_) -> float {   // only when x is not TMA-addressable
        const int k = kt_ * TILE_K + (int)warp * RPW + (int)(lane & (RPW - 1));
        return (!x_tma && kt_ < KT && k < p.K) ? in_bits_to_f32<F16>(__ldg(p.x + k)) : 0.f;
    };
    uint32_t stage = 0, phase = 0;
    for (int cb = (int)blockIdx.x; cb < p.col_blocks; cb += (int)gridDim.x) {
        float acc[NV][8];
#pragma unroll
        for (int v = 0; v < NV; ++v)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[v][e] = 0.f;
        float xv_next = load_x(slice);
        for (int kt = slice; kt < KT; kt += S) {
            const float xv = xv_next;
            xv_next = load_x(kt + S);
            mbar_wait(full_bar(stage), phase);
            if (trace && traced_tiles++ == 0) trace[3] = global_timer_ns();
            const uint8_t* tile = smem_gen + stage * L::TILE_BYTES + warp * RPW * (GEMV_COLS * 2) + lane * 16u;
            uint4 w[NV][RPW];
#pragma unroll
            for (int v = 0; v < NV; ++v)
#pragma unroll
                for (int r = 0; r < RPW; ++r)
                    w[v][r] = *reinterpret_cast<const uint4*>(tile + v * L::BOX_BYTES + r * (GEMV_COLS * 2));
            float xrow[RPW];
            if (x_tma) {   // this warp's RPW activations: broadcast reads of the stage's x slot
                const uint16_t* xs = reinterpret_cast<const uint16_t*>(smem_gen + L::X_OFF + stage * 128u) + warp * RPW;
#pragma unroll
                for (int r = 0; r < RPW; ++r) xrow[r] = in_bits_to_f32<F16>(xs[r]);
            } else {
#pragma unroll
                for (int r = 0; r < RPW; ++r) xrow[r] = __shfl_sync(0xffffffffu, xv, r);
            }
#pragma unroll
            for (int r = 0; r < RPW; ++r) {
#pragma unroll
                for (int v = 0; v < NV; ++v) fma8<F16>(acc[v], w[v][r], xrow[r]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        // ---- column block done for this slice: warps -> CTA -> (S > 1) slices ----
        if (trace) { trace[4] = global_timer_ns(); trace[6] = (unsigned long long)traced_tiles; }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            float4* r4 = reinterpret_cast<float4*>(red + warp * COLS + v * GEMV_COLS + lane * 8);
            r4[0] = make_float4(acc[v][0], acc[v][1], acc[v][2], acc[v][3]);
            r4[1] = make_float4(acc[v][4], acc[v][5], acc[v][6], acc[v][7]);
        }
        consumer_bar_sync();
        float s[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            s[v] = 0.f;
#pragma unroll
            for (int w8 = 0; w8 < GEMV_CONSUMER_WARPS; ++w8) s[v] += red[w8 * COLS + v * GEMV_COLS + tid];   // fixed order
        }
        bool store = (S == 1);
        if (!store && clus) {
            // DSMEM fix-up: slice r > 0 pushes its 256 partial sums into slice 0's shared memory with
            // st.async (each store counts its bytes on slice 0's mbarrier) and is done; slice 0 waits on
            // that barrier -- no global memory, no polling -- and adds own + slice 1 + ... in slice order
            // (the order of the other two protocols: identical bits)
            if constexpr (L::RECV_BYTES > 0) {
                cluster_wait();
                if (slice != 0) {
                    const uint32_t rbar = map_to_cta(recv_bar, 0);
                    const uint32_t dst = map_to_cta(smem_base + L::RECV_OFF + (uint32_t)((slice - 1) * COLS + (int)tid) * 4u, 0);
                    st_async_f32(dst, s[0], rbar);
                    if (trace) trace[7] = global_timer_ns();
                } else {
                    if (tid == 0) mbar_arrive_expect_tx(recv_bar, (uint32_t)(S - 1) * COLS * 4u);
                    if (trace) trace[7] = global_timer_ns();
                    mbar_wait(recv_bar, 0);
                    const float* recv = reinterpret_cast<const float*>(smem_gen + L::RECV_OFF);
                    for (int r = 1; r < S; ++r) s[0] += recv[(r - 1) * COLS + (int)tid];   // fixed order
                    store = true;
                }
            }
        } else if (!store && (p.flags & GEMV_FLAG_PACKED)) {
            unsigned long long* slots = p.packed + (size_t)cb * S * COLS + tid;
            if (slice != S - 1) {
#pragma unroll
                for (int v = 0; v < NV; ++v)
                    st_relaxed_gpu_u64(slots + (size_t)slice * COLS + v * GEMV_COLS,
                                       (1ull << 32) | (unsigned long long)__float_as_uint(s[v]));
                if (trace) trace[7] = global_timer_ns();
            } else {
                if (trace) trace[7] = global_timer_ns();
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const float own = s[v];
                    s[v] = 0.f;
                    // sixteen slots at a time: all loads of a round are in flight together, a round is repeated
                    // until every tag of the chunk shows, then the chunk is added in slice order
                    for (int q0 = 0; q0 < S - 1; q0 += 16) {
                        unsigned long long got[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) got[j] = 0ull;
#if TILEGEMM_WATCHDOG
                        uint64_t t0 = 0;
                        uint32_t rounds = 0;
#endif
                        for (;;) {
                            bool all = true;
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                if (q0 + j < S - 1 && (uint32_t)(got[j] >> 32) == 0u) {
                                    got[j] = ld_relaxed_gpu_u64(slots + (size_t)(q0 + j) * COLS + v * GEMV_COLS);
                                    all = all && (uint32_t)(got[j] >> 32) != 0u;
                                }
                            if (all) break;
#if TILEGEMM_WATCHDOG
                            if ((++rounds & 0xfffu) == 0) {
                                if (t0 == 0) t0 = global_timer_ns();
                                else if (global_timer_ns() - t0 > 4000000000ull) {
#if TILEGEMM_WATCHDOG >= 2
                                    printf("tilegemm watchdog: split-K slot wait timed out (block %d,%d thread %d)\n",
                                           (int)blockIdx.x, (int)blockIdx.y, (int)threadIdx.x);
#endif
                                    __trap();
                                }
                            }
#endif
                        }
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (q0 + j < S - 1) {
                                s[v] += __uint_as_float((uint32_t)got[j]);
                                st_relaxed_gpu_u64(slots + (size_t)(q0 + j) * COLS + v * GEMV_COLS, 0ull);   // re-arm
                            }
                    }
                    s[v] += own;
                }
                store = true;
            }
        } else if (!store) {
            float* part = p.partials + (size_t)cb * S * COLS + tid;
#pragma unroll
            for (int v = 0; v < NV; ++v) st_cg_f32(part + (size_t)slice * COLS + v * GEMV_COLS, s[v]);
            __threadfence();
            consumer_bar_sync();
            if (tid == 0) {
                const uint32_t old = atomicAdd(p.tickets + cb, 1u);
                const bool last = (old == (uint32_t)(S - 1));
                if (last) p.tickets[cb] = 0u;   // every slice has arrived: re-arm for the next launch
                *s_last = last ? 1u : 0u;
            }
            consumer_bar_sync();
            if (trace) trace[7] = global_timer_ns();
            if (*s_last) {
                __threadfence();
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    s[v] = 0.f;
                    for (int q0 = 0; q0 < S; q0 += 8) {   // eight independent loads in flight, added in slice order
                        float got[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if (q0 + j < S) got[j] = ld_cg_f32(part + (size_t)(q0 + j) * COLS + v * GEMV_COLS);
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if (q0 + j < S) s[v] += got[j];
                    }
                }
                store = true;
            }
        }
        if (store) {
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const int col = cb * COLS + v * GEMV_COLS + (int)tid;
                if (col < p.N) gemv_store(p.y, col, s[v], p.out_kind);
            }
        }
        consumer_bar_sync();   // red and s_last are free for the next column block
    }
    if (trace) trace[5] = global_timer_ns();
}

// Generic fallback: no alignment requirement on B when VEC == false.
template <bool VEC, bool F16>
__global__ void __launch_bounds__(256)
gemv_ldg_kernel(const GemvParams p) {
    __shared__ float red[8 * GEMV_COLS];
    __shared__ float part[GEMV_COLS];
    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const int n0 = (int)blockIdx.x * GEMV_COLS;
    const int col0 = n0 + (int)lane * 8;
    const int k_begin = (int)blockIdx.y * p.k_per_cta;
    const int k_end = min(p.K, k_begin + p.k_per_cta);
    // warp w takes a contiguous share of the CTA's K slice
    const int len = max(0, k_end - k_begin);
    const int per_warp = (len + 7) / 8;
    const int wb = k_begin + (int)warp * per_warp;
    const int we = min(k_end, wb + per_warp);
    const int ncols = min(8, p.N - col0);   // <= 0: this lane owns no column

    float acc[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = 0.f;

    auto load_row = [&](int k) -> uint4 {
        uint4 w = make_uint4(0u, 0u, 0u, 0u);
        const uint16_t* src = p.B + (int64_t)k * p.ldb + col0;
        if (VEC && ncols == 8) {
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w)
                         : "l"(src));
        } else if (ncols > 0) {
            uint32_t h[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) h[e] = (e < ncols) ? (uint32_t)__ldg(src + e) : 0u;
            w.x = h[0] | (h[1] << 16);
            w.y = h[2] | (h[3] << 16);
            w.z = h[4] | (h[5] << 16);
            w.w = h[6] | (h[7] << 16);
        }
        return w;
    };

    for (int k0 = wb; k0 < we; k0 += 32) {
        const int kk = k0 + (int)lane;
        const float xv = (kk < we) ? in_bits_to_f32<F16>(__ldg(p.x + kk)) : 0.f;
        const int nrows = min(32, we - k0);
        if (nrows == 32) {
#pragma unroll
            for (int r0 = 0; r0 < 32; r0 += 8) {
                uint4 w[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) w[u] = load_row(k0 + r0 + u);
#pragma unroll
                for (int u = 0; u < 8; ++u) fma8<F16>(acc, w[u], __shfl_sync(0xffffffffu, xv, r0 + u));
            }
        } else {
            for (int r = 0; r < nrows; ++r) {
                const uint4 w = load_row(k0 + r);
                fma8<F16>(acc, w, __shfl_sync(0xffffffffu, xv, r));
            }
        }
    }
    gemv_reduce_and_store<8>(acc, red, part, warp, lane, true, p, n0);
}

}  // namespace tg
