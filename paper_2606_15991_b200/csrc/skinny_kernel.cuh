// skinny_tc_kernel: C = A * B for a FEW activation rows (M <= 64, "decode with some tokens in flight",
// SURVEY.md 8(f)2) -- a weight stream like the M = 1 kernel, with the arithmetic on the tensor cores.
//
// Same definition as everywhere: C[m][j] = sum_k A[m][k] * B[k][j], fp32
// accumulation.  At these M every weight is still read exactly once and the work is HBM-bound
// (PAPER.md:347), but M FMAs per weight are too many for the CUDA cores from M = 5 on.  So the
// schedule is gemv_split_kernel's -- one CTA per (column block, K slice), a TMA ring of 64(k)-row
// weight tiles, interleaved split-K, two CTAs per SM, programmatic dependent launch -- and the
// product runs with the operands SWAPPED on tcgen05:
//
//     D[n][m] (+)= sum_k  W[k][n] * X[m][k]        MMA "A" = the weight tile   (128 n x 16 k, MN-major:
//                                                             row-major K x N needs no transpose)
//                                                  MMA "B" = the activations   (a_rows m x 16 k, K-major)
//
// so the tensor-core work is proportional to a_rows = 16, 32 or 64 (M rounded up; the rows past M are
// TMA zero fill), the accumulator is 128 TMEM lanes (n) x a_rows columns (m), and all four epilogue
// warps hold live data.  Bounds: none in the K loop -- the N, K and M tails arrive as
// zeros and the stores are clipped at (M, N).
//
// Split-K hand-over (S = gridDim.y <= 8 slices of a column block = one thread-block cluster along y):
// a reduce-scatter through distributed shared memory.  The column block's 128 columns are four
// groups of 32 (one epilogue warp's TMEM lane quarter); group g belongs to slice g mod S.  A slice
// pushes the partial sums of every group it does not own into the owner's shared memory with
// st.async (16 bytes per store, each counting itself on the owner's mbarrier) and is done; the owner
// waits on that barrier -- no global workspace, no tickets, no polling -- adds slice 0 + slice 1 + ...
// in slice order (fixed order: bitwise reproducible) and stores C.
#pragma once
#include "gemv_kernel.cuh"
#include "ptx.cuh"

namespace tg {

constexpr int SKINNY_THREADS = 192;       // warps 0-3: epilogue (warp w = TMEM lanes 32w..32w+31), warp 4: TMA producer, warp 5: TMEM + MMA issuer
constexpr int SKINNY_BK = 64;             // k rows per ring stage: one 128-byte swizzle row of the activations
constexpr int SKINNY_COLS = 128;          // weight columns per CTA = M of the MMA
constexpr int SKINNY_GROUPS = 4;          // hand-over granularity: 32 columns
constexpr int SKINNY_MAX_CLUSTER = 8;     // portable cluster size
constexpr int SKINNY_MAX_ROWS = 64;

struct SkinnyParams {
    void* C;
    int64_t ldc;          // elements
    int32_t M, N, K;
    int32_t k_tiles;      // ceil(K / 64), >= gridDim.y
    int32_t a_rows;       // 16, 32 or 64: rows of the activation box = N of the MMA
    int32_t out_kind;     // 0: fp32, 1: bf16, 2: f16
    int32_t in_f16;
    int32_t flags;        // GEMV_FLAG_B_IMMUTABLE
    int32_t l2_post;      // B_IMMUTABLE: k-tiles brought into L2 right after the dependency wait
};

// 16-byte store into another CTA's shared memory that counts its bytes on an mbarrier of that CTA
__device__ __forceinline__ void st_async_v4(uint32_t cluster_addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d,
                                            uint32_t cluster_bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];"
                 ::"r"(cluster_addr), "r"(a), "r"(b), "r"(c), "r"(d), "r"(cluster_bar)
                 : "memory");
}
// TMEM -> registers: this warp's 32 lanes x 16 consecutive 32-bit columns
__device__ __forceinline__ void tmem_ld_32x16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ float4 ld_shared_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}

// shared-memory layout (offsets from the 1024-byte aligned base); the activation stages depend on a_rows
template <int STAGES>
struct SkinnySmem {
    static constexpr uint32_t W_BOX_BYTES = 64 * SKINNY_BK * 2;            // one TMA box: 64 k-rows x 64 columns (128 B)
    static constexpr uint32_t W_STAGE = 2 * W_BOX_BYTES;                   // 128 columns
    static constexpr uint32_t X_OFF = STAGES * W_STAGE;
    static constexpr uint32_t NUM_BARS = 2 * STAGES + 2;
    __host__ __device__ static constexpr uint32_t x_stage(int a_rows) { return (uint32_t)a_rows * SKINNY_BK * 2; }
    __host__ __device__ static constexpr uint32_t bar_off(int a_rows) { return X_OFF + STAGES * x_stage(a_rows); }
    // receive buffer of the split-K reduce-scatter: [source slice (S-1)][owned group][m / 4][32 lanes][4 floats]
    __host__ __device__ static constexpr uint32_t recv_off(int a_rows) { return (bar_off(a_rows) + NUM_BARS * 8 + 16 + 127u) & ~127u; }
    __host__ __device__ static constexpr uint32_t recv_bytes(int S, int mp) {
        return S > 1 ? (uint32_t)(S - 1) * (uint32_t)((SKINNY_GROUPS + S - 1) / S) * (uint32_t)mp * 128u : 0u;
    }
    __host__ __device__ static constexpr uint32_t total(int a_rows, int S, int mp) {
        return recv_off(a_rows) + recv_bytes(S, mp) + 1024;   // + slack for 1024 B alignment
    }
};

template <int STAGES>
__global__ void __launch_bounds__(SKINNY_THREADS, 2)
skinny_tc_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_x,
                 const SkinnyParams p) {
    using L = SkinnySmem<STAGES>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const int S = (int)gridDim.y, slice = (int)blockIdx.y;   // S > 1: gridDim.y == cluster size, %cluster_ctarank == slice
    const int n0 = (int)blockIdx.x * SKINNY_COLS;
    const int a_rows = p.a_rows;
    const uint32_t x_stage = L::x_stage(a_rows);
    const uint32_t bar_base = smem_base + L::bar_off(a_rows);
    auto full_bar = [&](uint32_t s) { return bar_base + s * 8u; };
    auto empty_bar = [&](uint32_t s) { return bar_base + (STAGES + s) * 8u; };
    const uint32_t acc_bar = bar_base + 2 * STAGES * 8u;            // all MMAs of this CTA have completed
    const uint32_t recv_bar = acc_bar + 8u;                         // every partial sum this CTA combines has arrived
    volatile uint32_t* tmem_ptr_gen = reinterpret_cast<volatile uint32_t*>(smem_gen + L::bar_off(a_rows) + L::NUM_BARS * 8);
    const uint32_t TMEM_COLS = a_rows <= 32 ? 32u : 64u;            // >= a_rows, a power of two, 32 the smallest allocation

    // the next kernel of the stream may be scheduled as soon as slots free up: everything of ours that it could
    // disturb sits behind its own griddepcontrol.wait
    griddep_launch_dependents();

    // this slice's k-tiles: slice, slice + S, ...
    const int n_my = p.k_tiles > slice ? (p.k_tiles - slice + S - 1) / S : 0;

    // The producer's elected lane initialises the barriers and -- weights being immutable -- sends the
    // first ring-full of weight tiles on its way BEFORE the CTA-wide sync below: tensor-memory
    // allocation and the sync are then hidden behind the first HBM round trip.
    const uint32_t tx_bytes = L::W_STAGE + x_stage;   // full boxes, even when clipped
    auto issue_w = [&](uint32_t stage, int kt) {
        mbar_arrive_expect_tx(full_bar(stage), tx_bytes);
        tma_load_2d(smem_base + stage * L::W_STAGE, &tmap_w, full_bar(stage), n0, kt * SKINNY_BK);
        tma_load_2d(smem_base + stage * L::W_STAGE + L::W_BOX_BYTES, &tmap_w, full_bar(stage), n0 + 64, kt * SKINNY_BK);
    };
    const bool pre_w = (p.flags & GEMV_FLAG_B_IMMUTABLE) != 0;
    const int n_pre = pre_w ? (n_my < STAGES ? n_my : STAGES) : 0;
    bool producer_lane = false;
    if (warp == 4 && elect_one()) {
        producer_lane = true;
        prefetch_tmap(&tmap_w);
        prefetch_tmap(&tmap_x);
        for (uint32_t s = 0; s < (uint32_t)STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        mbar_init(acc_bar, 1);
        mbar_init(recv_bar, 1);
        fence_mbar_init();
        for (int j = 0; j < n_pre; ++j) issue_w((uint32_t)j, slice + j * S);
    }
    if (warp == 5) {
        tmem_alloc<1>(smem_u32(const_cast<uint32_t*>(tmem_ptr_gen)), TMEM_COLS);
        tmem_relinquish<1>();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr_gen;
    if (S > 1) cluster_arrive();   // "my barriers exist"; the matching wait sits in front of the first remote access

    if (warp == 4) {
        // ===== TMA producer: per k-tile two weight boxes (64 columns x 64 k, 128B-swizzled) and the
        //       a_rows x 64 activations of the same k range, all on the stage's barrier =====
        if (producer_lane) {
            auto issue_x = [&](uint32_t stage, int kt) {
                tma_load_2d(smem_base + L::X_OFF + stage * x_stage, &tmap_x, full_bar(stage), kt * SKINNY_BK, 0);
            };
            // the activations (which the previous kernel of the stream may have written) follow the dependency wait
            griddep_wait();
            for (int j = 0; j < n_pre; ++j) issue_x((uint32_t)j, slice + j * S);
            int i = n_pre;
            // the ring is full and its activations are on their way: meanwhile the next k-tiles go as far as L2
            if (pre_w)
                for (int j = 0; j < p.l2_post && i + j < n_my; ++j) {
                    tma_prefetch_l2_2d(&tmap_w, n0, (slice + (i + j) * S) * SKINNY_BK);
                    tma_prefetch_l2_2d(&tmap_w, n0 + 64, (slice + (i + j) * S) * SKINNY_BK);
                }
            uint32_t stage = (uint32_t)(n_pre % STAGES), phase = (uint32_t)(n_pre / STAGES);
            for (; i < n_my; ++i) {
                mbar_wait(empty_bar(stage), phase ^ 1u);
                issue_w(stage, slice + i * S);
                issue_x(stage, slice + i * S);
                if (++stage == (uint32_t)STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        __syncwarp();
    } else if (warp == 5) {
        // ===== MMA issuer (one lane): D[n][m] += W^T X^T, M = 128 (weight columns), N = a_rows, K = 16 =====
        if (elect_one()) {
            // instruction descriptor: D = f32, A = B = bf16 | f16, A MN-major (bit 15), B K-major
            const uint32_t ab_fmt = p.in_f16 ? 0u : 1u;
            const uint32_t idesc = (1u << 4) | (ab_fmt << 7) | (ab_fmt << 10) | (1u << 15) | (0u << 16) |
                                   ((uint32_t)(a_rows >> 3) << 17) | ((uint32_t)(SKINNY_COLS >> 4) << 24);
            // smem descriptors (version 1, SWIZZLE_128B):
            //   weights (MN-major):     LBO = one 64-column box (8192 B), SBO = 1024 B between 8-k groups
            //   activations (K-major):  LBO unused (= 1), SBO = 1024 B between 8-row groups
            constexpr uint64_t desc_hi = (uint64_t(1) << 46) | (uint64_t(2) << 61);
            constexpr uint64_t w_desc_base = desc_hi | (uint64_t(L::W_BOX_BYTES >> 4) << 16) | (uint64_t(1024 >> 4) << 32);
            constexpr uint64_t x_desc_base = desc_hi | (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32);
            uint32_t stage = 0, phase = 0;
            for (int i = 0; i < n_my; ++i) {
                mbar_wait(full_bar(stage), phase);
                tc_fence_after();
                const uint32_t sw = smem_base + stage * L::W_STAGE;
                const uint32_t sx = smem_base + L::X_OFF + stage * x_stage;
                const uint64_t w_desc = w_desc_base | (uint64_t)((sw & 0x3FFFFu) >> 4);
                const uint64_t x_desc = x_desc_base | (uint64_t)((sx & 0x3FFFFu) >> 4);
#pragma unroll
                for (int k = 0; k < SKINNY_BK / 16; ++k) {
                    // weights: +16 k-rows of 128 B = +2048 B; activations: +16 elements along K = +32 B in the swizzled row
                    umma_bf16<1>(tmem_base, w_desc + (uint64_t)(k * 128), x_desc + (uint64_t)(k * 2), idesc,
                                 (uint32_t)((i != 0) | (k != 0)));
                }
                umma_commit<1>(empty_bar(stage));
                if (++stage == (uint32_t)STAGES) { stage = 0; phase ^= 1u; }
            }
            umma_commit<1>(acc_bar);   // arrives once every MMA above has completed
        }
        __syncwarp();
    } else {
        // ===== epilogue: warp w holds columns n0 + 32 w + lane, a_rows values of m each =====
        const int mp = (p.M + 3) & ~3;                 // rows handed over: M rounded up to whole 16-byte stores (the extra rows are exact zeros)
        const int g = (int)warp;                       // this warp's group
        const int owner = g % S;
        const int slot = g / S;                        // which of the owner's groups
        const int slots = (SKINNY_GROUPS + S - 1) / S;
        const uint32_t recv_base = smem_base + L::recv_off(a_rows);
        const int n = n0 + g * 32 + (int)lane;
        auto store_c = [&](int m, float v) {
            if (m < p.M && n < p.N) {
                const int64_t idx = (int64_t)m * p.ldc + n;
                if (p.out_kind == 0) reinterpret_cast<float*>(p.C)[idx] = v;
                else if (p.out_kind == 1) reinterpret_cast<uint16_t*>(p.C)[idx] = f32_to_bf16_rne(v);
                else reinterpret_cast<uint16_t*>(p.C)[idx] = __half_as_ushort(__float2half_rn(v));
            }
        };
        if (S > 1 && threadIdx.x == 0 && slice < SKINNY_GROUPS) {   // this slice owns groups slice, slice + S, ...: expect their partial sums
            int owned = 0;
            for (int gg = slice; gg < SKINNY_GROUPS; gg += S) ++owned;
            mbar_arrive_expect_tx(recv_bar, (uint32_t)owned * (uint32_t)(S - 1) * (uint32_t)mp * 128u);
        }
        griddep_wait();   // C may still be in the previous kernel's use
        if (S > 1) cluster_wait();   // every peer's barriers exist (long since: this is off the critical path here)
        mbar_wait(acc_bar, 0);
        tc_fence_after();
        const uint32_t t_lane = tmem_base + ((warp * 32u) << 16);
        uint32_t v[16];
        if (S == 1) {
#pragma unroll 1
            for (int m0 = 0; m0 < p.M; m0 += 16) {
                tmem_ld_32x16(t_lane + (uint32_t)m0, v);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 16; ++j) store_c(m0 + j, __uint_as_float(v[j]));
            }
        } else if (owner != slice) {
            // ---- push this warp's group to its owner: [source][slot][m / 4][lane][4 floats] ----
            const uint32_t rbar = map_to_cta(recv_bar, (uint32_t)owner);
            const int src = slice < owner ? slice : slice - 1;
            const uint32_t dst0 = map_to_cta(recv_base + (uint32_t)((src * slots + slot) * (mp >> 2)) * 512u + lane * 16u, (uint32_t)owner);
#pragma unroll 1
            for (int m0 = 0; m0 < mp; m0 += 16) {
                tmem_ld_32x16(t_lane + (uint32_t)m0, v);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (m0 + 4 * j < mp)
                        st_async_v4(dst0 + (uint32_t)((m0 >> 2) + j) * 512u, v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3], rbar);
            }
        } else {
            // ---- combine this warp's group: slice 0 + slice 1 + ... (fixed order) ----
            mbar_wait(recv_bar, 0);
#pragma unroll 1
            for (int m0 = 0; m0 < mp; m0 += 16) {
                tmem_ld_32x16(t_lane + (uint32_t)m0, v);
                tmem_ld_wait();
                float acc[16];
#pragma unroll 1
                for (int s = 0; s < S; ++s) {
                    float val[16];
                    if (s == slice) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) val[j] = __uint_as_float(v[j]);
                    } else {
                        const int src = s < slice ? s : s - 1;
                        const uint32_t from = recv_base + (uint32_t)((src * slots + slot) * (mp >> 2) + (m0 >> 2)) * 512u + lane * 16u;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
                            if (m0 + 4 * j < mp) f = ld_shared_f4(from + (uint32_t)j * 512u);
                            val[4 * j] = f.x; val[4 * j + 1] = f.y; val[4 * j + 2] = f.z; val[4 * j + 3] = f.w;
                        }
                    }
                    if (s == 0) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] = val[j];
                    } else {
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] += val[j];
                    }
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) store_c(m0 + j, acc[j]);
            }
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == 5) {
        tc_fence_after();
        tmem_dealloc<1>(tmem_base, TMEM_COLS);
    }
}

}  // namespace tg
