// gemv_rows_kernel: the decode GEMV for M = 2..4 activation rows (a few tokens in flight).
//
// Same definition as everywhere: C[m][j] = sum_k A[m][k] * B[k][j], fp32
// accumulation.  At these M the work is still HBM-bound on the weights, so the
// schedule is gemv_split_kernel's -- a TMA ring of 64(k) x 256(n) weight tiles, interleaved split-K
// over a (column block, slice) grid, per-column-block ticket and fixed-order fix-up, programmatic
// dependent launch -- with every weight tile used MR times: each row of a tile is unpacked to fp32
// once and multiplied into MR accumulator sets.  The MR x 64 activations of a k-tile ride the ring
// with the tile (one TMA box over A), so the consumers never touch global memory in the loop.
// Requires A and B TMA-addressable; otherwise the selector takes the tensor-core path.
#pragma once
#include "gemv_kernel.cuh"

namespace tg {

struct GemvRowsParams {
    void* y;
    int64_t ldy;          // elements
    float* partials;      // [col_blocks][split][MR][256]
    uint32_t* tickets;    // [col_blocks], zero between launches
    int32_t N, K;
    int32_t k_tiles;
    int32_t col_blocks;
    int32_t out_kind;     // 0: fp32, 1: bf16, 2: f16
    int32_t flags;        // GEMV_FLAG_B_IMMUTABLE
};

template <int MR, int STAGES>
struct GemvRowsSmem {
    static constexpr uint32_t TILE_BYTES = GEMV_TILE_K * GEMV_COLS * 2;
    static constexpr uint32_t X_BYTES = MR * GEMV_TILE_K * 2;                   // per stage: MR rows of 64 activations
    static constexpr uint32_t X_OFF = STAGES * TILE_BYTES;
    static constexpr uint32_t RED_OFF = X_OFF + STAGES * 512;                   // 512 >= X_BYTES, keeps 128-byte alignment
    static constexpr uint32_t FLAG_OFF = RED_OFF + GEMV_CONSUMER_WARPS * GEMV_COLS * 4;
    static constexpr uint32_t BAR_OFF = FLAG_OFF + 16;
    static constexpr uint32_t TOTAL = BAR_OFF + 2 * STAGES * 8 + 128;
};

template <int MR, bool F16>
__global__ void __launch_bounds__(GEMV_TMA_THREADS, 2)
gemv_rows_kernel(const __grid_constant__ CUtensorMap tmap_b, const __grid_constant__ CUtensorMap tmap_x,
                 const GemvRowsParams p) {
    constexpr int STAGES = 3;
    using L = GemvRowsSmem<MR, STAGES>;
    constexpr int TILE_K = GEMV_TILE_K, RPW = TILE_K / GEMV_CONSUMER_WARPS;   // 8 rows of a tile per consumer warp
    static_assert(MR >= 2 && MR <= 4 && RPW == 8, "2..4 activation rows, 64-row tiles");
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    float* red = reinterpret_cast<float*>(smem_gen + L::RED_OFF);
    volatile uint32_t* s_last = reinterpret_cast<volatile uint32_t*>(smem_gen + L::FLAG_OFF);
    auto full_bar = [&](uint32_t s) { return smem_base + L::BAR_OFF + s * 8u; };
    auto empty_bar = [&](uint32_t s) { return smem_base + L::BAR_OFF + (STAGES + s) * 8u; };

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const int S = (int)gridDim.y, slice = (int)blockIdx.y;
    const int KT = p.k_tiles;

    if (threadIdx.x == 0) {
        prefetch_tmap(&tmap_b);
        prefetch_tmap(&tmap_x);
        for (uint32_t s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), GEMV_CONSUMER_WARPS);
        }
        fence_mbar_init();
    }
    __syncthreads();
    griddep_launch_dependents();

    if (warp == GEMV_CONSUMER_WARPS) {
        // ===== producer =====
        if (elect_one()) {
            constexpr uint32_t TX = L::TILE_BYTES + L::X_BYTES;   // full boxes, even when clipped
            auto issue_b = [&](uint32_t st, int cb, int kt) {
                mbar_arrive_expect_tx(full_bar(st), TX);
                tma_load_2d(smem_base + st * L::TILE_BYTES, &tmap_b, full_bar(st), cb * GEMV_COLS, kt * TILE_K);
            };
            auto issue_x = [&](uint32_t st, int kt) {
                tma_load_2d(smem_base + L::X_OFF + st * 512u, &tmap_x, full_bar(st), kt * TILE_K, 0);
            };
            auto next_unit = [&](int& cb, int& kt) {
                kt += S;
                if (kt >= KT) { kt = slice; cb += (int)gridDim.x; }
            };
            int cb = (int)blockIdx.x, kt = slice;
            uint32_t stage = 0, phase = 0;
            if ((p.flags & GEMV_FLAG_B_IMMUTABLE) && cb < p.col_blocks && kt < KT) {
                // weights first: the ring fills while the previous kernel drains; the activations (which
                // that kernel may have written) follow the dependency wait
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

    // ===== consumers: warp w owns rows 8w .. 8w+7 of every tile, lane l columns 8l .. 8l+7 =====
    griddep_wait();   // y and the workspace may still be in the previous kernel's use
    const uint32_t tid = threadIdx.x;   // 0..255
    uint32_t stage = 0, phase = 0;
    for (int cb = (int)blockIdx.x; cb < p.col_blocks; cb += (int)gridDim.x) {
        float acc[MR][8];
#pragma unroll
        for (int m = 0; m < MR; ++m)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[m][e] = 0.f;
        for (int kt = slice; kt < KT; kt += S) {
            mbar_wait(full_bar(stage), phase);
            const uint8_t* tile = smem_gen + stage * L::TILE_BYTES + warp * RPW * (GEMV_COLS * 2) + lane * 16u;
            const uint8_t* xs = smem_gen + L::X_OFF + stage * 512u + warp * RPW * 2;
            uint4 w[RPW], xq[MR];
#pragma unroll
            for (int r = 0; r < RPW; ++r) w[r] = *reinterpret_cast<const uint4*>(tile + r * (GEMV_COLS * 2));
#pragma unroll
            for (int m = 0; m < MR; ++m) xq[m] = *reinterpret_cast<const uint4*>(xs + m * (TILE_K * 2));   // broadcast: 8 activations
#pragma unroll
            for (int r = 0; r < RPW; ++r) {
                // unpack the row's 8 weights once, use them for every activation row
                const uint32_t u[4] = {w[r].x, w[r].y, w[r].z, w[r].w};
                float wf[8];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    wf[2 * i] = in_bits_to_f32<F16>((uint16_t)(u[i] & 0xffffu));
                    wf[2 * i + 1] = in_bits_to_f32<F16>((uint16_t)(u[i] >> 16));
                }
#pragma unroll
                for (int m = 0; m < MR; ++m) {
                    const uint32_t xv[4] = {xq[m].x, xq[m].y, xq[m].z, xq[m].w};
                    const uint16_t xb = (uint16_t)((r & 1) ? (xv[r >> 1] >> 16) : (xv[r >> 1] & 0xffffu));
                    const float xr = in_bits_to_f32<F16>(xb);
#pragma unroll
                    for (int e = 0; e < 8; ++e) acc[m][e] = fmaf(wf[e], xr, acc[m][e]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        // ---- column block done for this slice: warps -> CTA (row by row through `red`), then slices ----
        float s[MR];
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            float4* r4 = reinterpret_cast<float4*>(red + warp * GEMV_COLS + lane * 8);
            r4[0] = make_float4(acc[m][0], acc[m][1], acc[m][2], acc[m][3]);
            r4[1] = make_float4(acc[m][4], acc[m][5], acc[m][6], acc[m][7]);
            consumer_bar_sync();
            s[m] = 0.f;
#pragma unroll
            for (int w8 = 0; w8 < GEMV_CONSUMER_WARPS; ++w8) s[m] += red[w8 * GEMV_COLS + tid];   // fixed order
            consumer_bar_sync();
        }
        bool store = (S == 1);
        if (!store) {
            float* part = p.partials + (size_t)cb * S * MR * GEMV_COLS + tid;
#pragma unroll
            for (int m = 0; m < MR; ++m) st_cg_f32(part + ((size_t)slice * MR + m) * GEMV_COLS, s[m]);
            __threadfence();
            consumer_bar_sync();
            if (tid == 0) {
                const uint32_t old = atomicAdd(p.tickets + cb, 1u);
                const bool last = (old == (uint32_t)(S - 1));
                if (last) p.tickets[cb] = 0u;   // every slice has arrived: re-arm for the next launch
                *s_last = last ? 1u : 0u;
            }
            consumer_bar_sync();
            if (*s_last) {
                __threadfence();
#pragma unroll
                for (int m = 0; m < MR; ++m) {
                    s[m] = 0.f;
                    for (int q = 0; q < S; ++q) s[m] += ld_cg_f32(part + ((size_t)q * MR + m) * GEMV_COLS);   // fixed order
                }
                store = true;
            }
        }
        if (store) {
            const int col = cb * GEMV_COLS + (int)tid;
            if (col < p.N) {
#pragma unroll
                for (int m = 0; m < MR; ++m) {
                    if (p.out_kind == 0) reinterpret_cast<float*>(p.y)[(int64_t)m * p.ldy + col] = s[m];
                    else if (p.out_kind == 1) reinterpret_cast<uint16_t*>(p.y)[(int64_t)m * p.ldy + col] = f32_to_bf16_rne(s[m]);
                    else reinterpret_cast<uint16_t*>(p.y)[(int64_t)m * p.ldy + col] = __half_as_ushort(__float2half_rn(s[m]));
                }
            }
        }
        consumer_bar_sync();   // red and s_last are free for the next column block
    }
}

}  // namespace tg
