// Persistent, warp-specialised tcgen05 GEMM for sm_100a:  C = A * B, bf16 in, fp32 accumulate.
//
// What it computes: Listing 2 of the paper -- for each owned output tile,
// zero accumulator, sum over all K tiles of mma(x[bid_m,k], y[k,bid_n]), one store.  The
// schedule below is this build's own (the paper's tile shapes are not printed):
//
//   * one CTA (CG=1) or one CTA pair (CG=2, cta_group::2) owns exactly one output tile at a
//     time; tile -> owner is the pure function `tile_coords` + round-robin over clusters
//     ("each sub-tensor has exactly one owner");
//   * warp 0 : TMA producer  -- A box 64(k) x 128(m), B boxes 64(n) x 64(k), 128B swizzle,
//              out-of-bounds elements arrive as zeros (edge tiles), so the K loop
//              carries no bounds checks at all;
//   * warp 1 : MMA issuer    -- one thread, tcgen05.mma kind::f16 (bf16 x bf16 -> fp32 in TMEM),
//              A K-major, B MN-major (row-major K x N), tcgen05.commit frees smem stages;
//   * warp 2 : TMEM allocator (2 accumulator stages of BN columns);
//   * warps 4-11: epilogue   -- tcgen05.ld TMEM -> registers -> (fp32 | RNE bf16) -> swizzled smem
//              -> TMA store (clipped at M,N by the tensor map) or, when C is not 16-byte
//              addressable, clipped st.global from the staged tile.
//   TMEM holds two accumulator slots of BN columns.  NACC = 1: a tile is one slot wide and the
//   slots alternate, so tile i's epilogue overlaps tile i+1's main loop.  NACC = 2: a tile is both
//   slots wide (BM*CG x 2*BN, e.g. 256 x 512 for a CTA pair): every A stage feeds two MMAs, which
//   cuts the L2 -> shared-memory fill traffic per FLOP by a quarter (the kernel is power bound on
//   B200); each slot keeps its own full/empty barriers, so the next tile's
//   main loop restarts on slot 0 while the epilogue still drains slot 1.
//   MC = 1 (CTA pairs only): a cluster is TWO pairs, one tile row above the other, working on the same
//   tile column in step.  They need the same B panel, so each CTA fetches only every other 64-column
//   box of its B half and TMA multicasts it into its own shared memory and that of the CTA of the same
//   rank in the other pair: a third less L2 -> SM traffic per FLOP (the kernel is power bound).  A stage
//   is refilled only when BOTH pairs' MMAs have released it (every commit arrives at all four CTAs).
#pragma once
#include "ptx.cuh"

namespace tg {

constexpr int GEMM_BM = 128;      // rows per CTA (UMMA M = 128 * CG)
constexpr int GEMM_BK = 64;       // one 128-byte swizzle row of bf16
constexpr int GEMM_UMMA_K = 16;   // K per tcgen05.mma for 16-bit inputs
constexpr int GEMM_THREADS = 384;     // 4 control warps + 8 epilogue warps
constexpr int GEMM_EPI_WARP0 = 4;
constexpr uint32_t GEMM_EPI_BUF_BYTES = 2 * 32 * 64;   // per epilogue warp: two buffers of 32 rows x 64 B
constexpr uint32_t GEMM_PEER_BIT_MASK = 0xFEFFFFFFu;   // a shared-memory address with the bit that tells the two CTAs of a pair apart cleared
constexpr uint64_t GEMM_LOCKSTEP_PATIENCE_NS = 500000;  // a lockstep producer waits this long for the others (a window is ~30 us), then runs free

struct GemmParams {
    int32_t M, N, K;
    int32_t tiles_m, tiles_n;   // tile grid; a tile is (GEMM_BM*CG) x (BN*NACC)
    int32_t group_m;            // raster group height in tiles
    int32_t num_k_tiles;
    int32_t out_16;             // 0: fp32 C, 1: 16-bit C (bf16, or f16 when out_f16)
    int32_t out_f16;            // 16-bit C is IEEE binary16 instead of bf16
    int32_t in_f16;             // A and B are IEEE binary16 instead of bf16 (PAPER.md:300 measures f16)
    int32_t tma_store;          // 1: TMA store, 0: clipped st.global
    int32_t owner_mode;         // debug: write (tile << 8 | cta) instead of values
    void* C;
    int64_t ldc;                // elements
    // lockstep (large problems): the producers of all clusters advance through the schedule in
    // windows of `sync_window` k-tiles; a producer may run at most one window ahead of the slowest
    // cluster.  Co-running tiles then read the same k-slices of their shared A/B panels within a
    // window the L2 holds, instead of drifting apart over a long launch.  sync == nullptr: off.
    uint32_t* sync;             // [windows] arrival counters, zero at launch
    int32_t sync_window;
    int32_t sync_rounds;        // lockstep covers the first sync_rounds units of every cluster (all whole tiles)
    // Split-K for the last, partial wave (and for problems smaller than one wave): work units
    // [0, full_units) are whole tiles; the remaining tiles are cut into `split` slices of `kps`
    // k-tiles each, one unit per slice.  A slice's fp32 accumulators go to `partials`; the CTA that
    // draws the last of a tile's `split` tickets adds the slices in slice order (fixed order:
    // bitwise reproducible) and stores C.  split == 0: every unit is a whole tile.
    int32_t full_units, split, kps, total_units;
    int32_t a_rows;             // rows of the A box (16, 32, 64 or 128): for M <= 64 the rows past it are never loaded; the
                                // MMA reads whatever the stage holds there and those output rows are clipped
    int32_t up_offset;          // SwiGLU epilogue: column of B where the `up` half starts (= N, the width of C)
    float* partials;            // [split tiles][split][CG][8 warps][units][8 chunks][32 lanes][4 floats]
    uint32_t* tickets;          // [split tiles][CG], zero between launches
    // debug (tile_gemm_debug_trace): cluster c writes record c of 8 words -- [0] unused, clock cycles the MMA issuer
    // [1] waited for accumulator slots (once per tile), [2] spent in its loop in total, [3] k-tiles it issued; [4] cycles one
    // epilogue warp spent between "accumulator full" and "slot handed back" summed over its [5] tiles
    unsigned long long* trace;
    int32_t trace_cap;          // clusters that fit the trace buffer
};

// Work unit -> (tile, k-tile range, slice); slice < 0: a whole tile.  Pure function, all roles
// evaluate it identically.
struct GemmUnit {
    int t, k0, k1, slice;
};
template <bool SPLIT>
__device__ __forceinline__ GemmUnit gemm_unit(const GemmParams& p, int u) {
    GemmUnit r;
    if (!SPLIT || u < p.full_units) {
        r.t = u; r.k0 = 0; r.k1 = p.num_k_tiles; r.slice = -1;
    } else {
        const int v = u - p.full_units;
        r.t = p.full_units + v / p.split;
        r.slice = v - (v / p.split) * p.split;
        r.k0 = r.slice * p.kps;
        r.k1 = min(p.num_k_tiles, r.k0 + p.kps);
    }
    return r;
}
__device__ __forceinline__ float4 ld_cg_f4(const float* p) {
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_cg_f4(float* p, float a, float b, float c, float d) {
    asm volatile("st.global.cg.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ uint32_t ld_relaxed_gpu_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_add_relaxed_gpu_u32(uint32_t* p, uint32_t v) {
    asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Tile index -> tile coordinates.  Grouped raster: tiles are numbered down the rows of a
// group of `group_m` tile rows, then across columns, so that concurrently running tiles share
// A row panels and B column panels in L2.  Pure function, also evaluated on the host.
__host__ __device__ __forceinline__ void tile_coords(int t, int tiles_m, int tiles_n, int group_m, int& tm,
                                                     int& tn) {
    const int per_group = group_m * tiles_n;
    const int g = t / per_group;
    const int first_m = g * group_m;
    const int rows = (tiles_m - first_m) < group_m ? (tiles_m - first_m) : group_m;
    const int r = t - g * per_group;
    tm = first_m + r % rows;
    tn = r / rows;
}

template <int CG, int BN, int STAGES, int NACC>
struct GemmSmem {
    static constexpr uint32_t A_BYTES = GEMM_BM * GEMM_BK * 2;
    static constexpr uint32_t B_COLS = BN / CG;                 // B columns per accumulator slot loaded by each CTA
    static constexpr uint32_t B_BOXES = B_COLS / 64;
    static constexpr uint32_t B_BOX_BYTES = 64 * GEMM_BK * 2;   // 64 k-rows x 128 B
    static constexpr uint32_t B_ACC_BYTES = B_BOXES * B_BOX_BYTES;
    static constexpr uint32_t B_BYTES = NACC * B_ACC_BYTES;
    static constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr uint32_t EPI_OFF = STAGES * STAGE_BYTES;
    static constexpr uint32_t EPI_BYTES = 8 * GEMM_EPI_BUF_BYTES;
    static constexpr uint32_t BAR_OFF = EPI_OFF + EPI_BYTES;
    static constexpr uint32_t NUM_BARS = 2 * STAGES + 4;
    static constexpr uint32_t TMEM_PTR_OFF = BAR_OFF + NUM_BARS * 8;
    static constexpr uint32_t LAST_FLAG_OFF = TMEM_PTR_OFF + 8;   // split-K: "this CTA drew the last ticket"
    static constexpr uint32_t TOTAL = TMEM_PTR_OFF + 16 + 1024;   // + slack for 1024 B alignment
};

// SPLIT = false: every unit is a whole tile (the split-K epilogue is not even compiled in: it costs
// the hot epilogue registers); SPLIT = true: launches whose last wave is cut into K slices.
// EPI = 1 (needs NACC == 2): the SwiGLU epilogue of a fused gate/up projection.  B is K x 2N,
// [gate | up]; accumulator slot 0 takes the tile's gate columns, slot 1 the same columns of `up`
// (p.up_offset further right in B); the epilogue stores round_out(silu(gate) * up): the tile is
// BM*CG x BN, and the 2N-wide intermediate never reaches memory.
template <int CG, int BN, int STAGES, int NACC, bool SPLIT, int EPI = 0, int MC = 0>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                    const __grid_constant__ CUtensorMap tmap_c, const GemmParams p) {
    using L = GemmSmem<CG, BN, STAGES, NACC>;
    static_assert(CG == 1 || CG == 2, "cta_group is 1 or 2");
    static_assert(BN == 128 || BN == 256, "accumulator width");
    static_assert(NACC == 1 || NACC == 2, "a tile is one or two accumulator slots wide");
    constexpr bool SWIGLU = (EPI == 1);
    static_assert(!SWIGLU || (NACC == 2 && !SPLIT), "the SwiGLU epilogue pairs the two accumulator slots of a whole tile");
    static_assert(MC == 0 || (CG == 2 && !SPLIT), "B multicast joins two CTA pairs working on whole tiles");
    constexpr int TILE_N = SWIGLU ? BN : BN * NACC;   // width of the OUTPUT tile
    static_assert(L::TOTAL <= 232448, "exceeds 227 KB of shared memory");

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t crank = (CG == 2) ? cluster_ctarank() : 0u;    // rank in the cluster: 0..1, with MC 0..3
    const uint32_t rank = crank & 1u;                             // rank in the CTA pair (the pair's leader is 0)
    const uint32_t pair = MC ? (crank >> 1) : 0u;                 // MC: which of the cluster's two pairs = which of the unit's two tile rows
    const uint32_t lead = pair * 2u;                              // cluster rank of this pair's leader
    const int first_tile = (CG == 2) ? (int)cluster_id_x() : (int)blockIdx.x;
    const int tile_stride = (CG == 2) ? (int)num_clusters_x() : (int)gridDim.x;
    const int total_units = p.total_units;

    const uint32_t bar_base = smem_base + L::BAR_OFF;
    auto full_bar = [&](uint32_t s) { return bar_base + s * 8u; };
    auto empty_bar = [&](uint32_t s) { return bar_base + (STAGES + s) * 8u; };
    auto tmem_full_bar = [&](uint32_t a) { return bar_base + (2 * STAGES + a) * 8u; };
    auto tmem_empty_bar = [&](uint32_t a) { return bar_base + (2 * STAGES + 2 + a) * 8u; };
    volatile uint32_t* tmem_ptr_gen = reinterpret_cast<volatile uint32_t*>(smem_gen + L::TMEM_PTR_OFF);

    // ------------------------------------------------------------------ one-time setup
    if (warp == 0 && elect_one()) {
        prefetch_tmap(&tmap_a);
        prefetch_tmap(&tmap_b);
        prefetch_tmap(&tmap_c);
    }
    if (warp == 1 && elect_one()) {
        for (uint32_t s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);    // producer's arrive.expect_tx (+ TMA transaction bytes)
            mbar_init(empty_bar(s), MC ? 2 : 1);   // one tcgen05.commit per pair that reads the stage
        }
        for (uint32_t a = 0; a < 2; ++a) {
            mbar_init(tmem_full_bar(a), 1);           // one tcgen05.commit
            // lane 0 of every epilogue warp of the pair that drains this slot
            mbar_init(tmem_empty_bar(a), ((NACC == 2 && !SWIGLU) ? 4 : 8) * CG);
        }
        fence_mbar_init();
    }
    if (warp == 2) {
        tmem_alloc<CG>(smem_base + L::TMEM_PTR_OFF, 2 * BN);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr_gen;
    // programmatic dependent launch: this kernel's set-up above overlapped the previous kernel's
    // tail; every role waits for that kernel before its first global access, and the next kernel may
    // start its own set-up as our CTAs retire
    griddep_launch_dependents();

    // ------------------------------------------------------------------ warp roles
    if (warp == 0) {
        // ===== TMA producer (one lane) =====
        if (elect_one()) {
            uint32_t stage = 0, phase = 0;
            // lockstep bookkeeping (leader CTA of each cluster only; its partner is held back by the
            // shared pipeline): `pos` counts the k-tiles this cluster has issued over all its tiles
            const bool lockstep = p.sync != nullptr && crank == 0;
            // Lockstep is a locality hint, never a correctness condition: if the clusters this one
            // waits for do not show up in time (not co-resident: another kernel holds SMs, a MIG
            // slice, ...) it stops waiting for the rest of the launch and only keeps counting itself
            // in, so that nobody else waits for it.  The MMA order per tile does not change.
            bool lock_wait = lockstep;
            // the first sync_rounds units of every cluster are whole tiles: positions below sync_limit
            // exist in every cluster's schedule, so every window counter there reaches the cluster count
            const uint32_t sync_limit = (uint32_t)p.sync_rounds * (uint32_t)p.num_k_tiles;
            uint32_t pos = 0, next_sync = 0;
            const uint32_t stage_tx = (uint32_t)p.a_rows * (GEMM_BK * 2) + L::B_BYTES;   // bytes one CTA's boxes deliver per stage
            const int slot_stride = SWIGLU ? p.up_offset : BN;   // B column distance between the two accumulator slots
            griddep_wait();   // A, B (and the lockstep counters) may be the previous kernel's output
            for (int u = first_tile; u < total_units; u += tile_stride) {
                const GemmUnit un = gemm_unit<SPLIT>(p, u);
                int tm, tn;
                tile_coords(un.t, p.tiles_m, p.tiles_n, p.group_m, tm, tn);
                if constexpr (MC != 0) tm = tm * 2 + (int)pair;   // a unit is two tile rows, one per pair (a row past M is all zero fill)
                const int m0 = (tm * CG + (int)rank) * GEMM_BM;
                const int n0 = tn * TILE_N + (int)rank * (int)L::B_COLS;
                for (int kt = un.k0; kt < un.k1; ++kt, ++pos) {
                    if (lockstep && pos == next_sync && pos < sync_limit) {
                        const uint32_t w = pos / (uint32_t)p.sync_window;
                        red_add_relaxed_gpu_u32(p.sync + w, 1u);
                        if (w >= 1 && lock_wait) {   // every cluster must have entered window w-1
                            const uint64_t t0 = global_timer_ns();
                            uint32_t spins = 0;
                            while (ld_relaxed_gpu_u32(p.sync + (w - 1)) < (uint32_t)tile_stride) {
                                __nanosleep(64);
                                if ((++spins & 31u) == 0 && global_timer_ns() - t0 > GEMM_LOCKSTEP_PATIENCE_NS) {
                                    lock_wait = false;
                                    break;
                                }
                            }
                        }
                        next_sync += (uint32_t)p.sync_window;
                    }
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = smem_base + stage * L::STAGE_BYTES;
                    const uint32_t sb = sa + L::A_BYTES;
                    const int k0 = kt * GEMM_BK;
                    if constexpr (CG == 1) {
                        mbar_arrive_expect_tx(full_bar(stage), stage_tx);
                        tma_load_2d(sa, &tmap_a, full_bar(stage), k0, m0);
#pragma unroll
                        for (uint32_t j = 0; j < (uint32_t)NACC; ++j)
#pragma unroll
                            for (uint32_t b = 0; b < L::B_BOXES; ++b)
                                tma_load_2d(sb + j * L::B_ACC_BYTES + b * L::B_BOX_BYTES, &tmap_b, full_bar(stage),
                                            n0 + (int)j * slot_stride + (int)b * 64, k0);
                    } else {
                        // both CTAs' bytes are counted on the pair leader's barrier: the address is this CTA's
                        // own barrier with the pair-peer bit cleared, which cta_group::2 resolves in every
                        // destination CTA to the even CTA of ITS pair
                        const uint32_t lead_bar = full_bar(stage) & GEMM_PEER_BIT_MASK;
                        if (rank == 0) mbar_arrive_expect_tx(full_bar(stage), 2 * stage_tx);
                        tma_load_2d_cg2(sa, &tmap_a, lead_bar, k0, m0);
#pragma unroll
                        for (uint32_t j = 0; j < (uint32_t)NACC; ++j)
#pragma unroll
                            for (uint32_t b = 0; b < L::B_BOXES; ++b) {
                                const uint32_t dst = sb + j * L::B_ACC_BYTES + b * L::B_BOX_BYTES;
                                const int c0 = n0 + (int)j * slot_stride + (int)b * 64;
                                if constexpr (MC != 0) {
                                    // every other box is this pair's to fetch, for both CTAs of rank `rank`
                                    if (((j * L::B_BOXES + b) & 1u) == pair)
                                        tma_load_2d_cg2_mc(dst, &tmap_b, lead_bar, c0, k0, (uint16_t)(0x5u << rank));
                                } else {
                                    tma_load_2d_cg2(dst, &tmap_b, lead_bar, c0, k0);
                                }
                            }
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===== MMA issuer (one lane of the leader CTA) =====
        if (rank == 0 && elect_one()) {
            // instruction descriptor: D=f32, A=B=bf16|f16, A K-major, B MN-major, N = BN, M = 128*CG
            // (A/B format field: 0 = f16, 1 = bf16; same kind::f16 instruction and rate)
            const uint32_t ab_fmt = p.in_f16 ? 0u : 1u;
            const uint32_t idesc = (1u << 4) | (ab_fmt << 7) | (ab_fmt << 10) | (0u << 15) | (1u << 16) |
                                   ((uint32_t)(BN >> 3) << 17) | ((uint32_t)((GEMM_BM * CG) >> 4) << 24);
            // smem descriptors (version 1, SWIZZLE_128B):
            //   A (K-major):  LBO unused (=1), SBO = 1024 B between 8-row groups
            //   B (MN-major): LBO = one 64-column box (8192 B), SBO = 1024 B between 8-k groups
            constexpr uint64_t desc_hi = (uint64_t(1) << 46) | (uint64_t(2) << 61);
            constexpr uint64_t a_desc_base = desc_hi | (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32);
            constexpr uint64_t b_desc_base =
                desc_hi | (uint64_t(L::B_BOX_BYTES >> 4) << 16) | (uint64_t(1024 >> 4) << 32);
            // slot use: NACC == 1 -> slot = tile iteration & 1 (phase flips every 2nd tile);
            //           NACC == 2 -> both slots every tile (phase flips every tile)
            uint32_t stage = 0, phase = 0, it = 0;
            const bool traced = p.trace != nullptr && first_tile < p.trace_cap;
            long long t_acc = 0, n_kt = 0;   // the trace touches the tile boundary only: the K loop below stays as it is
            const long long t_begin = clock64();
            for (int u = first_tile; u < total_units; u += tile_stride, ++it) {
                const GemmUnit un = gemm_unit<SPLIT>(p, u);
                const uint32_t slot0 = (NACC == 2) ? 0u : (it & 1u);
                const uint32_t acc_phase = (NACC == 2) ? (it & 1u) : ((it >> 1) & 1u);
                n_kt += un.k1 - un.k0;
                for (int kt = un.k0; kt < un.k1; ++kt) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = smem_base + stage * L::STAGE_BYTES;
                    const uint32_t sb = sa + L::A_BYTES;
                    const uint64_t a_desc = a_desc_base | (uint64_t)((sa & 0x3FFFFu) >> 4);
#pragma unroll
                    for (uint32_t j = 0; j < (uint32_t)NACC; ++j) {
                        if (kt == un.k0) {   // the epilogue must have drained this slot
                            const long long t0 = traced ? clock64() : 0;
                            mbar_wait(tmem_empty_bar(slot0 + j), acc_phase ^ 1u);
                            if (traced) t_acc += clock64() - t0;
                            tc_fence_after();
                        }
                        const uint32_t d_tmem = tmem_base + (slot0 + j) * BN;
                        const uint64_t b_desc =
                            b_desc_base | (uint64_t)(((sb + j * L::B_ACC_BYTES) & 0x3FFFFu) >> 4);
#pragma unroll
                        for (int k = 0; k < GEMM_BK / GEMM_UMMA_K; ++k) {
                            // A: +16 elements along K = +32 B inside the swizzled row;
                            // B: +16 k-rows of 128 B = +2048 B
                            umma_bf16<CG>(d_tmem, a_desc + (uint64_t)(k * 2), b_desc + (uint64_t)(k * 128), idesc,
                                          (uint32_t)((kt != un.k0) | (k != 0)));
                        }
                        // accumulator slot ready for the epilogue after the last k-tile
                        if (kt == un.k1 - 1) umma_commit<CG>(tmem_full_bar(slot0 + j), (uint16_t)(3u << lead));
                    }
                    // smem stage reusable once these MMAs retire (MC: told to all four CTAs, the other pair multicasts into ours)
                    umma_commit<CG>(empty_bar(stage), MC ? (uint16_t)0xF : (uint16_t)3);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                if (p.num_k_tiles == 0) {   // owner-map mode: no MMAs, hand the slots over directly
#pragma unroll
                    for (uint32_t j = 0; j < (uint32_t)NACC; ++j) {
                        mbar_wait(tmem_empty_bar(slot0 + j), acc_phase ^ 1u);
                        umma_commit<CG>(tmem_full_bar(slot0 + j), (uint16_t)(3u << lead));
                    }
                }
            }
            if (traced) {
                unsigned long long* rec = p.trace + (size_t)first_tile * 8;
                rec[0] = 0ull;
                rec[1] = (unsigned long long)t_acc;
                rec[2] = (unsigned long long)(clock64() - t_begin);
                rec[3] = (unsigned long long)n_kt;
            }
        }
        __syncwarp();
    } else if (warp >= GEMM_EPI_WARP0) {
        // ===== epilogue: TMEM -> registers -> smem -> global =====
        // Eight warps: warp e drains TMEM lane quarter (e & 3) -- the only lanes it may address --
        // and column half (e >> 2) of the tile (NACC == 2: accumulator slot e >> 2).  The columns
        // are walked in units of 32 (one tcgen05.ld.32x32b.x32); the load of unit u+1 is in
        // flight while unit u is converted and staged; 64 bytes of C per row (one sub-chunk: 16 fp32
        // or 32 bf16 columns) are staged 64B-swizzled and leave with one TMA store, double buffered.
        const uint32_t ew = warp - GEMM_EPI_WARP0;
        const uint32_t q = ew & 3u;
        const uint32_t half = ew >> 2;
        constexpr int WARP_COLS = TILE_N / 2;
        constexpr int UNITS = WARP_COLS / 32;
        // staging: two 2 KB buffers per warp, each 32 rows x 64 B, 64B-swizzled (16-byte slot c of row r
        // sits at slot c ^ ((r >> 1) & 3): conflict-free st.shared.v4 and the layout the C tensor map expects)
        const uint32_t sbuf0 = smem_base + L::EPI_OFF + ew * GEMM_EPI_BUF_BYTES;
        const uint8_t* sgen0 = smem_gen + L::EPI_OFF + ew * GEMM_EPI_BUF_BYTES;
        const uint32_t sw = (lane >> 1) & 3u;
        const int out_16 = p.out_16;
        const int out_f16 = p.out_f16;
        const int sub_cols = out_16 ? 32 : 16;              // 64 B of C per row per sub-chunk
        // TMA stores clip at 16-byte granularity along a row (measured on B200): when N is not a
        // multiple of 16 bytes of elements the sub-chunk containing column N-1 takes the clipped
        // st.global path so that C[i][N..] is never written.
        const bool ragged_n = (p.N % (out_16 ? 8 : 4)) != 0;
        uint32_t it = 0, buf = 0;
        const bool dbg = p.trace != nullptr && first_tile < p.trace_cap && rank == 0 && ew == 4;   // tile_gemm_debug_trace: one warp per cluster
        long long dbg_drain = 0;
        volatile uint32_t* last_flag = reinterpret_cast<volatile uint32_t*>(smem_gen + L::LAST_FLAG_OFF);
        griddep_wait();   // C, the partials and the tickets may still be in the previous kernel's use
        for (int u_idx = first_tile; u_idx < total_units; u_idx += tile_stride, ++it) {
            const GemmUnit un = gemm_unit<SPLIT>(p, u_idx);
            const int t = un.t;
            int tm, tn;
            tile_coords(t, p.tiles_m, p.tiles_n, p.group_m, tm, tn);
            if constexpr (MC != 0) tm = tm * 2 + (int)pair;
            const int m0 = (tm * CG + (int)rank) * GEMM_BM + (int)q * 32;    // first row of this warp
            const int n_base = tn * TILE_N + (int)half * WARP_COLS;         // first column of this warp
            const uint32_t owner_val = ((uint32_t)t << 8) | (uint32_t)blockIdx.x;
            const uint32_t acc = (NACC == 2) ? half : (it & 1u);
            const uint32_t acc_phase = (NACC == 2) ? (it & 1u) : ((it >> 1) & 1u);
            const uint32_t t_acc = SWIGLU ? tmem_base + ((q * 32u) << 16) + half * (uint32_t)WARP_COLS   // gate; up is BN further
                                          : tmem_base + ((q * 32u) << 16) + acc * BN +
                                                ((NACC == 2) ? 0u : half * (uint32_t)WARP_COLS);
            // units of this warp that intersect C (warp-uniform); the rest is never loaded or stored
            int units = 0;
            if (m0 < p.M && n_base < p.N) {
                units = (p.N - n_base + 31) >> 5;
                if (units > UNITS) units = UNITS;
            }
            if constexpr (SWIGLU) {   // this warp reads the same columns of both slots
                mbar_wait_sleep(tmem_full_bar(0), acc_phase);
                mbar_wait_sleep(tmem_full_bar(1), acc_phase);
            } else {
                mbar_wait_sleep(tmem_full_bar(acc), acc_phase);
            }
            tc_fence_after();
            const long long dbg_t0 = dbg ? clock64() : 0;

            // stage 16 words (64 B) of this thread's row as columns [n0, n0 + sub_cols) and send them
            auto emit = [&](uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, uint32_t w4, uint32_t w5,
                            uint32_t w6, uint32_t w7, uint32_t w8, uint32_t w9, uint32_t w10, uint32_t w11,
                            uint32_t w12, uint32_t w13, uint32_t w14, uint32_t w15, int n0) {
                if (n0 >= p.N) return;                         // warp-uniform
                // the buffer written two sub-chunks ago must have been read by its TMA store
                if (lane == 0) tma_store_wait_read<1>();
                __syncwarp();
                const uint32_t sb = sbuf0 + buf * 2048u;
                const uint32_t ra = sb + lane * 64u;
                st_shared_v4(ra + ((0u ^ sw) << 4), w0, w1, w2, w3);
                st_shared_v4(ra + ((1u ^ sw) << 4), w4, w5, w6, w7);
                st_shared_v4(ra + ((2u ^ sw) << 4), w8, w9, w10, w11);
                st_shared_v4(ra + ((3u ^ sw) << 4), w12, w13, w14, w15);
                if (p.tma_store && !(ragged_n && n0 + sub_cols > p.N)) {
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        tma_store_2d(&tmap_c, sb, n0, m0);     // clipped at (N, M) by the tensor map
                        tma_store_commit();
                    }
                } else {
                    // C rows are not 16-byte addressable: clipped, row-coalesced stores from smem
                    __syncwarp();
                    const uint8_t* sg = sgen0 + buf * 2048u;
                    const int rows = (p.M - m0) < 32 ? (p.M - m0) : 32;
                    const int e = (int)lane;                   // column within the sub-chunk
                    if (out_16) {
                        uint16_t* Cb = reinterpret_cast<uint16_t*>(p.C);
                        if (n0 + e < p.N)
                            for (int r = 0; r < rows; ++r) {
                                const uint32_t off = (uint32_t)r * 64u +
                                                     ((((uint32_t)e >> 3) ^ (((uint32_t)r >> 1) & 3u)) << 4) +
                                                     ((uint32_t)e & 7u) * 2u;
                                Cb[(int64_t)(m0 + r) * p.ldc + n0 + e] = *reinterpret_cast<const uint16_t*>(sg + off);
                            }
                    } else {
                        uint32_t* Cf = reinterpret_cast<uint32_t*>(p.C);
                        // 16 columns per row: lanes 0-15 take even rows, lanes 16-31 odd rows
                        const int ec = e & 15;
                        if (n0 + ec < p.N)
                            for (int r = (e >> 4); r < rows; r += 2) {
                                const uint32_t off = (uint32_t)r * 64u +
                                                     ((((uint32_t)ec >> 2) ^ (((uint32_t)r >> 1) & 3u)) << 4) +
                                                     ((uint32_t)ec & 3u) * 4u;
                                Cf[(int64_t)(m0 + r) * p.ldc + n0 + ec] = *reinterpret_cast<const uint32_t*>(sg + off);
                            }
                    }
                    __syncwarp();
                    if (lane == 0) tma_store_commit();         // empty group: keeps wait_group.read<1> aligned
                }
                buf ^= 1u;
            };
            // one unit: `v` holds 32 consecutive columns of this thread's row
            auto stage_unit = [&](uint32_t (&v)[32], int u) {
                const int n0 = n_base + u * 32;
                if (out_16 && !out_f16) {
#define TG_PK(i) pack_bf16x2(__uint_as_float(v[2 * (i)]), __uint_as_float(v[2 * (i) + 1]))
                    emit(TG_PK(0), TG_PK(1), TG_PK(2), TG_PK(3), TG_PK(4), TG_PK(5), TG_PK(6), TG_PK(7), TG_PK(8),
                         TG_PK(9), TG_PK(10), TG_PK(11), TG_PK(12), TG_PK(13), TG_PK(14), TG_PK(15), n0);
#undef TG_PK
                } else if (out_16) {
#define TG_PK(i) pack_f16x2(__uint_as_float(v[2 * (i)]), __uint_as_float(v[2 * (i) + 1]))
                    emit(TG_PK(0), TG_PK(1), TG_PK(2), TG_PK(3), TG_PK(4), TG_PK(5), TG_PK(6), TG_PK(7), TG_PK(8),
                         TG_PK(9), TG_PK(10), TG_PK(11), TG_PK(12), TG_PK(13), TG_PK(14), TG_PK(15), n0);
#undef TG_PK
                } else {
                    if (p.owner_mode) {
#pragma unroll
                        for (int i = 0; i < 32; ++i) v[i] = owner_val;
                    }
                    emit(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7], v[8], v[9], v[10], v[11], v[12], v[13],
                         v[14], v[15], n0);
                    emit(v[16], v[17], v[18], v[19], v[20], v[21], v[22], v[23], v[24], v[25], v[26], v[27], v[28],
                         v[29], v[30], v[31], n0 + 16);
                }
            };
            // all TMEM reads of this accumulator slot are complete: hand it back to the MMA warp
            auto release_tmem = [&]() {
                if (dbg) dbg_drain += clock64() - dbg_t0;
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (SWIGLU) {
                        if constexpr (CG == 1) { mbar_arrive(tmem_empty_bar(0)); mbar_arrive(tmem_empty_bar(1)); }
                        else {
                            mbar_arrive_cluster_relaxed(map_to_cta(tmem_empty_bar(0), lead));
                            mbar_arrive_cluster_relaxed(map_to_cta(tmem_empty_bar(1), lead));
                        }
                    } else {
                        if constexpr (CG == 1) mbar_arrive(tmem_empty_bar(acc));
                        else mbar_arrive_cluster_relaxed(map_to_cta(tmem_empty_bar(acc), lead));
                    }
                }
            };

            uint32_t va[32], vb[32];
            if (SPLIT && un.slice >= 0) {
                // ---- one K slice of a split tile: park the fp32 accumulators, take a ticket; the CTA
                //      that draws the tile's last ticket adds all slices in slice order and stores C ----
                constexpr size_t WARP_FLOATS = (size_t)UNITS * 32 * 32;
                const int st = t - p.full_units;                      // index among the split tiles
                auto slot_of = [&](int slice) -> float* {
                    // per 32-column unit: [8 chunks][32 lanes][4 floats] -- a warp's st/ld.v4 covers 512 contiguous bytes
                    return p.partials + ((((size_t)st * p.split + slice) * CG + rank) * 8 + ew) * WARP_FLOATS + lane * 4;
                };
                float* mine = slot_of(un.slice);
                for (int uu = 0; uu < units; ++uu) {
                    tmem_ld_32x32(t_acc + (uint32_t)(uu * 32), va);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 32; i += 4)
                        st_cg_f4(mine + (size_t)uu * 1024 + i * 32, __uint_as_float(va[i]), __uint_as_float(va[i + 1]),
                                 __uint_as_float(va[i + 2]), __uint_as_float(va[i + 3]));
                }
                release_tmem();
                __threadfence();
                asm volatile("bar.sync 1, 256;" ::: "memory");        // the eight epilogue warps
                if (ew == 0 && lane == 0) {
                    uint32_t* tk = p.tickets + (size_t)st * CG + rank;
                    const uint32_t old = atomicAdd(tk, 1u);
                    const bool last = (old == (uint32_t)(p.split - 1));
                    if (last) *tk = 0u;                                 // every slice has arrived: re-arm
                    *last_flag = last ? 1u : 0u;
                }
                asm volatile("bar.sync 1, 256;" ::: "memory");
                const bool last = (*last_flag != 0u);
                asm volatile("bar.sync 1, 256;" ::: "memory");        // flag is free for the next unit
                if (last) {
                    __threadfence();
                    for (int uu = 0; uu < units; ++uu) {
#pragma unroll
                        for (int i = 0; i < 32; ++i) va[i] = 0u;        // +0.0f
                        for (int sl = 0; sl < p.split; ++sl) {          // fixed order
                            const float* src = slot_of(sl) + (size_t)uu * 1024;
#pragma unroll
                            for (int i = 0; i < 32; i += 4) {
                                const float4 f = ld_cg_f4(src + i * 32);
                                va[i] = __float_as_uint(__uint_as_float(va[i]) + f.x);
                                va[i + 1] = __float_as_uint(__uint_as_float(va[i + 1]) + f.y);
                                va[i + 2] = __float_as_uint(__uint_as_float(va[i + 2]) + f.z);
                                va[i + 3] = __float_as_uint(__uint_as_float(va[i + 3]) + f.w);
                            }
                        }
                        stage_unit(va, uu);
                    }
                }
                continue;
            }
            if constexpr (SWIGLU) {
                // h = silu(g) * u on the fp32 accumulators: g / (1 + e^-g) with ex2.approx and a fast
                // divide (relative error ~2^-21, far below the bf16/f16 output rounding)
                for (int uu = 0; uu < units; ++uu) {
                    tmem_ld_32x32(t_acc + (uint32_t)(uu * 32), va);
                    tmem_ld_32x32(t_acc + (uint32_t)(BN + uu * 32), vb);
                    tmem_ld_wait();
                    if (uu + 1 == units) release_tmem();
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        const float g = __uint_as_float(va[i]);
                        va[i] = __float_as_uint(__fdividef(g, 1.0f + __expf(-g)) * __uint_as_float(vb[i]));
                    }
                    stage_unit(va, uu);
                }
                if (units == 0) release_tmem();
                continue;
            }
            if (units > 0) tmem_ld_32x32(t_acc, va);
#pragma unroll 1
            for (int u = 0; u < units; u += 2) {
                tmem_ld_wait();                                            // va = unit u
                if (u + 1 < units) tmem_ld_32x32(t_acc + (uint32_t)((u + 1) * 32), vb);
                else release_tmem();
                stage_unit(va, u);
                if (u + 1 < units) {
                    tmem_ld_wait();                                        // vb = unit u + 1
                    if (u + 2 < units) tmem_ld_32x32(t_acc + (uint32_t)((u + 2) * 32), va);
                    else release_tmem();
                    stage_unit(vb, u + 1);
                }
            }
            if (units == 0) release_tmem();
        }
        if (dbg && lane == 0) {
            p.trace[(size_t)first_tile * 8 + 4] = (unsigned long long)dbg_drain;
            p.trace[(size_t)first_tile * 8 + 5] = (unsigned long long)it;
        }
        if (lane == 0) tma_store_wait_all<0>();
        __syncwarp();
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    if constexpr (CG == 2) cluster_sync(); else __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 2 * BN);
    }
}

}  // namespace tg
