/*
 * tile_gemm_debug.h -- the entries of libtilegemm.so that are NOT part of the contract in
 * tile_gemm.h: measurement probes, plan queries, test helpers and tuning overrides.  bench.py,
 * the tests and the profiling modules use them; a program that only computes needs none.
 *
 * Thread safety, in one sentence: the tuning keys and the trace buffer are process-global and
 * unsynchronised -- set them while no other thread is inside a library call, and expect every
 * thread's later launches to see them; the queries and probes are as thread-safe as tile_gemm.
 *
 * Conventions (status codes, streams, device pointers) are those of tile_gemm.h.
 */
#ifndef TILE_GEMM_DEBUG_H_
#define TILE_GEMM_DEBUG_H_

#include "tile_gemm.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Read-bandwidth probe of the measurement harness: adds the sum of
 * the n 32-bit words of `buf` (device, 16-byte aligned), taken as a 64-bit integer
 * modulo 2^64, to *out_sum (device, 8-byte aligned, not inside buf; the caller
 * zeroes it).  Integer arithmetic: exact and independent of the order.  Every word
 * is read exactly once with streaming 128-bit loads, one 32 KB tile per CTA: the
 * rate of this kernel on a buffer much larger than L2 is what a pure read of HBM
 * achieves on the box, the figure bench.py reports next to the GEMV's.
 * Errors: E_EXTENT, E_NULL, E_ALIGN, E_OVERFLOW (n > 2^40), E_ALIAS, E_DEVICE, E_CUDA.
 */
int tile_read_probe_u32(const uint32_t* buf, int64_t n, unsigned long long* out_sum, void* stream);

/*
 * Describes the tile configuration the GEMM path uses for a shape, so that a
 * host program can rebuild the owner map: out[0]=BM (rows per CTA),
 * out[1]=BN (columns per tile), out[2]=cta_group (1 or 2: CTAs per tile, tile
 * rows = BM*cta_group), out[3]=number of CTAs launched, out[4]=GROUP_M (tile
 * rows per raster group), out[5]=pipeline stages, out[6]=BK, out[7]=config id
 * (1..4; 6 = config 4 with two CTA pairs per cluster, tuning key 12: a work unit is then
 * two tile rows of one tile column, out[4] counts unit rows, and CTAs 4c..4c+3 own a unit).
 * Needs a CUDA device (SM count).  Returns a status code.
 */
int tile_gemm_query_config(int64_t M, int64_t N, int64_t K, int out_dtype, int32_t out[8]);

/*
 * What the selector does with a GEMM shape (M >= 2, operands assumed TMA-addressable)
 * beyond the tile configuration:
 * out[0] = config id (1..4: the tiled kernel's configurations; 5: the weight-streaming
 * tensor-core kernel of 2 <= M <= 64, one CTA per 128 columns and K slice),
 * out[1] = CTAs launched, out[2] = work units that are whole
 * tiles, out[3] = K slices per tile of the last, partial wave (config 5: per column
 * block; 0 = not cut), out[4] = k-tiles (of 64) per slice, out[5] = rounds the lockstep
 * producers cover (0 = off), out[6] = their window in k-tiles, out[7] = rows of the A box
 * (16, 32, 64 or 128: skinny M loads only the rows it has).  Needs a CUDA device (SM count).
 */
int tile_gemm_query_plan(int64_t M, int64_t N, int64_t K, int32_t out[8]);

/*
 * Test helper: `ctas` CTAs that each hold one SM (they ask for most of its shared memory) for `ns`
 * nanoseconds (<= 2e9) on `stream`, waiting for nothing but the clock.  Used to check that a
 * persistent GEMM whose CTAs cannot all be resident still completes (the lockstep producers give
 * up waiting for clusters that have not started).  Errors: E_EXTENT, E_OVERFLOW, E_DEVICE, E_CUDA.
 */
int tile_gemm_debug_occupy(int ctas, int64_t ns, void* stream);

/*
 * Timeline trace of the M = 1 kernel (gemv_split_kernel), for profiles/ (where a
 * bandwidth-bound launch loses time).  While `records` (DEVICE memory, 8-byte aligned, `capacity`
 * records of 8 x 64-bit words, owned by the caller) is set, CTA (bx, by) of every following launch
 * writes record by * gridDim.x + bx, when below capacity:
 *   [0] smid | bx << 16 | by << 32, then %globaltimer in ns at [1] kernel entry, [2] release of the
 *   dependency wait, [3] first tile in shared memory, [4] last tile consumed, [5] CTA done;
 *   [6] tiles consumed; [7] %globaltimer when this CTA's partial sums were handed over (split-K only).
 * The tiled GEMM kernel fills the same buffer while it is set: cluster c writes record c (when below
 * capacity): clock cycles its MMA issuer [1] waited for accumulator slots to be drained (taken once
 * per tile: the K loop itself is not touched), [2] spent in its loop in total, [3] k-tiles it issued;
 * [4] cycles one epilogue warp spent between "accumulator full" and "slot handed back", summed over
 * its [5] tiles; [0], [6], [7] unused.
 * Later launches overwrite earlier ones: point it at a fresh buffer per launch.  records == NULL
 * or capacity == 0 switches tracing off (one untaken branch per event).  Process-global like the
 * tuning keys.  Returns 0, E_EXTENT or E_ALIGN.
 */
int tile_gemm_debug_trace(unsigned long long* records, int64_t capacity);

/*
 * Tuning / test overrides, process-global, not thread-safe against concurrent
 * library calls; 0 always means "automatic".  Returns 0, or E_PATH for an unknown key.
 *   key 0  GEMM tile configuration: 1 = 1-CTA 128x128, 2 = 1-CTA 128x256, 3 = CTA pair
 *          256x256, 4 = CTA pair 256x512.
 *   key 1  GEMM GROUP_M: tile rows per raster group.
 *   key 2  maximum number of CTAs of a GEMM launch; also caps the GEMV grids.
 *   key 3  K slices: of the M = 1 kernel's column blocks, and (1 = never, >= 2 = that
 *          many) of the tiled GEMM's partial last wave.
 *   key 4  M = 1 kernel: 2 = 16-byte LDG, 3 = scalar LDG (both with a thread-block-cluster split-K; 3 is what
 *          weights that TMA cannot address get), 1 or 4 = TMA ring + interleaved split-K (the automatic
 *          choice when B is TMA-addressable).
 *   key 5  ring shape of the TMA-ring kernel {columns per CTA, rows per stage, stages, CTAs per SM}:
 *          2 = {256, 64, 3, 2} (automatic), 4 = {512, 32, 3, 2}, 6 = {512, 16, 4, 3}; other values mean 2
 *          (table kGemvShapes in csrc/tile_gemm.cu; the shapes that spilled were removed in round 3).
 *   key 6  flag bits: 0 = no programmatic dependent launch; 1 = kernel 4 reads x with global loads
 *          instead of through its TMA ring; 2 / 3 = GEMM lockstep producers forced on / off, bits
 *          8-15 = their window in k-tiles; 5 = full 128-row A box even for skinny M; 6 =
 *          tile_gemm_host in one shot instead of pipelined chunks.
 *   key 8  split-K hand-over of the M = 1 kernel (csrc/gemv_kernel.cuh): 1 = tickets only, 2 = tagged
 *          slots with a designated combiner where the launch fits the device, else tickets, 3 =
 *          thread-block cluster + DSMEM where the slice count is <= 8, else tickets; automatic =
 *          cluster, else tagged slots, else tickets.  All three add the partial sums in slice order.
 *   key 9  weight tiles the weight-streaming kernels send as far as L2 right behind the dependency
 *          wait (tile_gemm_static_b only): n >= 1 means n - 1 tiles; automatic = 2.
 *   key 10 automatic cluster size of the weight-streaming kernels: per cent of the occupancy
 *          calculator's resident-cluster figure that the column blocks may fill; automatic = 92.
 *   key 11 weight-streaming tensor-core kernel of 2 <= M <= 64: bits 0-3: 1 = never (the tiled
 *          kernel takes every GEMM shape), 2 = wherever it can run; bits 8-15 = K slices per
 *          column block (1..8); bits 16-23 = 32 or 64: an activation box of that many rows even for fewer;
 *          bits 24-27 = 3 or 4: ring stages (4 only up to 32 rows).
 *   key 12 config 4 with clusters of two CTA pairs that share each B stage through TMA multicast
 *          (csrc/gemm_kernel.cuh, MC = 1): 1 = never, 2 = whenever the shape has two tile rows and
 *          runs on config 4; automatic = never (measured slower on this part: clusters of four
 *          leave 16 of 148 SMs idle).  tile_gemm_query_config reports it as config 6.
 *   key 7  tile_add_f32 launch shape: bits 0-3 vectors per thread in {1,2,4,8}, bits 4-11 CTAs
 *          per SM (255 = one tile per CTA), bits 12-15 access mode (1 / 2 = 128-bit with / without
 *          streaming hints, 3 / 4 = 256-bit with / without).
 */
int tile_gemm_set_tuning(int key, int value);

#ifdef __cplusplus
}
#endif
#endif /* TILE_GEMM_DEBUG_H_ */
