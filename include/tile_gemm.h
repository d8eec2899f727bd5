/*
 * tile_gemm.h -- C ABI of libtilegemm.so: dense BF16 GEMM  C = A * B  with fp32
 * accumulation on one NVIDIA B200 (sm_100a), plus its M=1 decode GEMV and the
 * shape selector between them.
 *
 * Operation (Listing 2 "gemm_persistent"): z = x * y where z is
 * split into disjoint output tiles, each owned by exactly one tile program at a
 * time, x and y are shared read-only, the accumulator starts
 * at zero, all K tiles are summed and each
 * tile is stored once.  Edge tiles are legal: loads past the
 * tensor read as zero and stores past it are masked.  Every
 * shape / stride / pointer check is a *launch precondition*: it runs once at
 * this host entry before any work is queued and returns an error with its own
 * message; the device K loop contains no checks.
 *
 *     C[i*ldc + j] = round_out( sum_{k<K} A[i*lda + k] * B[k*ldb + j] )
 *
 * alpha = 1, beta = 0 (C is never read).  A is M x K and B is K x N, both
 * row-major bf16 (raw 16-bit patterns); products are exact, sums are carried in
 * fp32 in an unspecified but fixed order (results are bitwise reproducible run
 * to run for a given shape); round_out is identity for fp32 output and
 * round-to-nearest-even for bf16 output.  Only C[0..M) x [0..N) is written;
 * padding columns (j >= N when ldc > N) and everything else stay untouched.
 *
 * Conventions for every entry point below
 *   - lda, ldb, ldc are row strides in ELEMENTS (not bytes).
 *   - A, B, C are DEVICE pointers on the current CUDA device unless the entry
 *     says "host".  The caller owns them; the library keeps no reference after
 *     the work completes.  Calls are asynchronous: they return after enqueueing
 *     on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream)
 *     and never synchronise; buffers must stay valid until the stream reaches
 *     the work.  Internal state: a per-stream grow-only repack workspace and a
 *     tensor-map cache, both released by tile_gemm_shutdown().
 *   - Return value 0 = success; otherwise a TILE_GEMM_E_* code.  On any error
 *     nothing is enqueued and C is untouched.  tile_gemm_last_error() holds the
 *     detailed message of the calling thread's last failure.
 *   - No CPU fallback exists: on a machine without an sm_100 device compute
 *     entries fail with TILE_GEMM_E_DEVICE.
 *   - Degenerate extents (reading c8): M == 0 or N == 0 is a
 *     successful no-op; K == 0 writes zeros to C[0..M) x [0..N).
 *   - Base-pointer / stride alignment to 16 bytes is NOT a precondition: rows
 *     that TMA cannot address are first copied into an aligned workspace
 *     (TILE_GEMM_PATH_GEMM_REPACK) and misaligned C is written with clipped
 *     st.global stores from the epilogue.
 */
#ifndef TILE_GEMM_H_
#define TILE_GEMM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* out_dtype */
#define TILE_GEMM_OUT_F32 0
#define TILE_GEMM_OUT_BF16 1
#define TILE_GEMM_OUT_F16 2   /* IEEE binary16, RNE of the fp32 accumulator (tile_gemm_typed rows) */

/* in_dtype of tile_gemm_typed: element type of A and B */
#define TILE_GEMM_IN_BF16 0
#define TILE_GEMM_IN_F16 1    /* IEEE binary16: the precision the paper measures */

/* status codes */
#define TILE_GEMM_OK 0
#define TILE_GEMM_E_NULL 1        /* NULL A/B/C with a non-empty extent                    */
#define TILE_GEMM_E_EXTENT 2      /* negative M, N or K                                    */
#define TILE_GEMM_E_LDA 3         /* lda < K                                               */
#define TILE_GEMM_E_LDB 4         /* ldb < N                                               */
#define TILE_GEMM_E_LDC 5         /* ldc < N                                               */
#define TILE_GEMM_E_DTYPE 6       /* out_dtype is neither F32 nor BF16                     */
#define TILE_GEMM_E_ALIGN 7       /* A/B not 2-byte aligned, or C not element aligned      */
#define TILE_GEMM_E_ALIAS 8       /* C's byte range overlaps A's or B's      */
#define TILE_GEMM_E_OVERFLOW 9    /* byte offsets overflow int64 or tile counts int32      */
#define TILE_GEMM_E_DEVICE 10     /* no CUDA device, or the device is not sm_100           */
#define TILE_GEMM_E_CUDA 11       /* a CUDA runtime/driver call failed (code in message)   */
#define TILE_GEMM_E_PATH 12       /* force_path unknown or not applicable to this shape    */
#define TILE_GEMM_E_INTERNAL 13
#define TILE_GEMM_E_IN_DTYPE 14   /* in_dtype is neither BF16 nor F16                       */
#define TILE_GEMM_E_LIMIT 15      /* tile_gemv_no_alloc: the request needs more than its fixed scratch */
#define TILE_GEMM_NUM_STATUS 16

/* internal flag behind tile_gemm_static_b */
#define TILE_GEMM_FLAG_B_IMMUTABLE 1u

/* execution paths (what the selector returns / what force_path accepts) */
#define TILE_GEMM_PATH_AUTO 0         /* force_path only                                      */
#define TILE_GEMM_PATH_GEMM_TMA 1     /* tcgen05 GEMM, A and B read in place through TMA: the tiled
                                         persistent kernel, or for 2 <= M <= 64 the weight-streaming
                                         one (csrc/skinny_kernel.cuh); tile_gemm_query_plan (tile_gemm_debug.h) says which */
#define TILE_GEMM_PATH_GEMM_REPACK 2  /* same kernel after copying A and/or B to aligned rows */
#define TILE_GEMM_PATH_GEMV 3         /* M == 1 (any alignment): HBM-bound weight-streaming kernel on
                                         the CUDA cores                                       */
#define TILE_GEMM_PATH_ZERO 4         /* K == 0: C <- 0                                       */
#define TILE_GEMM_PATH_NOOP 5         /* M == 0 or N == 0                                     */

/*
 * The GEMM (Listing 2).  Validates, selects a path
 * (tile_gemm_select) and enqueues it on `stream`.
 */
int tile_gemm(const void* A, const void* B, void* C,
              int64_t M, int64_t N, int64_t K,
              int64_t lda, int64_t ldb, int64_t ldc,
              int out_dtype, void* stream);

/*
 * Same, with the path forced (tests / measurements): TILE_GEMM_PATH_AUTO,
 * _GEMM_TMA (fails with E_PATH when A or B is not TMA-addressable), _GEMM_REPACK
 * (always legal for K > 0) or _GEMV (requires M == 1).
 */
int tile_gemm_ex(const void* A, const void* B, void* C,
                 int64_t M, int64_t N, int64_t K,
                 int64_t lda, int64_t ldb, int64_t ldc,
                 int out_dtype, void* stream, int force_path);

/*
 * tile_gemm plus one promise from the caller: B holds weights -- no work that is
 * still in flight when this call's kernel starts (earlier in `stream` or on any
 * other stream) writes B.  The weight-streaming kernels (M == 1, and 2 <= M <= 64
 * with TMA-addressable operands) are launched with programmatic dependent launch
 * in either entry; with this promise they stream weight tiles
 * ahead of the wait on the previous kernel of the stream, so back-to-back
 * decode projections (a recorded decode step) keep HBM
 * busy across kernel boundaries.  A, C and every other rule are as in tile_gemm.
 */
int tile_gemm_static_b(const void* A, const void* B, void* C,
                       int64_t M, int64_t N, int64_t K,
                       int64_t lda, int64_t ldb, int64_t ldc,
                       int out_dtype, void* stream);

/*
 * The same GEMM with the element types spelled out (the paper's
 * own sweep, Figure 6b / PAPER.md:300, is in f16).  in_dtype = TILE_GEMM_IN_BF16
 * or TILE_GEMM_IN_F16 is the type of BOTH A and B (raw 16-bit patterns either
 * way); out_dtype = F32, BF16 or F16.  Same tensor-core instruction and rate for
 * both input types (tcgen05 kind::f16), fp32 accumulation, one RNE rounding of the
 * final accumulator for 16-bit outputs; all rules of tile_gemm apply, M == 1
 * included.  Errors: those of tile_gemm plus TILE_GEMM_E_IN_DTYPE.
 */
int tile_gemm_typed(const void* A, const void* B, void* C,
                    int64_t M, int64_t N, int64_t K,
                    int64_t lda, int64_t ldb, int64_t ldc,
                    int in_dtype, int out_dtype, void* stream);

/*
 * Fused gate/up projection with the SwiGLU epilogue (the MLP of
 * the Qwen3 engine the paper builds, PAPER.md:330-343 -- the paper names its fused
 * kernels around the projections without printing the formula, DESIGN.md c21):
 *     G = X * Wgu[:, 0..I),  U = X * Wgu[:, I..2I),
 *     H[i*ldh + j] = round_out( silu(G_ij) * U_ij ),  silu(g) = g / (1 + e^-g)
 * X: M x K bf16 (row stride ldx), Wgu: K x 2I bf16 (row stride ldw >= 2I), gate
 * columns first, then up; H: M x I, out_dtype F32, BF16 or F16 (row stride ldh).
 * Both projections accumulate in fp32 in tensor memory side by side; silu and the
 * product are evaluated in fp32 on the accumulators (fast exp and divide: relative
 * error about 2^-21) and rounded once; the 2I-wide intermediate never reaches
 * memory.  X and Wgu must be TMA-addressable (16-byte aligned base, ldx and ldw
 * multiples of 8) and I a multiple of 8 (the up half is fetched by TMA boxes that
 * start at column I, which the hardware wants on a 16-byte boundary): there is no
 * repack path here (TILE_GEMM_E_PATH otherwise).
 * K == 0 writes zeros.  All other rules and errors are tile_gemm's, with I in the
 * role of N for H and 2I for Wgu (E_LDB when ldw < 2I).
 */
int tile_gemm_swiglu(const void* X, const void* Wgu, void* H,
                     int64_t M, int64_t I, int64_t K,
                     int64_t ldx, int64_t ldw, int64_t ldh,
                     int out_dtype, void* stream);

/*
 * Element-wise add (Listing 1; measured at n = 2^28):
 *     z[i] = fl32(x[i] + y[i])   for i in [0, n)
 * one IEEE-754 binary32 addition per element (round to nearest even; NaN and
 * infinities as the hardware FADD produces them).  x, y, z: DEVICE pointers to n
 * contiguous floats, 4-byte aligned (16-byte aligned buffers take the 128-bit
 * path); z is exclusively owned: its byte range may not overlap x's or y's
 * (TILE_GEMM_E_ALIAS) while x and y may be the same buffer (shared
 * reads).  Only z[0..n) is written.  n == 0 is a successful no-op.  Errors:
 * E_EXTENT (n < 0), E_OVERFLOW (n > 2^40), E_NULL, E_ALIGN, E_ALIAS, E_DEVICE,
 * E_CUDA; nothing is enqueued on error.  Asynchronous on `stream`.  Launched with
 * programmatic dependent launch like every kernel of the library: a chain of
 * small adds overlaps each launch with its predecessor's execution.
 */
int tile_add_f32(const float* x, const float* y, float* z, int64_t n, void* stream);

/*
 * Recorded steps (the paper's graph mode, PAPER.md:290, 322-326:
 * "Graph captures the pipeline and replays all N kernels with one driver call",
 * and Grout's recorded decode step).  Between record_begin and
 * record_end every library call on `stream` (tile_gemm*, tile_add_f32) is
 * recorded instead of executed, in call order; record_end returns an opaque
 * step that tile_gemm_replay enqueues on any stream of the same device with ONE
 * driver call.  Recorded nodes keep the operand ADDRESSES: the caller keeps
 * those buffers alive and at the same place, and may rewrite their contents
 * between replays ("replayed nodes do not depend on addresses that change across
 * replays").  The same holds for the library's own memory: a step
 * OWNS the workspaces its nodes use (split-K partial sums and tickets, lockstep
 * counters, repacked operands).  They are allocated while recording, belong to no
 * other step and to no direct call, and live until tile_gemm_record_free -- so a
 * step stays valid whatever runs on any stream afterwards (larger shapes
 * included), it may be replayed on any stream of the same device, and replays of
 * different steps may overlap.  One step must not run concurrently with itself.
 * The M == 1 kernels keep their programmatic-dependent-launch edges inside the
 * step.  `stream` must not be NULL (the legacy default stream cannot be captured)
 * and must not already be recording (E_PATH); record_end on a stream that is not
 * recording fails with E_PATH.  The capture uses cudaStreamCaptureModeRelaxed (the
 * step's workspaces are cudaMalloc'ed while the stream captures, which the stricter
 * modes refuse).  Consequence for the caller: while the recording is open the runtime
 * no longer rejects potentially unsafe calls (cudaMalloc, cudaMemcpy, a legacy-stream
 * synchronisation, ...) made by this or any other host thread, as it would under the
 * default global mode -- keep such calls from touching the recording stream's work
 * yourself.  A recording that is still open at tile_gemm_shutdown is abandoned: its
 * workspaces are freed, the stream's capture is left for the caller to end.
 * A failed call while recording leaves the capture open; still call record_end
 * (it reports the invalidated capture and releases what the recording held).
 * Library calls on a stream the CALLER captures itself (cudaStreamBeginCapture)
 * work too, with the stream's ordinary workspaces: those must exist beforehand
 * (a call that would have to grow one fails with TILE_GEMM_E_CUDA and says so)
 * and are then kept until tile_gemm_shutdown.
 * tile_gemm_recorded_nodes returns the number of graph nodes (kernels and
 * workspace memsets) in a step, -1 for anything that is not a live step;
 * tile_gemm_launch_count grows by that number per replay.  tile_gemm_record_free
 * destroys a step and its workspaces (NULL is a no-op; it waits for replays still
 * in flight).
 */
int tile_gemm_record_begin(void* stream);
int tile_gemm_record_end(void* stream, void** step_out);
int tile_gemm_replay(void* step, void* stream);
int64_t tile_gemm_recorded_nodes(void* step);
int tile_gemm_record_free(void* step);

/*
 * The M = 1 product  y = x * B  (the decode GEMV) for callers that
 * must not, or cannot, allocate device memory.
 *
 * Why it exists.  tile_gemm keeps a grow-only workspace per stream and gets it from
 * cudaMalloc the first time a shape needs one.  Some programs cannot afford that
 * call: an inference server that hands every byte of HBM to its own pool at start-up
 * (weights, KV cache) leaves nothing for a library's cudaMalloc to find; a plug-in
 * running under a host whose memory policy forbids allocations after initialisation
 * has no permission to make it; and a latency-bound decode loop cannot take the
 * device-wide synchronisation and the unbounded duration that cudaMalloc / cudaFree
 * bring with them.  For those callers this entry never calls cudaMalloc, cudaFree or
 * any library routine that allocates device memory: its only scratch -- the fp32
 * partial sums of the K slices and one arrival ticket per 256-column block -- lives
 * in ONE array that is part of the library image itself,
 * TILE_GEMV_NO_ALLOC_SCRATCH_BYTES (1 MiB + 4 KiB) per GPU, present from the moment
 * a device loads the library until the process exits, whether or not this entry is
 * ever called.  The caller passes x, B and y exactly as to tile_gemm.
 *
 * Operation: y[j] = round_out( sum_{k<K} x[k] * B[k*ldb + j] ), 0 <= j < N; x (K
 * elements) and B (K x N, row stride ldb elements) hold in_dtype (TILE_GEMM_IN_BF16 /
 * _F16), y holds out_dtype (TILE_GEMM_OUT_F32 / _BF16 / _F16); all three are DEVICE
 * pointers on the current device, owned by the caller.  The kernel is the library's
 * default M = 1 kernel (csrc/gemv_kernel.cuh: TMA ring over 256-column blocks,
 * interleaved K slices, fp32 FMA) in its ticket hand-over: each slice stores its
 * partial sums to the scratch array, and the slice that arrives last adds all of
 * them in slice order and writes y.  The sum order is fixed by (N, K, slice count),
 * so results are bitwise reproducible from call to call; they equal tile_gemm's bits
 * when both run the same slice count and otherwise differ only by fp32 summation
 * order (same tolerance; identical for integer-valued inputs whose sums are exact).
 *
 * `split`: 0 = automatic (as many K slices per column block as keep every CTA
 * resident, at most what the scratch holds); > 0 = that many slices (values above
 * ceil(K / 64) mean ceil(K / 64)).
 *
 * Limits -- a request beyond them fails with TILE_GEMM_E_LIMIT, says which limit, and
 * enqueues nothing:
 *   N <= TILE_GEMV_NO_ALLOC_MAX_N (262144 columns = 1024 blocks of 256: one ticket each);
 *   ceil(N / 256) * slices <= TILE_GEMV_NO_ALLOC_MAX_TILES (1024 tiles of 256 partial sums).
 * Further preconditions: those of tile_gemm with M = 1 (same codes), plus B 16-byte
 * aligned with ldb a multiple of 8 (E_PATH otherwise: the repack path would need an
 * allocated copy), split >= 0 (E_EXTENT).  x and y need only element alignment.
 * N == 0 is a successful no-op, K == 0 writes zeros.
 *
 * Set-up on first use: the first call on each device looks up the device address of
 * the scratch array (cudaGetSymbolAddress with that device current -- the array's
 * name is only a host-side handle) and sets the kernel's shared-memory attribute;
 * the first call for a given (B, N, K, ldb) encodes a TMA descriptor into a host-side
 * cache.  Make that first call on a device before any stream capture begins.  Later
 * calls do no set-up.
 *
 * Sharing: every call on a device -- whatever the stream or host thread -- uses the
 * same array.  Each call clears the tickets it is about to use with a memset node
 * queued on `stream` ahead of the kernel (the array keeps the previous call's
 * contents; partial sums are always written before they are read) and launches
 * without programmatic dependent launch, so calls queued on ONE stream are safe back
 * to back.  Calls whose kernels can overlap on the GPU (different streams without
 * an ordering between them, or several host threads feeding different streams) RACE
 * on the scratch and produce wrong results: order them with events or keep them on
 * one stream.  tile_gemm and the other entries never touch this array and may run
 * concurrently with it.  Asynchronous on `stream`; tile_gemm_launch_count grows by one
 * per call (the memset is not counted).
 */
#define TILE_GEMV_NO_ALLOC_MAX_N 262144
#define TILE_GEMV_NO_ALLOC_MAX_TILES 1024
#define TILE_GEMV_NO_ALLOC_SCRATCH_BYTES 1052672   /* 1024 * 256 * 4 partial sums + 1024 * 4 tickets */
int tile_gemv_no_alloc(const void* x, const void* B, void* y,
                       int64_t N, int64_t K, int64_t ldb,
                       int in_dtype, int out_dtype, int split, void* stream);

/*
 * Launch preconditions + shape selector as a pure host function (PAPER.md:200:
 * "runs once per launch before any work is queued"; tile shapes
 * chosen per size).  Never dereferences A/B/C and makes no CUDA call.
 * Returns the TILE_GEMM_PATH_* the auto selector takes (> 0), or the NEGATED
 * status code (-TILE_GEMM_E_*) when a precondition fails.
 */
int tile_gemm_select(int64_t M, int64_t N, int64_t K,
                     int64_t lda, int64_t ldb, int64_t ldc,
                     const void* A, const void* B, const void* C, int out_dtype);

/*
 * End-to-end convenience entry on HOST buffers (pageable or pinned): copies A
 * and B to the device, runs tile_gemm, copies C[0..M) x [0..N) back (row pitch
 * ldc) and synchronises before returning.  Device staging buffers are grow-only
 * and owned by the library.  For M >= 2048 the rows of A go up in 1024-row chunks
 * (the last 1024 rows in halving chunks down to 128 rows, so that little is left to
 * do after the last byte has arrived) on one stream, each chunk's GEMM runs on a
 * second stream as soon as its rows and all of B have landed, and its rows of C
 * return on a third while the next chunk is still coming in (PCIe is full duplex).  Every chunk is an ordinary tile_gemm
 * call that plans itself, so fp32 results may differ from the one-shot order in
 * the last bits (same tolerance; identical for integer-valued inputs).  Pinned
 * host memory is needed for the copies to overlap.  This is the call bench.py's
 * `e2e` figure times.
 * Thread safety: the staging buffers, streams and events are kept per device and
 * the whole call runs under that device's lock -- concurrent callers on ONE GPU are
 * serialised (they would share its PCIe link anyway), never mixed; callers on
 * different GPUs do not wait for each other.
 */
int tile_gemm_host(const void* A_host, const void* B_host, void* C_host,
                   int64_t M, int64_t N, int64_t K,
                   int64_t lda, int64_t ldb, int64_t ldc, int out_dtype);

/*
 * Debug: run the GEMM kernel's own persistent schedule and epilogue (no loads,
 * no MMAs) and write, for every element of an M x N int32 matrix `owner`
 * (device, row stride ld_owner), the value (tile_index << 8) | cta_index of the
 * CTA that owns the element's output tile.  "Each sub-tensor has exactly one
 * owner": tests check the map is the documented function and
 * covers [0,M) x [0,N) exactly once.  K only selects the tile configuration.
 */
int tile_gemm_debug_owner_map(int32_t* owner, int64_t M, int64_t N, int64_t K,
                              int64_t ld_owner, int out_dtype, void* stream);

/* Number of kernels this library has launched in this process (all paths). */
int64_t tile_gemm_launch_count(void);

/* Static, human-readable name of a status code. */
const char* tile_gemm_status_string(int status);

/* Thread-local detailed message of the calling thread's last failing call. */
const char* tile_gemm_last_error(void);

/* Frees workspaces, staging buffers and the tensor-map cache.  The caller must
 * have synchronised all streams that ran library work. */
int tile_gemm_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* TILE_GEMM_H_ */
