// Host entry of libtilegemm.so: launch preconditions, shape selector, tensor-map cache,
// workspaces and kernel launches.  See include/tile_gemm.h for the contract.
//
// "An obligation becomes a launch precondition when every operand is known at launch ... The
// check moves into the generated launcher, runs once per launch before any work is queued, and
// returns an error on failure".  Everything validated here is exactly what lets
// the device K loops run without a single bounds check.
#include "../../include/tile_gemm.h"
#include "../../include/tile_gemm_debug.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "add_kernel.cuh"
#include "aux_kernels.cuh"
#include "gemm_kernel.cuh"
#include "gemv_kernel.cuh"
#include "skinny_kernel.cuh"

namespace {

// ------------------------------------------------------------------ errors
thread_local char g_err[640] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

const char* const kStatusNames[TILE_GEMM_NUM_STATUS] = {
    "ok",
    "null pointer with a non-empty extent",
    "negative extent",
    "lda < K",
    "ldb < N",
    "ldc < N",
    "unknown out_dtype",
    "pointer not aligned to its element size",
    "C overlaps A or B",
    "extent overflow",
    "no sm_100 CUDA device",
    "CUDA call failed",
    "path not applicable",
    "internal error",
    "unknown in_dtype",
    "request exceeds the fixed scratch of tile_gemv_no_alloc",
};

std::atomic<int64_t> g_launches{0};
std::atomic<unsigned long long*> g_trace{nullptr};   // tile_gemm_debug_trace
std::atomic<int64_t> g_trace_cap{0};
// The trace buffer a launch on `s` may write: none while `s` is capturing (a recorded step would keep the
// raw address and write through it on every replay, long after the caller has dropped the buffer).
unsigned long long* trace_for(cudaStream_t s) {
    unsigned long long* t = g_trace.load();
    if (!t) return nullptr;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cs) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return cs == cudaStreamCaptureStatusNone ? t : nullptr;
}
constexpr int kNumTune = 16;   // keys 0..12 are documented in include/tile_gemm_debug.h
std::atomic<int> g_tune[kNumTune];

// ------------------------------------------------------------------ preconditions + selector
struct Plan {
    int path = 0;
    int esize = 4;
    int64_t a_bytes = 0, b_bytes = 0, c_bytes = 0;   // byte spans of the three operands
    bool a_tma = false, b_tma = false, c_tma = false;
};

bool span_bytes(int64_t rows, int64_t cols, int64_t ld, int64_t esize, int64_t* out) {
    if (rows == 0 || cols == 0) { *out = 0; return true; }
    int64_t t;
    if (__builtin_mul_overflow(rows - 1, ld, &t)) return false;
    if (__builtin_add_overflow(t, cols, &t)) return false;
    if (__builtin_mul_overflow(t, esize, &t)) return false;
    *out = t;
    return true;
}

bool overlaps(const void* p, int64_t pn, const void* q, int64_t qn) {
    if (pn == 0 || qn == 0) return false;
    const uintptr_t a = (uintptr_t)p, b = (uintptr_t)q;
    return a < b + (uintptr_t)qn && b < a + (uintptr_t)pn;
}

constexpr int kAuxCtasPerSm = 16;      // grid cap of the grid-stride helper kernels (repack, zero fill), per SM

int check_and_select(const void* A, const void* B, const void* C, int64_t M, int64_t N, int64_t K, int64_t lda,
                     int64_t ldb, int64_t ldc, int in_dtype, int out_dtype, Plan* plan) {
    if (M < 0 || N < 0 || K < 0)
        return fail(TILE_GEMM_E_EXTENT, "negative extent: M=%lld N=%lld K=%lld", (long long)M, (long long)N,
                    (long long)K);
    if (out_dtype != TILE_GEMM_OUT_F32 && out_dtype != TILE_GEMM_OUT_BF16 && out_dtype != TILE_GEMM_OUT_F16)
        return fail(TILE_GEMM_E_DTYPE,
                    "out_dtype=%d is none of TILE_GEMM_OUT_F32 (0), TILE_GEMM_OUT_BF16 (1), TILE_GEMM_OUT_F16 (2)",
                    out_dtype);
    if (in_dtype != TILE_GEMM_IN_BF16 && in_dtype != TILE_GEMM_IN_F16)
        return fail(TILE_GEMM_E_IN_DTYPE, "in_dtype=%d is neither TILE_GEMM_IN_BF16 (0) nor TILE_GEMM_IN_F16 (1)",
                    in_dtype);
    if (lda < K) return fail(TILE_GEMM_E_LDA, "lda=%lld < K=%lld", (long long)lda, (long long)K);
    if (ldb < N) return fail(TILE_GEMM_E_LDB, "ldb=%lld < N=%lld", (long long)ldb, (long long)N);
    if (ldc < N) return fail(TILE_GEMM_E_LDC, "ldc=%lld < N=%lld", (long long)ldc, (long long)N);
    const int64_t lim = (int64_t)INT32_MAX - 1024;
    if (M > lim || N > lim || K > lim)
        return fail(TILE_GEMM_E_OVERFLOW, "extent above 2^31-1025: M=%lld N=%lld K=%lld", (long long)M, (long long)N,
                    (long long)K);
    plan->esize = (out_dtype == TILE_GEMM_OUT_F32) ? 4 : 2;
    if (!span_bytes(M, K, lda, 2, &plan->a_bytes) || !span_bytes(K, N, ldb, 2, &plan->b_bytes) ||
        !span_bytes(M, N, ldc, plan->esize, &plan->c_bytes))
        return fail(TILE_GEMM_E_OVERFLOW, "operand byte span overflows int64");
    if (lda > (int64_t(1) << 38) || ldb > (int64_t(1) << 38) || ldc > (int64_t(1) << 38))
        return fail(TILE_GEMM_E_OVERFLOW, "row stride above 2^38 elements");
    const int64_t tiles = ((M + 127) / 128) * ((N + 127) / 128);
    if (tiles > lim) return fail(TILE_GEMM_E_OVERFLOW, "output tile count %lld overflows int32", (long long)tiles);
    if (M == 0 || N == 0) { plan->path = TILE_GEMM_PATH_NOOP; return TILE_GEMM_OK; }
    if (C == nullptr) return fail(TILE_GEMM_E_NULL, "C is NULL but M*N > 0");
    if (K > 0 && A == nullptr) return fail(TILE_GEMM_E_NULL, "A is NULL but M*K > 0");
    if (K > 0 && B == nullptr) return fail(TILE_GEMM_E_NULL, "B is NULL but K*N > 0");
    if (((uintptr_t)A & 1) || ((uintptr_t)B & 1))
        return fail(TILE_GEMM_E_ALIGN, "A (%p) or B (%p) is not 2-byte aligned", A, B);
    if ((uintptr_t)C & (uintptr_t)(plan->esize - 1))
        return fail(TILE_GEMM_E_ALIGN, "C (%p) is not %d-byte aligned", C, plan->esize);
    if (overlaps(C, plan->c_bytes, A, plan->a_bytes))
        return fail(TILE_GEMM_E_ALIAS, "C [%p,+%lld) overlaps A [%p,+%lld): the output must be exclusively owned", C,
                    (long long)plan->c_bytes, A, (long long)plan->a_bytes);
    if (overlaps(C, plan->c_bytes, B, plan->b_bytes))
        return fail(TILE_GEMM_E_ALIAS, "C [%p,+%lld) overlaps B [%p,+%lld): the output must be exclusively owned", C,
                    (long long)plan->c_bytes, B, (long long)plan->b_bytes);
    // TMA addressability: 16-byte aligned base and 16-byte multiple row pitch
    plan->a_tma = (((uintptr_t)A & 15) == 0) && (lda % 8 == 0);
    plan->b_tma = (((uintptr_t)B & 15) == 0) && (ldb % 8 == 0);
    plan->c_tma = (((uintptr_t)C & 15) == 0) && ((ldc * plan->esize) % 16 == 0);
    if (K == 0) plan->path = TILE_GEMM_PATH_ZERO;
    else if (M == 1) plan->path = TILE_GEMM_PATH_GEMV;
    else plan->path = (plan->a_tma && plan->b_tma) ? TILE_GEMM_PATH_GEMM_TMA : TILE_GEMM_PATH_GEMM_REPACK;
    return TILE_GEMM_OK;
}

// ------------------------------------------------------------------ device
struct DevInfo {
    bool probed = false;
    int status = TILE_GEMM_E_DEVICE;
    int sms = 0;
};
DevInfo g_dev[64];
std::mutex g_mu;

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(TILE_GEMM_E_CUDA, "%s failed: %s (%d)", #expr, cudaGetErrorString(e_), (int)e_); \
    } while (0)

int current_device(int* dev, int* sms) {
    int d = -1;
    cudaError_t e = cudaGetDevice(&d);
    if (e != cudaSuccess || d < 0 || d >= 64)
        return fail(TILE_GEMM_E_DEVICE, "no usable CUDA device: %s; this library has no CPU fallback",
                    cudaGetErrorString(e));
    std::lock_guard<std::mutex> lk(g_mu);
    DevInfo& di = g_dev[d];
    if (!di.probed) {
        int major = 0, minor = 0, sms_ = 0;
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, d);
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, d);
        cudaDeviceGetAttribute(&sms_, cudaDevAttrMultiProcessorCount, d);
        di.probed = true;
        di.sms = sms_;
        di.status = (major == 10 && minor == 0) ? TILE_GEMM_OK : TILE_GEMM_E_DEVICE;
        if (di.status != TILE_GEMM_OK)
            snprintf(g_err, sizeof g_err, "device %d is sm_%d%d; the kernels are built for sm_100a only", d, major,
                     minor);
    }
    if (di.status != TILE_GEMM_OK) {
        if (g_err[0] == 0) snprintf(g_err, sizeof g_err, "device %d is not sm_100", d);
        return di.status;
    }
    *dev = d;
    *sms = di.sms;
    return TILE_GEMM_OK;
}

// ------------------------------------------------------------------ tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

struct MapKey {
    uintptr_t p;
    uint64_t d0, d1, pitch;
    uint32_t b0, b1, dtype, swizzle;
    bool operator==(const MapKey& o) const {
        return p == o.p && d0 == o.d0 && d1 == o.d1 && pitch == o.pitch && b0 == o.b0 && b1 == o.b1 &&
               dtype == o.dtype && swizzle == o.swizzle;
    }
};
struct MapKeyHash {
    size_t operator()(const MapKey& k) const {
        uint64_t h = 1469598103934665603ull;
        const uint64_t v[6] = {k.p, k.d0, k.d1, k.pitch, ((uint64_t)k.b0 << 32) | k.b1,
                               ((uint64_t)k.dtype << 32) | k.swizzle};
        for (uint64_t x : v) { h ^= x; h *= 1099511628211ull; }
        return (size_t)h;
    }
};
std::unordered_map<MapKey, CUtensorMap, MapKeyHash> g_maps;

// 2-D row-major tensor [d1 rows][d0 cols] of `esize`-byte elements with row pitch `pitch` bytes.
int get_tensor_map(CUtensorMap* out, const void* base, int dtype_bytes, bool is_float32, uint64_t d0, uint64_t d1,
                   uint64_t pitch, uint32_t b0, uint32_t b1, int swizzle_bytes) {
    MapKey key{(uintptr_t)base, d0, d1, pitch, b0, b1, (uint32_t)(is_float32 ? 4 : dtype_bytes),
               (uint32_t)swizzle_bytes};
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_maps.find(key);
    if (it != g_maps.end()) { *out = it->second; return TILE_GEMM_OK; }
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || fn == nullptr || qres != cudaDriverEntryPointSuccess)
            return fail(TILE_GEMM_E_CUDA, "cuTensorMapEncodeTiled entry point unavailable: %s", cudaGetErrorString(e));
        g_encode = (EncodeTiledFn)fn;
    }
    const cuuint64_t dims[2] = {d0, d1};
    const cuuint64_t strides[1] = {pitch};
    const cuuint32_t box[2] = {b0, b1};
    const cuuint32_t estr[2] = {1, 1};
    const CUtensorMapDataType dt = is_float32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
    CUtensorMap m;
    CUresult r = g_encode(&m, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                                                : CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return fail(TILE_GEMM_E_CUDA,
                    "cuTensorMapEncodeTiled failed (%d) for base=%p dims=(%llu,%llu) pitch=%llu box=(%u,%u)", (int)r,
                    base, (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)pitch, b0, b1);
    if (g_maps.size() > 8192) g_maps.clear();
    g_maps.emplace(key, m);
    *out = m;
    return TILE_GEMM_OK;
}

// ------------------------------------------------------------------ workspaces
// Library-owned device memory.  Lifetime rules (a replayed node must not depend on
// an address that changes across replays):
//   * direct calls use one WorkspaceSet per (device, stream), grown by free + allocate (cudaFree
//     synchronises, so no in-flight kernel loses its buffer);
//   * a recorded step (tile_gemm_record_begin .. _end) owns a PRIVATE WorkspaceSet: the addresses
//     baked into its nodes belong to the step, live until tile_gemm_record_free and are shared with
//     no direct call and no other step, whichever stream it is replayed on.  A buffer that must grow
//     while the step is still being recorded is retired (kept for the nodes already captured), not freed;
//   * a stream that the CALLER is capturing (its own cudaStreamBeginCapture) gets the per-stream set,
//     which is then pinned: it is never freed before tile_gemm_shutdown, and growing it under that
//     capture is refused (cudaMalloc is not allowed in a foreign capture).
struct Buf {
    void* p = nullptr;
    size_t n = 0;
};
struct WorkspaceSet {
    Buf repack;     // 16-byte pitched copies of operands TMA cannot address
    Buf sync;       // GEMM lockstep window counters, zeroed before each launch that uses them
    Buf partials;   // split-K fp32 partial sums (GEMV: [col_blocks][split][cols]; GEMM: per split tile)
    Buf tickets;    // split-K arrival tickets, zero between launches (the last arrival re-arms them)
    Buf packed;     // M = 1 tagged split-K slots {fp32, tag}, all zero between launches (the combiner re-arms them)
    bool pinned = false;           // baked into a graph this library does not own
    std::vector<void*> retired;    // outgrown buffers that captured nodes may still reference
};
struct Recording {
    int dev = 0;
    WorkspaceSet ws;
};
std::unordered_map<uint64_t, WorkspaceSet> g_wsets;            // (device, stream) -> direct-call workspaces
std::unordered_map<uintptr_t, Recording*> g_recording;         // streams between record_begin and record_end
std::vector<void*> g_retired;                                   // retired buffers of pinned per-stream sets

// tile_gemm_host: one staging set per device, used under that device's own lock for the whole call
struct HostStage {
    std::mutex mu;
    Buf a, b, c;
    cudaStream_t in = nullptr, compute = nullptr, out = nullptr;   // copy-in, GEMMs, copy-out
    std::vector<cudaEvent_t> events;
};
HostStage g_host[64];

int grow(Buf& b, size_t need) {
    if (b.n >= need) return TILE_GEMM_OK;
    if (b.p) CUDA_TRY(cudaFree(b.p));   // cudaFree synchronises: no in-flight user remains
    b.p = nullptr;
    b.n = 0;
    const size_t sz = (need + ((size_t)1 << 20) - 1) & ~(((size_t)1 << 20) - 1);
    CUDA_TRY(cudaMalloc(&b.p, sz));
    b.n = sz;
    return TILE_GEMM_OK;
}

// The workspace set a call on stream `s` uses, and whether its buffers may be (re)allocated now.
struct WsRef {
    WorkspaceSet* ws;
    bool ours;       // a recording of this library
    bool foreign;    // the caller's own capture
};
WsRef workspace_set(int dev, cudaStream_t s) {   // g_mu held
    auto it = g_recording.find((uintptr_t)s);
    if (it != g_recording.end()) return {&it->second->ws, true, false};
    WorkspaceSet& w = g_wsets[((uint64_t)dev << 56) ^ (uint64_t)(uintptr_t)s];
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const bool cap = cudaStreamIsCapturing(s, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone;
    if (cap) w.pinned = true;
    return {&w, false, cap};
}

// make `b` at least `need` bytes under the rules above; *fresh is set when the buffer is new
int ensure(const WsRef& r, Buf& b, size_t need, const char* what, bool* fresh = nullptr) {
    if (fresh) *fresh = false;
    if (b.n >= need) return TILE_GEMM_OK;
    if (r.foreign)
        return fail(TILE_GEMM_E_CUDA,
                    "the %s workspace of this stream must grow during the caller's stream capture; run the shape "
                    "once on the stream before capturing, or record with tile_gemm_record_begin", what);
    if ((r.ours || r.ws->pinned) && b.p) {   // captured nodes may hold the old address
        (r.ours ? r.ws->retired : g_retired).push_back(b.p);
        b.p = nullptr;
        b.n = 0;
    }
    int rc = grow(b, need);
    if (rc) return rc;
    if (fresh) *fresh = true;
    return TILE_GEMM_OK;
}

int workspace_for(int dev, cudaStream_t s, size_t need, void** out) {
    std::lock_guard<std::mutex> lk(g_mu);
    const WsRef r = workspace_set(dev, s);
    int rc = ensure(r, r.ws->repack, need, "operand repack");
    if (rc) return rc;
    *out = r.ws->repack.p;
    return TILE_GEMM_OK;
}

int sync_workspace_for(int dev, cudaStream_t s, size_t bytes, uint32_t** out) {
    std::lock_guard<std::mutex> lk(g_mu);
    const WsRef r = workspace_set(dev, s);
    int rc = ensure(r, r.ws->sync, bytes, "GEMM lockstep");
    if (rc) return rc;
    *out = (uint32_t*)r.ws->sync.p;
    return TILE_GEMM_OK;
}

// split-K workspace: fp32 partials and one ticket per (column block | tile, CTA rank)
int gemv_workspace_for(int dev, cudaStream_t s, size_t partial_bytes, size_t ticket_bytes, float** partials,
                       uint32_t** tickets) {
    std::lock_guard<std::mutex> lk(g_mu);
    const WsRef r = workspace_set(dev, s);
    int rc = ensure(r, r.ws->partials, partial_bytes, "split-K partial sum");
    if (rc) return rc;
    bool fresh = false;
    rc = ensure(r, r.ws->tickets, ticket_bytes, "split-K ticket", &fresh);
    if (rc) return rc;
    // a new ticket buffer starts at zero (in a recording this is a memset node: every replay re-zeroes it)
    if (fresh) CUDA_TRY(cudaMemsetAsync(r.ws->tickets.p, 0, r.ws->tickets.n, s));
    *partials = (float*)r.ws->partials.p;
    *tickets = (uint32_t*)r.ws->tickets.p;
    return TILE_GEMM_OK;
}

// tagged split-K slots of the M = 1 kernel (gemv_kernel.cuh, GEMV_FLAG_PACKED)
int packed_workspace_for(int dev, cudaStream_t s, size_t bytes, unsigned long long** out) {
    std::lock_guard<std::mutex> lk(g_mu);
    const WsRef r = workspace_set(dev, s);
    bool fresh = false;
    int rc = ensure(r, r.ws->packed, bytes, "split-K slot", &fresh);
    if (rc) return rc;
    if (fresh) CUDA_TRY(cudaMemsetAsync(r.ws->packed.p, 0, r.ws->packed.n, s));
    *out = (unsigned long long*)r.ws->packed.p;
    return TILE_GEMM_OK;
}

void free_workspace_set(WorkspaceSet& w) {
    for (Buf* b : {&w.repack, &w.sync, &w.partials, &w.tickets, &w.packed}) {
        if (b->p) cudaFree(b->p);
        *b = Buf();
    }
    for (void* q : w.retired) cudaFree(q);
    w.retired.clear();
}

// ------------------------------------------------------------------ GEMM launch
struct GemmConfig {
    int id;       // 1: 1-CTA 128x128, 2: 1-CTA 128x256, 3: 2-CTA 256x256, 4: 2-CTA 256x512
    int cg, bn, stages, nacc;
    int tile_n() const { return bn * nacc; }
};
const GemmConfig kConfigs[5] = {{0, 0, 0, 0, 0}, {1, 1, 128, 6, 1}, {2, 1, 256, 4, 1}, {3, 2, 256, 6, 1},
                                {4, 2, 256, 4, 2}};

// split-K of the last wave: at most kGemmMaxSplit slices of at least kGemmMinSliceKTiles k-tiles each
constexpr int kGemmMaxSplit = 16, kGemmMinSliceKTiles = 4;

// The last, partial wave of `rem` tiles on `slots` clusters, in microseconds, and the slice count that
// gets it: a whole tile at the per-cluster share of ~1500 TFLOP/s, or ceil(rem * c / slots) rounds of
// 1/c-tile units plus what a slice costs on top (its fp32 accumulators go through L2 once as a store
// and once as a load of the fix-up, ~100 GB/s per cluster, and a ticket round trip) -- measured on
// B200: ~8 us for a 256x512 slice, ~3.5 us for 128x128.  Cutting pays for long K loops and for
// problems below one wave (skinny M).
// cost-model constants (B200, measured): what the whole chip sustains on this kernel's main loop, in
// FLOP per microsecond; a slice's fixed cost; the rate at which one cluster moves a slice's partials
constexpr double kModelChipFlopPerUs = 1500e6, kModelSliceFixedUs = 3.0, kModelSliceBytesPerUs = 100e3;

double last_wave_us(int64_t rem, int64_t slots, int tile_m, int tile_n, int cg, int64_t k_tiles, int sms, int64_t* slices) {
    const double tile_us = 2.0 * tile_m * tile_n * (double)k_tiles * tg::GEMM_BK / (kModelChipFlopPerUs * cg / (double)sms);
    const double ovh_us = kModelSliceFixedUs + (double)tile_m * tile_n * 4.0 / kModelSliceBytesPerUs;
    *slices = 1;
    if (rem <= 0) return 0.0;
    double best = tile_us;
    int64_t sl_max = k_tiles / kGemmMinSliceKTiles;
    if (sl_max > kGemmMaxSplit) sl_max = kGemmMaxSplit;
    if (k_tiles < 2 * kGemmMinSliceKTiles || g_tune[3].load() == 1) return best;
    for (int64_t c = 2; c <= sl_max; ++c) {
        const double rounds = (double)((rem * c + slots - 1) / slots);
        const double cost = rounds / (double)c * tile_us + (rounds + 0.5 * (double)c) * ovh_us;
        if (cost < best * 0.97) { best = cost; *slices = c; }
    }
    return best;
}

// estimated time of the whole launch with tiles of tile_m x tile_n on `slots` clusters
double launch_us(int64_t M, int64_t N, int64_t K, int tile_m, int tile_n, int cg, int sms) {
    const int64_t slots = sms / cg, k_tiles = (K + tg::GEMM_BK - 1) / tg::GEMM_BK;
    const int64_t tiles = ((M + tile_m - 1) / tile_m) * ((N + tile_n - 1) / tile_n);
    const double tile_us = 2.0 * tile_m * tile_n * (double)k_tiles * tg::GEMM_BK / (kModelChipFlopPerUs * cg / (double)sms);
    int64_t sl;
    return (double)(tiles / slots) * tile_us + last_wave_us(tiles % slots, slots, tile_m, tile_n, cg, k_tiles, sms, &sl);
}

GemmConfig choose_config(int64_t M, int64_t N, int64_t K, int sms) {
    const int forced = g_tune[0].load();
    if (forced >= 1 && forced <= 4) return kConfigs[forced];
    // One row of 128-tall tiles covers M: a CTA pair's second CTA would own rows that do not exist, and the
    // launch is a weight stream where many narrow tiles keep more SMs pulling (measured at M = 8 on the decode
    // shapes: 128x128 tiles 4.4 / 3.9 / 6.3 / 5.0 TB/s, 128x256 3.5 / 3.2 / 5.8 / 4.5, the pair kernels 5.2 on
    // K = 5120, N = 51200 where they used to be chosen).
    if (M <= tg::GEMM_BM) return kConfigs[1];
    const int64_t t3 = ((M + 255) / 256) * ((N + 255) / 256);
    const int64_t t4 = ((M + 255) / 256) * ((N + 511) / 512);
    // the 256x512 tile moves a quarter less operand data per FLOP (the kernel is power bound,
    // DESIGN.md "Power"); take it unless its coarser wave quantisation -- after the last wave has
    // been cut along K where that pays -- costs more than that buys
    // a 256x512 tile occupies both accumulator slots, so ~2 us of each tile's epilogue are not hidden
    // behind the next main loop (calibrated on steady-state A/Bs: K = 5120 prefers 256x256 by 1-7 %,
    // K >= 8192 prefers 256x512 by 3-4 %)
    const double exposed4 = 2.0 * (double)((t4 + sms / 2 - 1) / (sms / 2));
    if (t4 >= sms / 2 &&
        launch_us(M, N, K, 256, 512, 2, sms) + exposed4 <= launch_us(M, N, K, 256, 256, 2, sms) * 1.06)
        return kConfigs[4];
    // from four fifths of a wave of CTA pairs on, 256x256 pair tiles beat 128x256 single-CTA tiles (same-process A/B:
    // 2048^3 980 vs 947 TF/s, 2048 x 2048 x 8192 1183 vs 1116, 1536 x 3072 x 2048 1036 vs 1013; level at K <= 1024)
    if (t3 * 5 >= (int64_t)(sms / 2) * 4) return kConfigs[3];
    const int64_t t2 = ((M + 127) / 128) * ((N + 255) / 256);
    if (t2 * 4 >= (int64_t)sms * 3) return kConfigs[2];
    return kConfigs[1];
}

// How many work-unit owners (CTA pairs for cg = 2, CTAs for cg = 1) of a tile configuration the device
// holds at once, from the occupancy calculator (GPC layout, shared memory, registers): the persistent
// grid is never larger, so that every CTA of a launch is resident when nothing else runs on the device.
template <int CG, int BN, int STAGES, int NACC, int MC = 0>
int query_resident_units(int sms) {
    using L = tg::GemmSmem<CG, BN, STAGES, NACC>;
    auto kern = tg::gemm_tcgen05_kernel<CG, BN, STAGES, NACC, false, 0, MC>;
    constexpr int CL = CG * (MC ? 2 : 1);   // CTAs per cluster
    int n = 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::TOTAL) == cudaSuccess) {
        if (CG == 2) {
            cudaLaunchConfig_t cfg;
            memset(&cfg, 0, sizeof cfg);
            cfg.gridDim = dim3((unsigned)(sms / CL * CL), 1, 1);
            cfg.blockDim = dim3(tg::GEMM_THREADS, 1, 1);
            cfg.dynamicSmemBytes = L::TOTAL;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = CL;
            attr[0].val.clusterDim.y = 1;
            attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) n = 0;
        } else {
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, tg::GEMM_THREADS, L::TOTAL) == cudaSuccess)
                n = per_sm * sms;
        }
    }
    cudaGetLastError();   // a failed query is not an error of the call that asked
    if (n <= 0 || n > sms / CL) n = sms / CL;   // one CTA per SM at most: a CTA allocates all of tensor memory
    return n;
}

// config ids 1..4, and 5 = config 4 with two pairs per cluster (B multicast): resident clusters
int resident_units(int id, int dev, int sms) {
    static std::atomic<int> cache[6][64];
    int v = cache[id][dev].load();
    if (v > 0) return v;
    switch (id) {
        case 1: v = query_resident_units<1, 128, 6, 1>(sms); break;
        case 2: v = query_resident_units<1, 256, 4, 1>(sms); break;
        case 3: v = query_resident_units<2, 256, 6, 1>(sms); break;
        case 4: v = query_resident_units<2, 256, 4, 2>(sms); break;
        default: v = query_resident_units<2, 256, 4, 2, 1>(sms); break;
    }
    cache[id][dev].store(v);
    return v;
}

// lockstep defaults: on from kLockstepMinTiles tiles per cluster and kLockstepMinKTiles k-tiles
constexpr int kLockstepMinTiles = 2, kLockstepMinKTiles = 256, kLockstepWindow = 32;

struct GemmLaunch {
    GemmConfig cfg;
    tg::GemmParams p;
    int ctas;
    bool mc = false;   // two CTA pairs per cluster, one tile row above the other, B multicast (gemm_kernel.cuh, MC = 1)
};

constexpr bool kGemmMulticastDefault = false;

void plan_gemm(int64_t M, int64_t N, int64_t K, int in_dtype, int out_dtype, int dev, int sms, GemmLaunch* gl,
               bool allow_split = false, bool allow_mc = true) {
    gl->cfg = choose_config(M, N, K, sms);
    const int tile_m = tg::GEMM_BM * gl->cfg.cg;
    tg::GemmParams& p = gl->p;
    memset(&p, 0, sizeof p);
    p.M = (int32_t)M; p.N = (int32_t)N; p.K = (int32_t)K;
    p.tiles_m = (int32_t)((M + tile_m - 1) / tile_m);
    p.tiles_n = (int32_t)((N + gl->cfg.tile_n() - 1) / gl->cfg.tile_n());
    int gm = g_tune[1].load();
    if (gm <= 0) gm = 16;   // steady-state A/B at 8192^3 and 16384^3: 16 tile rows per raster group beat 8 by 1-2 % (pairs) and tie at M = 4096
    p.group_m = gm < p.tiles_m ? gm : p.tiles_m;
    p.num_k_tiles = (int32_t)((K + tg::GEMM_BK - 1) / tg::GEMM_BK);
    p.out_16 = out_dtype != TILE_GEMM_OUT_F32;
    p.out_f16 = out_dtype == TILE_GEMM_OUT_F16;
    p.in_f16 = in_dtype == TILE_GEMM_IN_F16;
    int64_t tiles = (int64_t)p.tiles_m * p.tiles_n;
    // B multicast across two pairs (tuning key 12: 1 = never, 2 = whenever the configuration has it): a work unit
    // becomes two tile rows of the same tile column, and no unit is cut along K
    const int mc_tune = g_tune[12].load();
    gl->mc = gl->cfg.id == 4 && allow_mc && p.tiles_m >= 2 && mc_tune != 1 && (mc_tune == 2 || kGemmMulticastDefault);
    if (gl->mc) {
        p.tiles_m = (p.tiles_m + 1) / 2;
        p.group_m = (p.group_m + 1) / 2;
        tiles = (int64_t)p.tiles_m * p.tiles_n;
        allow_split = false;
    }
    int max_units = resident_units(gl->mc ? 5 : gl->cfg.id, dev, sms);
    const int cap = g_tune[2].load();
    const int cl = gl->cfg.cg * (gl->mc ? 2 : 1);   // CTAs per cluster
    if (cap > 0 && cap / cl >= 1 && cap / cl < max_units) max_units = cap / cl;
    // Split-K for the partial last wave: `rem` tiles are left after the whole waves;
    // cut each into floor(clusters / rem) slices so that the last round is one short, full wave.
    p.full_units = (int32_t)tiles;
    p.total_units = (int32_t)tiles;
    p.split = 0;
    p.kps = p.num_k_tiles;
    const int64_t rem = tiles % max_units;
    const int split_tune = g_tune[3].load();   // key 3 also overrides the GEMM split: 1 = never, >= 2 = that many slices
    if (allow_split && rem > 0 && split_tune != 1 && p.num_k_tiles >= 2 * kGemmMinSliceKTiles) {
        int64_t sl_max = p.num_k_tiles / kGemmMinSliceKTiles;
        if (sl_max > kGemmMaxSplit) sl_max = kGemmMaxSplit;
        int64_t sl = 1;
        last_wave_us(rem, max_units, tile_m, gl->cfg.tile_n(), gl->cfg.cg, p.num_k_tiles, sms, &sl);
        if (split_tune >= 2) sl = split_tune < sl_max ? split_tune : sl_max;
        if (sl >= 2) {
            const int64_t kps = (p.num_k_tiles + sl - 1) / sl;
            sl = (p.num_k_tiles + kps - 1) / kps;              // no empty slice
            if (sl >= 2) {
                p.split = (int32_t)sl;
                p.kps = (int32_t)kps;
                p.full_units = (int32_t)(tiles - rem);
                p.total_units = (int32_t)(tiles - rem + rem * sl);
            }
        }
    }
    int64_t units = p.total_units;
    if (units > max_units) units = max_units;
    gl->ctas = (int)units * cl;
}

template <int CG, int BN, int STAGES, int NACC, bool SPLIT, int EPI = 0, int MC = 0>
int launch_gemm_inst(const CUtensorMap& ta, const CUtensorMap& tb, const CUtensorMap& tc, const tg::GemmParams& p,
                     int ctas, cudaStream_t s, int dev) {
    using L = tg::GemmSmem<CG, BN, STAGES, NACC>;
    auto kern = tg::gemm_tcgen05_kernel<CG, BN, STAGES, NACC, SPLIT, EPI, MC>;
    static bool configured[64] = {};
    if (!configured[dev]) {
        CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::TOTAL));
        configured[dev] = true;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)ctas, 1, 1);
    cfg.blockDim = dim3(tg::GEMM_THREADS, 1, 1);
    cfg.dynamicSmemBytes = L::TOTAL;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (CG == 2) {   // a 1-CTA "cluster" attribute would still take the driver's cluster launch path
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = CG * (MC ? 2 : 1);
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    if ((g_tune[6].load() & 1) == 0) {   // tuning key 6 bit 0: no programmatic dependent launch
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, ta, tb, tc, p));
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

int launch_gemm(const GemmLaunch& gl, const CUtensorMap& ta, const CUtensorMap& tb, const CUtensorMap& tc,
                cudaStream_t s, int dev) {
    if (gl.mc) return launch_gemm_inst<2, 256, 4, 2, false, 0, 1>(ta, tb, tc, gl.p, gl.ctas, s, dev);
    switch (gl.cfg.id) {
#define TG_GEMM_CASE(id, CG, BN, ST, NA)                                                              \
    case id:                                                                                         \
        return gl.p.split > 0 ? launch_gemm_inst<CG, BN, ST, NA, true>(ta, tb, tc, gl.p, gl.ctas, s, dev) \
                              : launch_gemm_inst<CG, BN, ST, NA, false>(ta, tb, tc, gl.p, gl.ctas, s, dev);
        TG_GEMM_CASE(1, 1, 128, 6, 1)
        TG_GEMM_CASE(2, 1, 256, 4, 1)
        TG_GEMM_CASE(3, 2, 256, 6, 1)
        TG_GEMM_CASE(4, 2, 256, 4, 2)
#undef TG_GEMM_CASE
    }
    return fail(TILE_GEMM_E_INTERNAL, "unknown GEMM config %d", gl.cfg.id);
}

// Lockstep producers: only where a launch is long enough for clusters to drift (several whole
// tiles per cluster, long K loops); tuning key 6: bit 2 forces it on, bit 3 off, bits 8-15 = window.
// rounds the lockstep covers (0: off) and its window, from the plan alone
void lockstep_plan(const GemmLaunch& gl, int64_t* rounds_out, int* window_out) {
    const int tune = g_tune[6].load();
    const int clusters = gl.ctas / (gl.cfg.cg * (gl.mc ? 2 : 1));
    // rounds in which every cluster owns a whole tile: lockstep covers exactly these
    const int64_t rounds = clusters > 0 ? gl.p.full_units / clusters : 0;
    bool on = rounds >= kLockstepMinTiles && gl.p.num_k_tiles >= kLockstepMinKTiles;
    if (tune & 4) on = rounds >= 1 && gl.p.num_k_tiles >= 1;
    if (tune & 8) on = false;
    int window = (tune >> 8) & 255;
    if (window <= 0) window = kLockstepWindow;
    *rounds_out = on ? rounds : 0;
    *window_out = window;
}

int setup_lockstep(GemmLaunch& gl, int dev, cudaStream_t s) {
    int rc = TILE_GEMM_OK;
    {
        int64_t rounds = 0;
        int window = 0;
        lockstep_plan(gl, &rounds, &window);
        if (rounds > 0) {
            const int64_t windows = (rounds * gl.p.num_k_tiles + window - 1) / window + 1;
            gl.p.sync_rounds = (int32_t)rounds;
            uint32_t* sync = nullptr;
            rc = sync_workspace_for(dev, s, (size_t)windows * 4, &sync);
            if (rc) return rc;
            CUDA_TRY(cudaMemsetAsync(sync, 0, (size_t)windows * 4, s));
            gl.p.sync = sync;
            gl.p.sync_window = window;
        }
    }
    return rc;
}

// ------------------------------------------------------------------ skinny M: weight stream on the tensor cores
// skinny_tc_kernel (skinny_kernel.cuh): 128 weight columns per CTA, a three- or four-stage ring, two CTAs per SM.
// Measured on B200 against the 256-column and the deeper-ring variants, and against the
// tiled GEMM: it wins up to M = 48 on the decode shapes, and up to M = 64 where the column blocks run unsliced.
constexpr int kSkinnyClusterMarginPct = 92, kSkinnyMinKTilesPerSlice = 4, kSkinnyL2PostTiles = 2;
// Two CTAs per SM by shared memory (<= 112 KB each): a four-stage ring up to 32 activation rows, three stages for 33..64
// (8 KB of activations per stage, and up to 32 KB of hand-over buffer).  The occupancy calculator is no help here: for a
// kernel that allocates tensor memory it answers one CTA per SM (it cannot know how many columns), while
// the hardware co-schedules two (32 or 64 of 512 columns each; ncu: launch__occupancy_limit_shared_mem = 2).  How
// many CLUSTERS fit is a property of the GPC layout at two CTAs per SM, which the M = 1 kernel -- same
// occupancy, no tensor memory -- gets from the calculator: gemv_cluster_capacity.
constexpr int kSkinnyCtasPerSm = 2;
constexpr uint32_t kSkinnySmemLimit = (228 * 1024) / 2 - 1024;   // per CTA at two per SM, less the 1 KB the driver reserves
// Ring depth: four stages, three where that buys a CTA -- 33..64 rows (two CTAs per SM at all), and 17..32 rows on column
// blocks that run unsliced (61 KB: THREE CTAs per SM, so that e.g. the 400 column blocks of N = 51200 are one wave of the
// 444 slots instead of 1.35 waves of 296; measured at M = 32: 6.18 vs 5.52 TB/s, tiled GEMM 5.90).
inline int skinny_stages(int a_rows, bool unsliced) { return a_rows <= 16 ? 4 : a_rows == 32 ? (unsliced ? 3 : 4) : 3; }
inline uint32_t skinny_smem(int stages, int a_rows, int S, int mp) {
    return stages == 4 ? tg::SkinnySmem<4>::total(a_rows, S, mp) : tg::SkinnySmem<3>::total(a_rows, S, mp);
}
static_assert(tg::SkinnySmem<4>::total(32, tg::SKINNY_MAX_CLUSTER, 32) <= kSkinnySmemLimit, "two skinny CTAs must fit one SM's shared memory");
int gemv_cluster_capacity(int cs, int dev, int sms);

struct SkinnyPlan {
    bool ok = false;   // false: the tiled GEMM takes the shape
    int split = 1, col_blocks = 0, a_rows = 16, stages = 4;
};

// K slices of a skinny launch (tuning key 11 bits 8-15 force them).  Column blocks that fill the CTA slots
// (two per SM) run unsliced: the hardware scheduler and the next launch of the stream fill the slots as
// CTAs retire.  Fewer column blocks are cut into the largest number of slices (= cluster size) whose
// clusters all fit the device at once with slots to spare -- clusters of the next launch can only start
// where a whole cluster's worth of slots is free (the M = 1 kernel's rule).
SkinnyPlan plan_skinny(int64_t M, int64_t N, int64_t K, int dev, int sms) {
    SkinnyPlan sp;
    sp.a_rows = M <= 16 ? 16 : M <= 32 ? 32 : 64;
    const int tune = g_tune[11].load();
    const int want_split = (tune >> 8) & 255, want_rows = (tune >> 16) & 255;
    if ((want_rows == 32 || want_rows == 64) && want_rows > sp.a_rows) sp.a_rows = want_rows;
    const int mp = (int)((M + 3) & ~int64_t(3));
    const int64_t k_tiles = (K + tg::SKINNY_BK - 1) / tg::SKINNY_BK;
    const int64_t cb = (N + tg::SKINNY_COLS - 1) / tg::SKINNY_COLS;
    const int64_t slots1 = (int64_t)sms * kSkinnyCtasPerSm;
    if (cb > 0x7fffffff) return sp;
    sp.col_blocks = (int)cb;
    sp.split = 1;
    int margin = g_tune[10].load();
    if (margin <= 0) margin = kSkinnyClusterMarginPct;
    // Where the 128x128 tiles of the GEMM kernel are level or ahead (measured on the decode shapes; tuning
    // key 11 mode 2 overrides): 49..64 rows on weights that have to be sliced (within +-3 %).
    const bool unsliced = cb * 100 > slots1 * margin;
    if (want_split == 0 && (tune & 15) != 2 && M > 48 && !unsliced) return sp;
    sp.ok = true;
    sp.stages = skinny_stages(sp.a_rows, unsliced && want_split <= 1);
    if (((tune >> 24) & 15) == 3 || (((tune >> 24) & 15) == 4 && sp.a_rows <= 32)) sp.stages = (tune >> 24) & 15;   // key 11 bits 24-27
    if (want_split > 0) {
        sp.split = (int)(want_split < k_tiles ? want_split : k_tiles);
        if (sp.split > tg::SKINNY_MAX_CLUSTER) sp.split = tg::SKINNY_MAX_CLUSTER;
        while (sp.split > 1 && skinny_smem(sp.stages, sp.a_rows, sp.split, mp) > kSkinnySmemLimit) --sp.split;
        return sp;
    }
    for (int64_t cs = tg::SKINNY_MAX_CLUSTER; cs >= 2; --cs) {
        if (cs > k_tiles || k_tiles / cs < kSkinnyMinKTilesPerSlice) continue;
        if (skinny_smem(sp.stages, sp.a_rows, (int)cs, mp) > kSkinnySmemLimit) continue;   // the hand-over buffer of 33..64 rows: up to 5 slices
        if (cb * cs * 100 > slots1 * margin) continue;
        if (cb * 100 > (int64_t)gemv_cluster_capacity((int)cs, dev, sms) * margin) continue;
        sp.split = (int)cs;
        break;
    }
    return sp;
}

int run_skinny(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
               int64_t ldc, int in_dtype, int out_dtype, cudaStream_t s, int dev, const SkinnyPlan& sp, unsigned flags) {
    tg::SkinnyParams p;
    memset(&p, 0, sizeof p);
    p.C = C;
    p.ldc = ldc;
    p.M = (int32_t)M; p.N = (int32_t)N; p.K = (int32_t)K;
    p.k_tiles = (int32_t)((K + tg::SKINNY_BK - 1) / tg::SKINNY_BK);
    p.a_rows = sp.a_rows;
    p.out_kind = out_dtype;
    p.in_f16 = in_dtype == TILE_GEMM_IN_F16;
    p.flags = (flags & TILE_GEMM_FLAG_B_IMMUTABLE) ? tg::GEMV_FLAG_B_IMMUTABLE : 0;
    const int post = g_tune[9].load();                       // tuning key 9: n >= 1 -> n - 1 tiles
    p.l2_post = post > 0 ? post - 1 : kSkinnyL2PostTiles;
    CUtensorMap tw, tx;
    int rc = get_tensor_map(&tw, B, 2, false, (uint64_t)N, (uint64_t)K, (uint64_t)ldb * 2, 64u, 64u, 128);
    if (rc) return rc;
    rc = get_tensor_map(&tx, A, 2, false, (uint64_t)K, (uint64_t)M, (uint64_t)lda * 2, 64u, (uint32_t)sp.a_rows, 128);
    if (rc) return rc;
    const int smem = (int)skinny_smem(sp.stages, sp.a_rows, sp.split, (int)((M + 3) & ~int64_t(3)));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)sp.col_blocks, (unsigned)sp.split, 1);
    cfg.blockDim = dim3(tg::SKINNY_THREADS, 1, 1);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if ((g_tune[6].load() & 1) == 0) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (sp.split > 1) {   // the slices of a column block form one cluster along y
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = 1;
        attr[na].val.clusterDim.y = (unsigned)sp.split;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    static bool configured[64] = {};
    if (!configured[dev]) {
        CUDA_TRY(cudaFuncSetAttribute(tg::skinny_tc_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSkinnySmemLimit));
        CUDA_TRY(cudaFuncSetAttribute(tg::skinny_tc_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSkinnySmemLimit));
        configured[dev] = true;
    }
    if (sp.stages == 4) CUDA_TRY(cudaLaunchKernelEx(&cfg, tg::skinny_tc_kernel<4>, tw, tx, p));
    else CUDA_TRY(cudaLaunchKernelEx(&cfg, tg::skinny_tc_kernel<3>, tw, tx, p));
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

// does the weight-streaming tensor-core kernel take this GEMM shape?  (tuning key 11 bits 0-3: 1 = never, 2 = wherever it can run)
bool skinny_applies(int64_t M, int64_t K, const Plan& plan, bool force_repack) {
    if ((g_tune[11].load() & 15) == 1 || force_repack || !plan.a_tma || !plan.b_tma || K <= 0 || M > tg::SKINNY_MAX_ROWS) return false;
    const int forced_cfg = g_tune[0].load();
    return !(forced_cfg >= 1 && forced_cfg <= 4);   // a forced tile configuration means the tiled kernel
}

int c_tensor_map(CUtensorMap* tc, void* C, int64_t M, int64_t N, int64_t ldc, int out_16) {
    // one epilogue sub-chunk: 32 rows x 64 bytes, 64B-swizzled in shared memory (a 16-bit C is
    // described as bf16 whichever 16-bit format it holds: tiled TMA moves bits, it never converts)
    return get_tensor_map(tc, C, out_16 ? 2 : 4, !out_16, (uint64_t)N, (uint64_t)M,
                          (uint64_t)ldc * (out_16 ? 2 : 4), out_16 ? 32u : 16u, 32u, 64);
}

int run_gemm(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
             int64_t ldc, int in_dtype, int out_dtype, cudaStream_t s, const Plan& plan, bool force_repack, int dev,
             int sms, unsigned flags = 0u) {
    const int out_16 = out_dtype != TILE_GEMM_OUT_F32;
    if (skinny_applies(M, K, plan, force_repack)) {
        const SkinnyPlan sp = plan_skinny(M, N, K, dev, sms);
        if (sp.ok) return run_skinny(A, B, C, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, s, dev, sp, flags);
    }
    const bool rep_a = force_repack || !plan.a_tma;
    const bool rep_b = force_repack || !plan.b_tma;
    const uint16_t* Ap = (const uint16_t*)A;
    const uint16_t* Bp = (const uint16_t*)B;
    if (rep_a || rep_b) {
        const int64_t lda2 = (K + 7) & ~int64_t(7), ldb2 = (N + 7) & ~int64_t(7);
        const size_t a_sz = rep_a ? (((size_t)M * lda2 * 2 + 255) & ~(size_t)255) : 0;
        const size_t b_sz = rep_b ? (((size_t)K * ldb2 * 2 + 255) & ~(size_t)255) : 0;
        void* ws = nullptr;
        int rc = workspace_for(dev, s, a_sz + b_sz, &ws);
        if (rc) return rc;
        if (rep_a) {
            const int64_t chunks = M * (lda2 >> 3);
            const int64_t cap_blocks = (int64_t)sms * kAuxCtasPerSm;
            const int blocks = (int)((chunks + 255) / 256 < cap_blocks ? (chunks + 255) / 256 : cap_blocks);
            tg::repack_rows_kernel<<<blocks, 256, 0, s>>>(Ap, lda, (uint16_t*)ws, lda2, M, K);
            CUDA_TRY(cudaGetLastError());
            g_launches.fetch_add(1);
            Ap = (const uint16_t*)ws;
            lda = lda2;
        }
        if (rep_b) {
            uint16_t* dst = (uint16_t*)((char*)ws + a_sz);
            const int64_t chunks = K * (ldb2 >> 3);
            const int64_t cap_blocks = (int64_t)sms * kAuxCtasPerSm;
            const int blocks = (int)((chunks + 255) / 256 < cap_blocks ? (chunks + 255) / 256 : cap_blocks);
            tg::repack_rows_kernel<<<blocks, 256, 0, s>>>(Bp, ldb, dst, ldb2, K, N);
            CUDA_TRY(cudaGetLastError());
            g_launches.fetch_add(1);
            Bp = dst;
            ldb = ldb2;
        }
    }
    GemmLaunch gl;
    plan_gemm(M, N, K, in_dtype, out_dtype, dev, sms, &gl, true);
    if (gl.p.split > 0) {
        const size_t split_tiles = (size_t)((int64_t)gl.p.tiles_m * gl.p.tiles_n - gl.p.full_units);
        const size_t tile_floats = (size_t)tg::GEMM_BM * gl.cfg.cg * gl.cfg.tile_n();
        int rc2 = gemv_workspace_for(dev, s, split_tiles * gl.p.split * tile_floats * 4, split_tiles * gl.cfg.cg * 4 + 1024,
                                     &gl.p.partials, &gl.p.tickets);
        if (rc2) return rc2;
    }
    gl.p.tma_store = plan.c_tma ? 1 : 0;
    gl.p.C = C;
    gl.p.ldc = ldc;
    CUtensorMap ta, tb, tc;
    // skinny M: an A box only as tall as M needs (measured: 13 us of 36 at M <= 12, K = 5120, where the
    // 128-row box is almost all zero fill)
    gl.p.a_rows = M <= 16 ? 16 : M <= 32 ? 32 : M <= 64 ? 64 : 128;
    if (g_tune[6].load() & 32) gl.p.a_rows = 128;   // tuning key 6 bit 5: always the full box
    int rc = get_tensor_map(&ta, Ap, 2, false, (uint64_t)K, (uint64_t)M, (uint64_t)lda * 2, 64u, (uint32_t)gl.p.a_rows, 128);
    if (rc) return rc;
    rc = get_tensor_map(&tb, Bp, 2, false, (uint64_t)N, (uint64_t)K, (uint64_t)ldb * 2, 64u, 64u, 128);
    if (rc) return rc;
    if (plan.c_tma) {
        rc = c_tensor_map(&tc, C, M, N, ldc, out_16);
        if (rc) return rc;
    } else {
        tc = ta;   // never dereferenced by the clipped st.global epilogue; must still be a valid map
    }
    rc = setup_lockstep(gl, dev, s);
    if (rc) return rc;
    gl.p.trace = trace_for(s);                                     // tile_gemm_debug_trace: 8 words per cluster
    gl.p.trace_cap = (int32_t)g_trace_cap.load();
    return launch_gemm(gl, ta, tb, tc, s, dev);
}

// ------------------------------------------------------------------ GEMV launch
template <int COLS, int TILE_K, int STAGES, int MIN_CTAS, bool F16>
int launch_gemv_split(const void* B, int64_t N, int64_t K, int64_t ldb, tg::GemvSplitParams& p, int gx, int split,
                      bool pdl, cudaStream_t s, int dev) {
    using L = tg::GemvSplitSmem<COLS, TILE_K, STAGES>;
    auto kern = tg::gemv_split_kernel<COLS, TILE_K, STAGES, MIN_CTAS, F16>;
    static bool configured[64] = {};
    if (!configured[dev]) {
        CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::TOTAL));
        configured[dev] = true;
    }
    CUtensorMap tb;
    int rc = get_tensor_map(&tb, B, 2, false, (uint64_t)N, (uint64_t)K, (uint64_t)ldb * 2, (uint32_t)tg::GEMV_COLS,
                            (uint32_t)TILE_K, 0);
    if (rc) return rc;
    // x as a [1][K] tensor with a TILE_K-element box: zero fill past K, like the weight rows
    CUtensorMap tx = tb;
    if (p.flags & tg::GEMV_FLAG_X_TMA) {
        rc = get_tensor_map(&tx, p.x, 2, false, (uint64_t)K, 1, ((uint64_t)K * 2 + 15) & ~(uint64_t)15,
                            (uint32_t)TILE_K, 1u, 0);
        if (rc) return rc;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)gx, (unsigned)split, 1);
    cfg.blockDim = dim3(tg::GEMV_TMA_THREADS, 1, 1);
    cfg.dynamicSmemBytes = L::TOTAL;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (p.flags & tg::GEMV_FLAG_CLUSTER) {   // the slices of a column block form one cluster along y
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = 1;
        attr[na].val.clusterDim.y = (unsigned)split;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, tb, tx, p));
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

// clusters of `cs` CTAs of the default M = 1 kernel the device holds at once (occupancy calculator, cached)
int gemv_cluster_capacity(int cs, int dev, int sms) {
    static std::atomic<int> cache[tg::GEMV_MAX_CLUSTER + 1][64];
    if (cs < 1 || cs > tg::GEMV_MAX_CLUSTER) return 0;
    int v = cache[cs][dev].load();
    if (v > 0) return v;
    using L = tg::GemvSplitSmem<256, 64, 3>;
    auto kern = tg::gemv_split_kernel<256, 64, 3, 2, false>;
    int n = 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::TOTAL) == cudaSuccess) {
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3(64, (unsigned)cs, 1);
        cfg.blockDim = dim3(tg::GEMV_TMA_THREADS, 1, 1);
        cfg.dynamicSmemBytes = L::TOTAL;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 1;
        attr[0].val.clusterDim.y = (unsigned)cs;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) n = 0;
    }
    cudaGetLastError();
    if (n <= 0) n = (sms * 2) / (cs + 1);   // conservative guess
    cache[cs][dev].store(n);
    return n;
}

// CTAs of one ring shape of the split kernel that the CURRENT context can hold at once, from the occupancy
// calculator (it sees the shared-memory carve-out and the registers this build really uses) times the SM count;
// cached per device.  The tagged-slot hand-over is only taken when the whole launch fits this figure: its
// combiner CTAs poll for their column block's other slices, so those must be able to become resident.
template <int COLS, int TILE_K, int STAGES, int MIN_CTAS, bool F16>
int gemv_resident_ctas(int dev, int sms) {
    static std::atomic<int> cache[64];
    int v = cache[dev].load();
    if (v != 0) return v > 0 ? v : 0;
    using L = tg::GemvSplitSmem<COLS, TILE_K, STAGES>;
    auto kern = tg::gemv_split_kernel<COLS, TILE_K, STAGES, MIN_CTAS, F16>;
    int per_sm = 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L::TOTAL) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, tg::GEMV_TMA_THREADS, (size_t)L::TOTAL) != cudaSuccess)
        per_sm = 0;
    cudaGetLastError();
    v = per_sm > 0 ? per_sm * sms : -1;   // -1: unknown, treated as "nothing is provably resident"
    cache[dev].store(v);
    return v > 0 ? v : 0;
}

// measured on B200: two units into L2 behind the dependency wait; clusters sized to 92 % of capacity
// (same-process A/B of 80 / 88 / 92 / 96 / 100 %: 92 and 96 give N = 10240 six slices instead of five, +1.1 %; 100 % makes
// every other launch of N = 8192 run in two waves, -17 %)
constexpr int kGemvL2PostUnits = 2, kGemvClusterMarginPct = 92;

// ring shapes of the split kernel: {columns per CTA, rows per stage, stages, CTAs per SM}.  Round 3 keeps the three
// that compile without spills -- 2 is the default; 4 and 6 stay selectable (tuning key 5) because they exercise the
// NV = 2 column layout and the 16-row stage in the tests.  Ids 1, 3, 5, 7, 8 (measured slower, 4-432 B of spill
// stores each) are gone; asking for them gives the default.
struct GemvShape { int cols, tile_k, stages, occ; };
constexpr int kNumGemvShapes = 8;
const GemvShape kGemvShapes[kNumGemvShapes + 1] = {{0, 0, 0, 0},     {0, 0, 0, 0},    {256, 64, 3, 2},
                                                   {0, 0, 0, 0},     {512, 32, 3, 2}, {0, 0, 0, 0},
                                                   {512, 16, 4, 3},  {0, 0, 0, 0},    {0, 0, 0, 0}};

// Default M = 1 kernel: interleaved split-K over a (column block, slice) grid (gemv_kernel.cuh).
int run_gemv_split(const void* x, const void* B, void* y, int64_t N, int64_t K, int64_t ldb, int in_dtype,
                   int out_dtype, cudaStream_t s, int dev, int sms, unsigned flags) {
    int shape = g_tune[5].load();
    if (shape < 1 || shape > kNumGemvShapes || kGemvShapes[shape].cols == 0) shape = 2;
    const GemvShape gs = kGemvShapes[shape];
    const int64_t col_blocks = (N + gs.cols - 1) / gs.cols;
    const int64_t k_tiles = (K + gs.tile_k - 1) / gs.tile_k;
    // CTA budget: all CTAs co-resident
    int64_t budget = (int64_t)sms * gs.occ;
    const int cap = g_tune[2].load();
    if (cap > 0 && cap < budget) budget = cap;
    int64_t gx = col_blocks < budget ? col_blocks : budget;
    int64_t split = g_tune[3].load();
    if (split <= 0) {
        split = budget / gx;
        if (split == 1 && col_blocks <= budget && col_blocks * 2 > budget) {
            // Between half a wave and one wave of column blocks some SMs would hold two CTAs and the
            // others one; the single ones finish early and the rest of the launch runs latency bound
            // (measured: 200 blocks on 296 slots stream at 6.48 TB/s, 6.67 with four slices each).
            // Slice finer so that the CTAs come in waves the hardware scheduler balances, and pick
            // the slice count whose last wave is fullest; keep >= 16 tiles per CTA.
            double best = (double)col_blocks / (double)budget;
            for (int64_t c = 2; c <= 8 && k_tiles / c >= 16; ++c) {
                const double waves = (double)(col_blocks * c) / (double)budget;
                const double eff = waves / (double)(int64_t)(waves + 0.999999);
                if (eff > best + 0.05) { best = eff; split = c; }
            }
        }
    }
    // Fix-up protocol (gemv_kernel.cuh; tuning key 8: 0 auto, 1 tickets, 2 tagged slots else tickets, 3 cluster
    // else tickets).  Cluster: default ring shape, one column block per CTA, S <= 8 -- and when the automatic S is
    // within reach (<= 10) it becomes the largest cluster size whose clusters all fit the device at once with
    // slots to spare (key 10: per cent of the occupancy calculator's figure, default 92), because clusters of the
    // next kernel can only start where a whole cluster's worth of slots is free.
    const int fix_mode = g_tune[8].load();
    const bool cluster_ok = (fix_mode == 0 || fix_mode == 3) && shape == 2 && gx == col_blocks;
    if (cluster_ok && g_tune[3].load() <= 0 && split > 1 && split <= tg::GEMV_MAX_CLUSTER + 2) {
        int margin = g_tune[10].load();
        if (margin <= 0) margin = kGemvClusterMarginPct;
        for (int64_t cs = tg::GEMV_MAX_CLUSTER; cs >= 2; --cs)
            if (col_blocks * 100 <= (int64_t)gemv_cluster_capacity((int)cs, dev, sms) * margin && k_tiles / cs >= 4) {
                if (cs <= split) split = cs;
                break;
            }
    }
    if (split > k_tiles) split = k_tiles;
    if (split > 65535) split = 65535;
    if (split < 1) split = 1;
    tg::GemvSplitParams p;
    memset(&p, 0, sizeof p);
    p.x = (const uint16_t*)x;
    p.y = y;
    p.N = (int32_t)N;
    p.K = (int32_t)K;
    p.k_tiles = (int32_t)k_tiles;
    p.col_blocks = (int32_t)col_blocks;
    p.out_kind = out_dtype;
    p.flags = (flags & TILE_GEMM_FLAG_B_IMMUTABLE) ? tg::GEMV_FLAG_B_IMMUTABLE : 0;
    if ((((uintptr_t)x) & 15) == 0 && (g_tune[6].load() & 2) == 0) p.flags |= tg::GEMV_FLAG_X_TMA;
    p.trace = trace_for(s);
    p.trace_cap = (int32_t)g_trace_cap.load();
    const int post = g_tune[9].load();                       // tuning key 9: n >= 1 -> n - 1 units
    p.l2_post = post > 0 ? post - 1 : kGemvL2PostUnits;
    if (split > 1) {
        int rc = TILE_GEMM_OK;
        const bool f16_in = in_dtype == TILE_GEMM_IN_F16;
        int64_t resident = 0;
        if (!(cluster_ok && split <= tg::GEMV_MAX_CLUSTER) && (fix_mode == 0 || fix_mode == 2)) {
#define TG_GEMV_RES(id, C, T, ST, O)                                                                  \
    case id:                                                                                          \
        resident = f16_in ? gemv_resident_ctas<C, T, ST, O, true>(dev, sms)                           \
                          : gemv_resident_ctas<C, T, ST, O, false>(dev, sms);                         \
        break;
            switch (shape) {
                TG_GEMV_RES(2, 256, 64, 3, 2)
                TG_GEMV_RES(4, 512, 32, 3, 2)
                TG_GEMV_RES(6, 512, 16, 4, 3)
            }
#undef TG_GEMV_RES
        }
        if (cluster_ok && split <= tg::GEMV_MAX_CLUSTER) {
            p.flags |= tg::GEMV_FLAG_CLUSTER;
        } else if ((fix_mode == 0 || fix_mode == 2) && gx * split <= budget && gx * split <= resident) {
            // tagged slots: the designated combiner polls, so every CTA of the launch must fit the device at once
            // -- by the nominal figure the plan was made with AND by what the occupancy calculator reports for this
            // context.  Anything that is not provably one wave keeps the tickets, which cannot wait on anybody.
            rc = packed_workspace_for(dev, s, (size_t)col_blocks * split * gs.cols * 8, &p.packed);
            p.flags |= tg::GEMV_FLAG_PACKED;
        } else {
            rc = gemv_workspace_for(dev, s, (size_t)col_blocks * split * gs.cols * 4, (size_t)col_blocks * 4,
                                    &p.partials, &p.tickets);
        }
        if (rc) return rc;
    }
    const bool pdl = (g_tune[6].load() & 1) == 0;
    const bool f16 = in_dtype == TILE_GEMM_IN_F16;
#define TG_GEMV_CASE(id, C, T, ST, O)                                                                        \
    case id:                                                                                                 \
        return f16 ? launch_gemv_split<C, T, ST, O, true>(B, N, K, ldb, p, (int)gx, (int)split, pdl, s, dev) \
                   : launch_gemv_split<C, T, ST, O, false>(B, N, K, ldb, p, (int)gx, (int)split, pdl, s, dev);
    switch (shape) {
        TG_GEMV_CASE(2, 256, 64, 3, 2)
        TG_GEMV_CASE(4, 512, 32, 3, 2)
        TG_GEMV_CASE(6, 512, 16, 4, 3)
    }
#undef TG_GEMV_CASE
    return fail(TILE_GEMM_E_INTERNAL, "unknown GEMV ring shape %d", shape);
}

int run_gemv(const void* x, const void* B, void* y, int64_t N, int64_t K, int64_t ldb, int in_dtype, int out_dtype,
             cudaStream_t s, const Plan& plan, int dev, int sms, unsigned flags) {
    const bool f16 = in_dtype == TILE_GEMM_IN_F16;
    int variant = g_tune[4].load();   // 0 auto, 2 LDG 16-byte, 3 LDG scalar, 1 / 4 the TMA ring with interleaved split-K
    if (plan.b_tma && (variant == 0 || variant == 1 || variant == 4))
        return run_gemv_split(x, B, y, N, K, ldb, in_dtype, out_dtype, s, dev, sms, flags);
    tg::GemvParams p;
    p.x = (const uint16_t*)x;
    p.B = (const uint16_t*)B;
    p.y = y;
    p.N = (int32_t)N;
    p.K = (int32_t)K;
    p.ldb = ldb;
    p.out_kind = out_dtype;
    if (!plan.b_tma || variant != 2) variant = 3;   // 2 = 16-byte loads (needs 16-byte addressable rows), else scalar loads
    const int64_t xblocks = (N + tg::GEMV_COLS - 1) / tg::GEMV_COLS;
    // split-K: as many slices as keep every CTA co-resident (2 per SM) with >= 2 tiles each
    int split = g_tune[3].load();
    if (split <= 0) {
        split = 1;
        const int64_t slots = (int64_t)sms * 2;
        for (int c = 2; c <= 8; ++c)
            if (xblocks * c <= slots && K / c >= 2 * tg::GEMV_TILE_K) split = c;
    }
    if (split > 8) split = 8;
    int64_t kper = (K + split - 1) / split;
    kper = (kper + tg::GEMV_TILE_K - 1) / tg::GEMV_TILE_K * tg::GEMV_TILE_K;
    split = (int)((K + kper - 1) / kper);
    p.k_per_cta = (int32_t)kper;

    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)xblocks, (unsigned)split, 1);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 1;
    attr[0].val.clusterDim.y = (unsigned)split;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    {
        cfg.blockDim = dim3(256, 1, 1);
        cfg.dynamicSmemBytes = 0;
        auto kern = variant == 2 ? (f16 ? tg::gemv_ldg_kernel<true, true> : tg::gemv_ldg_kernel<true, false>)
                                 : (f16 ? tg::gemv_ldg_kernel<false, true> : tg::gemv_ldg_kernel<false, false>);
        CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, p));
    }
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

int run_zero(void* C, int64_t M, int64_t N, int64_t ldc, int esize, cudaStream_t s, int sms) {
    const int64_t total = M * N;
    const int64_t cap_blocks = (int64_t)sms * kAuxCtasPerSm / 2;
    const int blocks = (int)((total + 255) / 256 < cap_blocks ? (total + 255) / 256 : cap_blocks);
    tg::zero_fill_kernel<<<blocks, 256, 0, s>>>(C, M, N, ldc, esize);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

}  // namespace

// ====================================================================== C ABI
extern "C" {

int tile_gemm_select(int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb, int64_t ldc, const void* A,
                     const void* B, const void* C, int out_dtype) {
    Plan plan;
    const int rc = check_and_select(A, B, C, M, N, K, lda, ldb, ldc, TILE_GEMM_IN_BF16, out_dtype, &plan);
    return rc ? -rc : plan.path;
}

}  // extern "C"

namespace {
int gemm_entry(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
               int64_t ldc, int in_dtype, int out_dtype, void* stream, int force_path, unsigned flags) {
    Plan plan;
    int rc = check_and_select(A, B, C, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, &plan);
    if (rc) return rc;
    if (force_path < TILE_GEMM_PATH_AUTO || force_path > TILE_GEMM_PATH_GEMV)
        return fail(TILE_GEMM_E_PATH, "force_path=%d is not AUTO, GEMM_TMA, GEMM_REPACK or GEMV", force_path);
    if (plan.path == TILE_GEMM_PATH_NOOP) return TILE_GEMM_OK;
    int path = plan.path;
    if (force_path != TILE_GEMM_PATH_AUTO && path != TILE_GEMM_PATH_ZERO) {
        if (force_path == TILE_GEMM_PATH_GEMV && M != 1)
            return fail(TILE_GEMM_E_PATH, "the GEMV path needs M == 1 (M=%lld)", (long long)M);
        if (force_path == TILE_GEMM_PATH_GEMM_TMA && !(plan.a_tma && plan.b_tma))
            return fail(TILE_GEMM_E_PATH, "GEMM_TMA needs 16-byte aligned A/B with lda, ldb multiples of 8");
        path = force_path;
    }
    int dev = 0, sms = 0;
    rc = current_device(&dev, &sms);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    switch (path) {
        case TILE_GEMM_PATH_ZERO: return run_zero(C, M, N, ldc, plan.esize, s, sms);
        case TILE_GEMM_PATH_GEMV:
            return run_gemv(A, B, C, N, K, ldb, in_dtype, out_dtype, s, plan, dev, sms, flags);
        case TILE_GEMM_PATH_GEMM_TMA:
            return run_gemm(A, B, C, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, s, plan, false, dev, sms, flags);
        case TILE_GEMM_PATH_GEMM_REPACK:   // forced: repack both operands; auto: only what TMA cannot address
            return run_gemm(A, B, C, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, s, plan,
                            force_path == TILE_GEMM_PATH_GEMM_REPACK, dev, sms, flags);
    }
    return fail(TILE_GEMM_E_INTERNAL, "unhandled path %d", path);
}
}  // namespace

extern "C" {

int tile_gemm_ex(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
                 int64_t ldc, int out_dtype, void* stream, int force_path) {
    return gemm_entry(A, B, C, M, N, K, lda, ldb, ldc, TILE_GEMM_IN_BF16, out_dtype, stream, force_path, 0u);
}

int tile_gemm_static_b(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda,
                       int64_t ldb, int64_t ldc, int out_dtype, void* stream) {
    return gemm_entry(A, B, C, M, N, K, lda, ldb, ldc, TILE_GEMM_IN_BF16, out_dtype, stream, TILE_GEMM_PATH_AUTO,
                      TILE_GEMM_FLAG_B_IMMUTABLE);
}

int tile_gemm(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
              int64_t ldc, int out_dtype, void* stream) {
    return tile_gemm_ex(A, B, C, M, N, K, lda, ldb, ldc, out_dtype, stream, TILE_GEMM_PATH_AUTO);
}

int tile_gemm_typed(const void* A, const void* B, void* C, int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
                    int64_t ldc, int in_dtype, int out_dtype, void* stream) {
    return gemm_entry(A, B, C, M, N, K, lda, ldb, ldc, in_dtype, out_dtype, stream, TILE_GEMM_PATH_AUTO, 0u);
}

// tile_add_f32 launch shape (measured on B200 at n = 2^28)
constexpr int kAddDefaultPerSm = 255, kAddDefaultUnroll = 1, kAddDefaultMode = 1;

int tile_gemm_swiglu(const void* X, const void* Wgu, void* H, int64_t M, int64_t I, int64_t K, int64_t ldx,
                     int64_t ldw, int64_t ldh, int out_dtype, void* stream) {
    // the preconditions of tile_gemm on (X, Wgu[:, :I], H), then the ones the second half adds
    Plan plan;
    int rc = check_and_select(X, Wgu, H, M, I, K, ldx, ldw, ldh, TILE_GEMM_IN_BF16, out_dtype, &plan);
    if (rc) return rc;
    if (I > ((int64_t)INT32_MAX - 1024) / 2)
        return fail(TILE_GEMM_E_OVERFLOW, "2*I = %lld columns of the fused weight overflow int32", (long long)(2 * I));
    if (ldw < 2 * I) return fail(TILE_GEMM_E_LDB, "ldw=%lld < 2*I=%lld", (long long)ldw, (long long)(2 * I));
    int64_t w_bytes = 0;
    if (!span_bytes(K, 2 * I, ldw, 2, &w_bytes)) return fail(TILE_GEMM_E_OVERFLOW, "operand byte span overflows int64");
    if (overlaps(H, plan.c_bytes, Wgu, w_bytes))
        return fail(TILE_GEMM_E_ALIAS, "H [%p,+%lld) overlaps Wgu [%p,+%lld): the output must be exclusively owned", H,
                    (long long)plan.c_bytes, Wgu, (long long)w_bytes);
    if (plan.path == TILE_GEMM_PATH_NOOP) return TILE_GEMM_OK;
    if (K > 0 && !(plan.a_tma && plan.b_tma))
        return fail(TILE_GEMM_E_PATH,
                    "tile_gemm_swiglu needs 16-byte aligned X and Wgu with ldx and ldw multiples of 8 (no repack path)");
    if (K > 0 && I % 8 != 0)   // the up half is read through TMA boxes that start at column I: 16-byte granularity (measured)
        return fail(TILE_GEMM_E_PATH, "tile_gemm_swiglu needs I (%lld) to be a multiple of 8", (long long)I);
    int dev = 0, sms = 0;
    rc = current_device(&dev, &sms);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if (K == 0) return run_zero(H, M, I, ldh, plan.esize, s, sms);   // silu(0) * 0 = 0
    GemmLaunch gl;
    gl.cfg = kConfigs[4];
    tg::GemmParams& p = gl.p;
    memset(&p, 0, sizeof p);
    p.M = (int32_t)M; p.N = (int32_t)I; p.K = (int32_t)K;
    p.tiles_m = (int32_t)((M + 255) / 256);
    p.tiles_n = (int32_t)((I + 255) / 256);            // the output tile is 256 x 256: gate and up slots side by side in TMEM
    int gm = g_tune[1].load();
    if (gm <= 0) gm = 16;
    p.group_m = gm < p.tiles_m ? gm : p.tiles_m;
    p.num_k_tiles = (int32_t)((K + tg::GEMM_BK - 1) / tg::GEMM_BK);
    p.out_16 = out_dtype != TILE_GEMM_OUT_F32;
    p.out_f16 = out_dtype == TILE_GEMM_OUT_F16;
    p.up_offset = (int32_t)I;
    const int64_t tiles = (int64_t)p.tiles_m * p.tiles_n;
    p.full_units = p.total_units = (int32_t)tiles;
    p.kps = p.num_k_tiles;
    const int64_t slots = resident_units(gl.cfg.id, dev, sms);
    const int64_t clusters = tiles < slots ? tiles : slots;
    gl.ctas = (int)clusters * 2;
    p.tma_store = plan.c_tma ? 1 : 0;
    p.C = H;
    p.ldc = ldh;
    CUtensorMap ta, tb, tc;
    p.a_rows = 128;
    rc = get_tensor_map(&ta, X, 2, false, (uint64_t)K, (uint64_t)M, (uint64_t)ldx * 2, 64u, 128u, 128);
    if (rc) return rc;
    rc = get_tensor_map(&tb, Wgu, 2, false, (uint64_t)(2 * I), (uint64_t)K, (uint64_t)ldw * 2, 64u, 64u, 128);
    if (rc) return rc;
    if (plan.c_tma) {
        rc = c_tensor_map(&tc, H, M, I, ldh, p.out_16);
        if (rc) return rc;
    } else {
        tc = ta;
    }
    rc = setup_lockstep(gl, dev, s);
    if (rc) return rc;
    return launch_gemm_inst<2, 256, 4, 2, false, 1>(ta, tb, tc, p, gl.ctas, s, dev);
}

int tile_read_probe_u32(const uint32_t* buf, int64_t n, unsigned long long* out_sum, void* stream) {
    if (n < 0) return fail(TILE_GEMM_E_EXTENT, "negative extent: n=%lld", (long long)n);
    if (!out_sum) return fail(TILE_GEMM_E_NULL, "out_sum is NULL");
    if (n > 0 && !buf) return fail(TILE_GEMM_E_NULL, "buf is NULL but n > 0");
    if (((uintptr_t)buf & 15) || ((uintptr_t)out_sum & 7))
        return fail(TILE_GEMM_E_ALIGN, "buf (%p) must be 16-byte and out_sum (%p) 8-byte aligned", (const void*)buf, (void*)out_sum);
    if (n > (int64_t(1) << 40)) return fail(TILE_GEMM_E_OVERFLOW, "n=%lld above 2^40 words", (long long)n);
    if (overlaps(out_sum, 8, buf, n * 4)) return fail(TILE_GEMM_E_ALIAS, "out_sum lies inside buf");
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    if (n == 0) return TILE_GEMM_OK;
    const int64_t tile = (int64_t)tg::PROBE_THREADS * tg::PROBE_UNROLL;
    const int64_t grid = ((n >> 2) + tile - 1) / tile + ((n >> 2) % tile == 0 ? 1 : 0);   // the last CTA also owns the < 4-word tail
    tg::read_probe_kernel<<<(unsigned)grid, tg::PROBE_THREADS, 0, (cudaStream_t)stream>>>(buf, n, out_sum);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

int tile_add_f32(const float* x, const float* y, float* z, int64_t n, void* stream) {
    if (n < 0) return fail(TILE_GEMM_E_EXTENT, "negative extent: n=%lld", (long long)n);
    if (n == 0) return TILE_GEMM_OK;
    if (n > (int64_t(1) << 40)) return fail(TILE_GEMM_E_OVERFLOW, "n=%lld above 2^40 elements", (long long)n);
    if (!x || !y || !z) return fail(TILE_GEMM_E_NULL, "x (%p), y (%p) or z (%p) is NULL but n > 0", x, y, z);
    if (((uintptr_t)x | (uintptr_t)y | (uintptr_t)z) & 3)
        return fail(TILE_GEMM_E_ALIGN, "x (%p), y (%p) or z (%p) is not 4-byte aligned", x, y, z);
    if (overlaps(z, n * 4, x, n * 4) || overlaps(z, n * 4, y, n * 4))
        return fail(TILE_GEMM_E_ALIAS, "z [%p,+%lld) overlaps x (%p) or y (%p): the output must be exclusively owned",
                    z, (long long)(n * 4), x, y);
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const uintptr_t all = (uintptr_t)x | (uintptr_t)y | (uintptr_t)z;
    const bool vec = (all & 15) == 0;
    // tuning key 7: bits 0-3 vectors per thread, bits 4-11 CTAs per SM (255 = one tile per CTA),
    // bits 12-15 mode (0 auto, 1 = 128-bit + hints, 2 = 128-bit plain, 3 = 256-bit + hints, 4 = 256-bit plain)
    const int tune = g_tune[7].load();
    int unroll = tune & 15, per_sm = (tune >> 4) & 255, mode = (tune >> 12) & 15;
    if (per_sm <= 0) per_sm = kAddDefaultPerSm;
    if (unroll != 1 && unroll != 2 && unroll != 4 && unroll != 8) unroll = kAddDefaultUnroll;
    if (mode < 1 || mode > 4) mode = kAddDefaultMode;
    if ((mode == 3 || mode == 4) && (all & 31)) mode -= 2;   // 256-bit accesses need 32-byte alignment
    if (vec) {
        const int vw = mode >= 3 ? 8 : 4;
        const int64_t tile = (int64_t)tg::ADD_THREADS * unroll * vw;
        const int64_t tiles = (n + tile - 1) / tile;
        int64_t grid = per_sm == 255 ? tiles : (int64_t)sms * per_sm;
        if (grid > tiles) grid = tiles;
        if (grid > 0x7fffffff) grid = 0x7fffffff;
        if (grid < 1) grid = 1;
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3((unsigned)grid, 1, 1);
        cfg.blockDim = dim3(tg::ADD_THREADS, 1, 1);
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = (g_tune[6].load() & 1) ? 0 : 1;   // tuning key 6 bit 0: no programmatic dependent launch
#define TG_ADD_CASE(U, VW, H) CUDA_TRY(cudaLaunchKernelEx(&cfg, tg::add_f32_vec_kernel<U, VW, H>, x, y, z, n))
#define TG_ADD_MODE(U)                                      \
    switch (mode) {                                         \
        case 1: TG_ADD_CASE(U, 4, true); break;             \
        case 2: TG_ADD_CASE(U, 4, false); break;            \
        case 3: TG_ADD_CASE(U, 8, true); break;             \
        default: TG_ADD_CASE(U, 8, false); break;           \
    }
        switch (unroll) {
            case 1: TG_ADD_MODE(1) break;
            case 2: TG_ADD_MODE(2) break;
            case 4: TG_ADD_MODE(4) break;
            default: TG_ADD_MODE(8) break;
        }
#undef TG_ADD_MODE
#undef TG_ADD_CASE
    } else {
        int64_t grid = (n + tg::ADD_THREADS - 1) / tg::ADD_THREADS;
        if (grid > (int64_t)sms * 8) grid = (int64_t)sms * 8;
        tg::add_f32_scalar_kernel<<<(unsigned)grid, tg::ADD_THREADS, 0, s>>>(x, y, z, n);
    }
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

// ---------------------------------------------------------------- recorded steps
namespace {
struct Recorded {
    uint32_t magic;
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    int64_t nodes;
    Recording* rec;   // the step's private workspaces: every address its nodes hold lives as long as the step
};
constexpr uint32_t kRecordedMagic = 0x7167656d;
}  // namespace

int tile_gemm_record_begin(void* stream) {
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    if (stream == nullptr)
        return fail(TILE_GEMM_E_PATH, "recording needs an explicit stream: the legacy default stream cannot be captured");
    {
        std::lock_guard<std::mutex> lk(g_mu);
        if (g_recording.count((uintptr_t)stream))
            return fail(TILE_GEMM_E_PATH, "stream %p is already recording a step", stream);
    }
    // relaxed mode: the step's private workspaces are allocated (cudaMalloc) while the stream captures
    CUDA_TRY(cudaStreamBeginCapture((cudaStream_t)stream, cudaStreamCaptureModeRelaxed));
    Recording* rec = new Recording();
    rec->dev = dev;
    std::lock_guard<std::mutex> lk(g_mu);
    g_recording[(uintptr_t)stream] = rec;
    return TILE_GEMM_OK;
}

int tile_gemm_record_end(void* stream, void** step_out) {
    if (!step_out) return fail(TILE_GEMM_E_NULL, "step_out is NULL");
    *step_out = nullptr;
    Recording* rec = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_recording.find((uintptr_t)stream);
        if (it == g_recording.end())
            return fail(TILE_GEMM_E_PATH, "stream %p is not recording (tile_gemm_record_begin was not called on it)", stream);
        rec = it->second;
        g_recording.erase(it);
    }
    auto drop = [&]() {
        free_workspace_set(rec->ws);
        delete rec;
    };
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture((cudaStream_t)stream, &graph);
    if (e != cudaSuccess || !graph) {
        drop();
        return fail(TILE_GEMM_E_CUDA, "the capture on this stream was invalidated: %s (%d)", cudaGetErrorString(e), (int)e);
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    if (e != cudaSuccess) {
        cudaGraphDestroy(graph);
        drop();
        return fail(TILE_GEMM_E_CUDA, "cudaGraphInstantiate failed: %s (%d)", cudaGetErrorString(e), (int)e);
    }
    size_t n = 0;
    cudaGraphGetNodes(graph, nullptr, &n);
    Recorded* r = new Recorded{kRecordedMagic, graph, exec, (int64_t)n, rec};
    *step_out = r;
    return TILE_GEMM_OK;
}

int tile_gemm_replay(void* step, void* stream) {
    Recorded* r = (Recorded*)step;
    if (!r || r->magic != kRecordedMagic) return fail(TILE_GEMM_E_NULL, "not a recorded step: %p", step);
    CUDA_TRY(cudaGraphLaunch(r->exec, (cudaStream_t)stream));
    g_launches.fetch_add(r->nodes);
    return TILE_GEMM_OK;
}

int64_t tile_gemm_recorded_nodes(void* step) {
    Recorded* r = (Recorded*)step;
    return (r && r->magic == kRecordedMagic) ? r->nodes : -1;
}

int tile_gemm_record_free(void* step) {
    Recorded* r = (Recorded*)step;
    if (!r) return TILE_GEMM_OK;
    if (r->magic != kRecordedMagic) return fail(TILE_GEMM_E_NULL, "not a recorded step: %p", step);
    cudaGraphExecDestroy(r->exec);
    cudaGraphDestroy(r->graph);
    if (r->rec) {
        free_workspace_set(r->rec->ws);   // cudaFree synchronises with replays still in flight
        delete r->rec;
    }
    r->magic = 0;
    delete r;
    return TILE_GEMM_OK;
}

constexpr int64_t kHostChunkRows = 1024, kHostTailRows = 128;

int tile_gemm_host(const void* A_host, const void* B_host, void* C_host, int64_t M, int64_t N, int64_t K,
                   int64_t lda, int64_t ldb, int64_t ldc, int out_dtype) {
    Plan plan;
    int rc = check_and_select(A_host, B_host, C_host, M, N, K, lda, ldb, ldc, TILE_GEMM_IN_BF16, out_dtype, &plan);
    if (rc) return rc;
    if (plan.path == TILE_GEMM_PATH_NOOP) return TILE_GEMM_OK;
    int dev = 0, sms = 0;
    rc = current_device(&dev, &sms);
    if (rc) return rc;
    // One host call at a time PER DEVICE: the staging buffers, the three streams and the events of the
    // current device are used for the whole call.  Threads that target the same GPU block here (they
    // would share its PCIe link anyway) and never see each other's staging data; threads on different
    // GPUs share nothing and run side by side.
    HostStage& hs = g_host[dev];
    std::lock_guard<std::mutex> host_lk(hs.mu);
    if (!hs.in) CUDA_TRY(cudaStreamCreateWithFlags(&hs.in, cudaStreamNonBlocking));
    if ((rc = grow(hs.a, (size_t)plan.a_bytes + 16))) return rc;
    if ((rc = grow(hs.b, (size_t)plan.b_bytes + 16))) return rc;
    if ((rc = grow(hs.c, (size_t)plan.c_bytes + 16))) return rc;
    cudaStream_t s = hs.in;
    // Large M: rows of A go up in chunks, each chunk's GEMM starts as soon as its rows (and all of B)
    // have landed, and its rows of C go back while the next chunk is still coming in.  PCIe is full
    // duplex, so the call costs about max(H2D, D2H) instead of H2D + GEMM + D2H.  Every chunk is an
    // ordinary tile_gemm call that plans itself (tile configuration, K slices), so the fp32 bits may
    // differ from one whole-problem call by a different summation order: same tolerance, and the
    // same bits for integer-valued inputs.
    const int64_t chunk = kHostChunkRows;
    if (K > 0 && M >= 2 * chunk && (g_tune[6].load() & 64) == 0) {   // tuning key 6 bit 6: one shot
        // chunk heights: kHostChunkRows while more than that is left, then the rest halves down to
        // kHostTailRows -- what follows the last uploaded byte (that chunk's GEMM and its copy-out) is the only
        // part of the call nothing overlaps, so the last chunk is small
        std::vector<int64_t> heights;
        int64_t left = M;
        while (left > chunk) { heights.push_back(chunk); left -= chunk; }
        while (left > 2 * kHostTailRows) { heights.push_back(left / 2); left -= left / 2; }
        if (left > kHostTailRows) { heights.push_back(left - kHostTailRows); left = kHostTailRows; }
        heights.push_back(left);
        const int64_t nchunks = (int64_t)heights.size();
        if (!hs.compute) CUDA_TRY(cudaStreamCreateWithFlags(&hs.compute, cudaStreamNonBlocking));
        if (!hs.out) CUDA_TRY(cudaStreamCreateWithFlags(&hs.out, cudaStreamNonBlocking));
        while ((int64_t)hs.events.size() < 2 * nchunks + 1) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            hs.events.push_back(e);
        }
        const char* Ah = (const char*)A_host;
        char* Ch = (char*)C_host;
        char* Ad = (char*)hs.a.p;
        char* Cd = (char*)hs.c.p;
        CUDA_TRY(cudaMemcpyAsync(hs.b.p, B_host, (size_t)plan.b_bytes, cudaMemcpyHostToDevice, s));
        int64_t r0 = 0;
        for (int64_t i = 0; i < nchunks; ++i) {
            const int64_t rows = heights[i];
            const size_t a_off = (size_t)r0 * lda * 2, a_len = ((size_t)(rows - 1) * lda + K) * 2;
            CUDA_TRY(cudaMemcpyAsync(Ad + a_off, Ah + a_off, a_len, cudaMemcpyHostToDevice, s));
            CUDA_TRY(cudaEventRecord(hs.events[2 * i], s));
            CUDA_TRY(cudaStreamWaitEvent(hs.compute, hs.events[2 * i], 0));
            rc = tile_gemm(Ad + a_off, hs.b.p, Cd + (size_t)r0 * ldc * plan.esize, rows, N, K, lda, ldb, ldc, out_dtype,
                           (void*)hs.compute);
            if (rc) { cudaDeviceSynchronize(); return rc; }
            CUDA_TRY(cudaEventRecord(hs.events[2 * i + 1], hs.compute));
            CUDA_TRY(cudaStreamWaitEvent(hs.out, hs.events[2 * i + 1], 0));
            CUDA_TRY(cudaMemcpy2DAsync(Ch + (size_t)r0 * ldc * plan.esize, (size_t)ldc * plan.esize,
                                       Cd + (size_t)r0 * ldc * plan.esize, (size_t)ldc * plan.esize,
                                       (size_t)N * plan.esize, (size_t)rows, cudaMemcpyDeviceToHost, hs.out));
            r0 += rows;
        }
        CUDA_TRY(cudaStreamSynchronize(hs.out));
        CUDA_TRY(cudaStreamSynchronize(s));
        return TILE_GEMM_OK;
    }
    if (plan.a_bytes) CUDA_TRY(cudaMemcpyAsync(hs.a.p, A_host, (size_t)plan.a_bytes, cudaMemcpyHostToDevice, s));
    if (plan.b_bytes) CUDA_TRY(cudaMemcpyAsync(hs.b.p, B_host, (size_t)plan.b_bytes, cudaMemcpyHostToDevice, s));
    rc = tile_gemm(hs.a.p, hs.b.p, hs.c.p, M, N, K, lda, ldb, ldc, out_dtype, (void*)s);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpy2DAsync(C_host, (size_t)ldc * plan.esize, hs.c.p, (size_t)ldc * plan.esize,
                               (size_t)N * plan.esize, (size_t)M, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return TILE_GEMM_OK;
}

int tile_gemm_query_config(int64_t M, int64_t N, int64_t K, int out_dtype, int32_t out[8]) {
    if (M <= 0 || N <= 0 || K < 0 || !out) return fail(TILE_GEMM_E_EXTENT, "query needs M, N > 0, K >= 0");
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    GemmLaunch gl;
    plan_gemm(M, N, K, TILE_GEMM_IN_BF16, out_dtype, dev, sms, &gl);
    out[0] = tg::GEMM_BM;
    out[1] = gl.cfg.tile_n();
    out[2] = gl.cfg.cg;
    out[3] = gl.ctas;
    out[4] = gl.p.group_m;
    out[5] = gl.cfg.stages;
    out[6] = tg::GEMM_BK;
    out[7] = gl.mc ? 6 : gl.cfg.id;
    return TILE_GEMM_OK;
}

int tile_gemm_query_plan(int64_t M, int64_t N, int64_t K, int32_t out[8]) {
    if (M <= 1 || N <= 0 || K <= 0 || !out) return fail(TILE_GEMM_E_EXTENT, "the plan query needs M >= 2, N > 0, K > 0");
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    {   // skinny M with TMA-addressable operands (assumed here: the query sees no pointers): the weight-streaming kernel
        Plan aligned;
        aligned.a_tma = aligned.b_tma = true;
        if (skinny_applies(M, K, aligned, false)) {
            const SkinnyPlan sp = plan_skinny(M, N, K, dev, sms);
            if (sp.ok) {
                const int64_t k_tiles = (K + tg::SKINNY_BK - 1) / tg::SKINNY_BK;
                out[0] = 5;
                out[1] = sp.col_blocks * sp.split;
                out[2] = 0;
                out[3] = sp.split > 1 ? sp.split : 0;
                out[4] = (int32_t)((k_tiles + sp.split - 1) / sp.split);
                out[5] = 0;
                out[6] = 0;
                out[7] = sp.a_rows;
                return TILE_GEMM_OK;
            }
        }
    }
    GemmLaunch gl;
    plan_gemm(M, N, K, TILE_GEMM_IN_BF16, TILE_GEMM_OUT_BF16, dev, sms, &gl, true);
    int64_t rounds = 0;
    int window = 0;
    lockstep_plan(gl, &rounds, &window);
    out[0] = gl.cfg.id;
    out[1] = gl.ctas;
    out[2] = gl.p.full_units;
    out[3] = gl.p.split;
    out[4] = gl.p.kps;
    out[5] = (int32_t)rounds;
    out[6] = rounds > 0 ? window : 0;
    out[7] = M <= 16 ? 16 : M <= 32 ? 32 : M <= 64 ? 64 : 128;
    return TILE_GEMM_OK;
}

int tile_gemm_debug_owner_map(int32_t* owner, int64_t M, int64_t N, int64_t K, int64_t ld_owner, int out_dtype,
                              void* stream) {
    if (M <= 0 || N <= 0 || K < 0) return fail(TILE_GEMM_E_EXTENT, "owner map needs M, N > 0, K >= 0");
    if (!owner) return fail(TILE_GEMM_E_NULL, "owner is NULL");
    if (ld_owner < N) return fail(TILE_GEMM_E_LDC, "ld_owner=%lld < N=%lld", (long long)ld_owner, (long long)N);
    if ((uintptr_t)owner & 3) return fail(TILE_GEMM_E_ALIGN, "owner (%p) is not 4-byte aligned", (void*)owner);
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    GemmLaunch gl;
    plan_gemm(M, N, K, TILE_GEMM_IN_BF16, out_dtype, dev, sms, &gl);
    gl.p.num_k_tiles = 0;   // same schedule and epilogue, no loads and no MMAs
    gl.p.out_16 = 0;        // the map itself is written through the 32-bit epilogue
    gl.p.out_f16 = 0;
    gl.p.owner_mode = 1;
    gl.p.C = owner;
    gl.p.ldc = ld_owner;
    const bool c_tma = (((uintptr_t)owner & 15) == 0) && ((ld_owner * 4) % 16 == 0);
    gl.p.tma_store = c_tma ? 1 : 0;
    CUtensorMap tc;
    if (c_tma) {
        rc = c_tensor_map(&tc, owner, M, N, ld_owner, 0);
    } else {
        // any valid descriptor: it is prefetched but never used by the clipped-store epilogue
        static void* dummy = nullptr;
        if (!dummy) CUDA_TRY(cudaMalloc(&dummy, 32 * 128));
        rc = get_tensor_map(&tc, dummy, 4, true, 32, 32, 128, 16u, 32u, 64);
    }
    if (rc) return rc;
    return launch_gemm(gl, tc, tc, tc, (cudaStream_t)stream, dev);
}

int tile_gemm_debug_occupy(int ctas, int64_t ns, void* stream) {
    if (ctas < 0 || ns < 0) return fail(TILE_GEMM_E_EXTENT, "negative extent: ctas=%d ns=%lld", ctas, (long long)ns);
    if (ns > 2000000000ll) return fail(TILE_GEMM_E_OVERFLOW, "ns=%lld above 2 s", (long long)ns);
    int dev = 0, sms = 0;
    int rc = current_device(&dev, &sms);
    if (rc) return rc;
    if (ctas == 0) return TILE_GEMM_OK;
    constexpr int smem = 200 * 1024;   // more than half an SM: one CTA per SM
    static bool configured[64] = {};
    if (!configured[dev]) {
        CUDA_TRY(cudaFuncSetAttribute(tg::occupy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured[dev] = true;
    }
    tg::occupy_kernel<<<(unsigned)ctas, 128, smem, (cudaStream_t)stream>>>((unsigned long long)ns);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return TILE_GEMM_OK;
}

int tile_gemm_debug_trace(unsigned long long* records, int64_t capacity) {
    if (capacity < 0 || capacity > INT32_MAX) return fail(TILE_GEMM_E_EXTENT, "trace capacity %lld out of range", (long long)capacity);
    if (records && ((uintptr_t)records & 7)) return fail(TILE_GEMM_E_ALIGN, "trace buffer (%p) is not 8-byte aligned", (void*)records);
    g_trace.store(capacity > 0 ? records : nullptr);
    g_trace_cap.store(records ? capacity : 0);
    return TILE_GEMM_OK;
}

int tile_gemm_set_tuning(int key, int value) {
    if (key < 0 || key >= kNumTune) return fail(TILE_GEMM_E_PATH, "unknown tuning key %d", key);
    g_tune[key].store(value);
    return TILE_GEMM_OK;
}

int64_t tile_gemm_launch_count(void) { return g_launches.load(); }

const char* tile_gemm_status_string(int status) {
    if (status < 0 || status >= TILE_GEMM_NUM_STATUS) return "unknown status";
    return kStatusNames[status];
}

const char* tile_gemm_last_error(void) { return g_err; }

int tile_gemm_shutdown(void) {
    for (HostStage& hs : g_host) hs.mu.lock();   // index order; tile_gemm_host holds at most one of them
    std::lock_guard<std::mutex> lk(g_mu);
    for (auto& kv : g_wsets) free_workspace_set(kv.second);
    g_wsets.clear();
    // a step whose record_end never came: its private workspaces go too (the caller's capture, if it is
    // still open, is the caller's to end; record_end on that stream now reports E_PATH)
    for (auto& kv : g_recording) {
        free_workspace_set(kv.second->ws);
        delete kv.second;
    }
    g_recording.clear();
    for (void* q : g_retired) cudaFree(q);
    g_retired.clear();
    for (HostStage& hs : g_host) {
        for (Buf* b : {&hs.a, &hs.b, &hs.c}) {
            if (b->p) cudaFree(b->p);
            *b = Buf();
        }
        if (hs.in) { cudaStreamDestroy(hs.in); hs.in = nullptr; }
        if (hs.compute) { cudaStreamDestroy(hs.compute); hs.compute = nullptr; }
        if (hs.out) { cudaStreamDestroy(hs.out); hs.out = nullptr; }
        for (cudaEvent_t e : hs.events) cudaEventDestroy(e);
        hs.events.clear();
    }
    g_maps.clear();
    for (HostStage& hs : g_host) hs.mu.unlock();
    return TILE_GEMM_OK;
}

}  // extern "C"

// ====================================================================== M = 1 without any device allocation
// tile_gemv_no_alloc (include/tile_gemm.h): the split-K M = 1 kernel in its ticket protocol, with the fp32 partial
// sums and the tickets in the file-scope device array below instead of a cudaMalloc'ed workspace.  Nothing else in
// the library touches this array and no other entry point is routed through this code.
//
// Every context that loads the library holds the array (1 MiB + 4 KiB) until the process exits.  Layout:
//   [0, kNoAllocPartialBytes)                      float partials[tile][256], tile = column block * S + slice
//   [kNoAllocPartialBytes, + 4 * MAX_TILES)        uint32_t tickets[column block]
constexpr size_t kNoAllocPartialBytes = (size_t)TILE_GEMV_NO_ALLOC_MAX_TILES * tg::GEMV_COLS * sizeof(float);
constexpr size_t kNoAllocTicketBytes = (size_t)TILE_GEMV_NO_ALLOC_MAX_TILES * sizeof(uint32_t);
static_assert(kNoAllocPartialBytes + kNoAllocTicketBytes == TILE_GEMV_NO_ALLOC_SCRATCH_BYTES,
              "the header states the size of the scratch array");
static_assert(TILE_GEMV_NO_ALLOC_MAX_N == TILE_GEMV_NO_ALLOC_MAX_TILES * tg::GEMV_COLS, "one ticket per column block");

static __device__ __align__(256) unsigned char g_no_alloc_scratch[TILE_GEMV_NO_ALLOC_SCRATCH_BYTES];

namespace {
// In host code `g_no_alloc_scratch` is only the handle the runtime registered for the symbol, not an address the
// GPU can use: the device address is looked up once per device (with that device current) and kept here.
std::mutex g_no_alloc_mu;
void* g_no_alloc_ptr[64] = {};

int no_alloc_scratch(int dev, unsigned char** out) {   // `dev` is the current device
    std::lock_guard<std::mutex> lk(g_no_alloc_mu);
    if (g_no_alloc_ptr[dev] == nullptr) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_no_alloc_scratch);
        if (e != cudaSuccess || ptr == nullptr) {
            cudaGetLastError();
            return fail(TILE_GEMM_E_CUDA, "cudaGetSymbolAddress(no-alloc scratch) failed on device %d: %s (%d)", dev,
                        cudaGetErrorString(e), (int)e);
        }
        g_no_alloc_ptr[dev] = ptr;
    }
    *out = (unsigned char*)g_no_alloc_ptr[dev];
    return TILE_GEMM_OK;
}
}  // namespace

extern "C" {

int tile_gemv_no_alloc(const void* x, const void* B, void* y, int64_t N, int64_t K, int64_t ldb, int in_dtype,
                       int out_dtype, int split, void* stream) {
    // ---- launch preconditions: those of tile_gemm at M = 1, then the ones the fixed scratch adds ----
    Plan plan;
    int rc = check_and_select(x, B, y, 1, N, K, K, ldb, N, in_dtype, out_dtype, &plan);
    if (rc) return rc;
    if (split < 0) return fail(TILE_GEMM_E_EXTENT, "negative K-slice count: split=%d", split);
    if (N > TILE_GEMV_NO_ALLOC_MAX_N)
        return fail(TILE_GEMM_E_LIMIT,
                    "N=%lld is above TILE_GEMV_NO_ALLOC_MAX_N=%d, the widest output the fixed %d-byte scratch array "
                    "has tickets for; use tile_gemm (which allocates its workspace) or split the columns over calls",
                    (long long)N, TILE_GEMV_NO_ALLOC_MAX_N, TILE_GEMV_NO_ALLOC_SCRATCH_BYTES);
    const int64_t col_blocks = (N + tg::GEMV_COLS - 1) / tg::GEMV_COLS;
    const int64_t k_tiles = (K + 63) / 64;
    if (split > 1 && col_blocks * (split < k_tiles ? split : k_tiles) > TILE_GEMV_NO_ALLOC_MAX_TILES)
        return fail(TILE_GEMM_E_LIMIT,
                    "split=%d over %lld column blocks needs %lld partial-sum tiles; the fixed scratch array holds "
                    "TILE_GEMV_NO_ALLOC_MAX_TILES=%d (pass split = 0 for a count that fits)",
                    split, (long long)col_blocks, (long long)(col_blocks * (split < k_tiles ? split : k_tiles)),
                    TILE_GEMV_NO_ALLOC_MAX_TILES);
    if (plan.path == TILE_GEMM_PATH_NOOP) return TILE_GEMM_OK;
    if (K > 0 && !plan.b_tma)
        return fail(TILE_GEMM_E_PATH,
                    "tile_gemv_no_alloc reads B through TMA: B (%p) must be 16-byte aligned and ldb (%lld) a multiple "
                    "of 8 (the repack path of tile_gemm would need an allocated copy)", B, (long long)ldb);
    int dev = 0, sms = 0;
    rc = current_device(&dev, &sms);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if (K == 0) return run_zero(y, 1, N, N, plan.esize, s, sms);

    // ---- plan: the default ring shape (256 columns, 64 rows per stage, 3 stages, 2 CTAs per SM) ----
    const int64_t budget = (int64_t)sms * 2;
    const int64_t gx = col_blocks < budget ? col_blocks : budget;
    int64_t S = split;
    if (S == 0) {
        S = budget / gx;                                                    // as many slices as stay co-resident
        const int64_t fit = TILE_GEMV_NO_ALLOC_MAX_TILES / col_blocks;     // >= 1: col_blocks <= MAX_TILES
        if (S > fit) S = fit;
    }
    if (S > k_tiles) S = k_tiles;
    if (S > 65535) S = 65535;
    if (S < 1) S = 1;

    tg::GemvSplitParams p;
    memset(&p, 0, sizeof p);
    p.x = (const uint16_t*)x;
    p.y = y;
    p.N = (int32_t)N;
    p.K = (int32_t)K;
    p.k_tiles = (int32_t)k_tiles;
    p.col_blocks = (int32_t)col_blocks;
    p.out_kind = out_dtype;
    p.flags = (((uintptr_t)x) & 15) == 0 ? tg::GEMV_FLAG_X_TMA : 0;   // neither CLUSTER nor PACKED: tickets
    p.l2_post = 0;
    if (S > 1) {
        unsigned char* scratch = nullptr;
        rc = no_alloc_scratch(dev, &scratch);
        if (rc) return rc;
        p.partials = (float*)scratch;
        p.tickets = (uint32_t*)(scratch + kNoAllocPartialBytes);
        // The array keeps whatever the last call left.  Partial sums are written before they are read, the
        // tickets must start at zero: clear the ones this launch draws, in stream order ahead of the kernel.
        CUDA_TRY(cudaMemsetAsync(p.tickets, 0, (size_t)col_blocks * sizeof(uint32_t), s));
    }
    // no programmatic dependent launch: two calls in a row on one stream must not overlap on the shared scratch
    return in_dtype == TILE_GEMM_IN_F16
               ? launch_gemv_split<256, 64, 3, 2, true>(B, N, K, ldb, p, (int)gx, (int)S, false, s, dev)
               : launch_gemv_split<256, 64, 3, 2, false>(B, N, K, ldb, p, (int)gx, (int)S, false, s, dev);
}

}  // extern "C"
