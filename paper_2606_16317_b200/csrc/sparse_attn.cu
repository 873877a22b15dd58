// C-ABI of the tile-skipping attention forward (include/sparse_attn.h): argument validation,
// TMA tensor maps, launch.  No CPU fallback: without an sm_100 device every compute call fails.
#include "../../include/sparse_attn.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "fwd_kernel.cuh"
#include "reorder_kernel.cuh"
#include "rowcurve_kernel.cuh"
#include "select_kernel.cuh"
#include "stats_kernel.cuh"

// K / V ring depths of the D = 128 kernels (Q 64 KB + (NK + NV) x 32 KB must fit in 227 KB)
constexpr int DSA_NK = 3;
constexpr int DSA_NV = 2;

namespace {

thread_local char g_last_error[512] = "";
std::atomic<int64_t> g_launches{0};
std::atomic<int64_t> g_reorder_launches{0};

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_last_error, sizeof g_last_error, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                           \
    do {                                                                                         \
        cudaError_t err__ = (expr);                                                              \
        if (err__ != cudaSuccess)                                                                \
            return fail(SPARSE_ATTN_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(err__)); \
    } while (0)

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode_fn(EncodeTiledFn* out) {
    static std::once_flag once;
    static EncodeTiledFn cached = nullptr;
    static cudaError_t first_err = cudaSuccess;
    std::call_once(once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        first_err = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (first_err == cudaSuccess && qres == cudaDriverEntryPointSuccess) cached = reinterpret_cast<EncodeTiledFn>(fn);
    });
    if (!cached)
        return fail(SPARSE_ATTN_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available (%s)", cudaGetErrorString(first_err));
    *out = cached;
    return 0;
}

// bf16 [BH, N, D] tensor, box = 64 columns (128 B, SWIZZLE_128B) x `rows` tokens of one head.
// Out-of-range tokens (ragged last tile) are zero-filled by TMA and never bleed into the next head.
int make_tmap(EncodeTiledFn enc, CUtensorMap* tm, const void* base, int BH, int N, int D, int rows) {
    cuuint64_t dims[3] = {static_cast<cuuint64_t>(D), static_cast<cuuint64_t>(N), static_cast<cuuint64_t>(BH)};
    cuuint64_t strides[2] = {static_cast<cuuint64_t>(D) * 2, static_cast<cuuint64_t>(N) * D * 2};
    cuuint32_t box[3] = {64, static_cast<cuuint32_t>(rows), 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(SPARSE_ATTN_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return 0;
}

template <int D, int BC, int G, int NK, int NV, bool kSparse, bool kDebug, int SUB = 1>
int launch(const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv, const dsa::FwdArgs& args, int BH,
           cudaStream_t stream) {
    using L = dsa::SmemLayout<D, BC, NK, NV>;
    auto kernel = dsa::sparse_attn_fwd_kernel<D, BC, G, NK, NV, kSparse, kDebug, SUB>;
    // per device and cheap: set on every launch, so that any device / thread of the process may call the library
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, L::kDynamicBytes));
    dim3 grid((args.n_mma_tiles + 1) / 2, BH, 1);
    kernel<<<grid, dsa::kNumThreads, L::kDynamicBytes, stream>>>(tq, tk, tv, args);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return 0;
}

struct Resolved {
    int tile_q, tile_k;
    float scale, lambda;
    cudaStream_t stream;
    uint8_t* skip_mask;
    float* margin;
    const uint8_t* mask_in;
    uint64_t* cycles;
};

// Host-side validation shared by the device and host-buffer entry points.
int validate(const void* q, const void* k, const void* v, void* out, int B, int H, int N, int D,
             const sparse_attn_params* p, int mode, Resolved* r) {
    g_last_error[0] = '\0';
    if (!q || !k || !v || !out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "q, k, v and out must not be NULL");
    if (mode < SPARSE_ATTN_DENSE || mode > SPARSE_ATTN_MASK) return fail(SPARSE_ATTN_ERR_MODE, "mode %d not in {0,1,2,3}", mode);
    if (B <= 0 || H <= 0 || N <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N must be positive (got %d, %d, %d)", B, H, N);
    if (static_cast<long long>(B) * H > 65535) return fail(SPARSE_ATTN_ERR_SHAPE, "B*H = %lld exceeds 65535", (long long)B * H);
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %d exceeds 2^24", N);
    if (D != 64 && D != 128) return fail(SPARSE_ATTN_ERR_HEAD_DIM, "D = %d not in {64, 128}", D);
    if (!p && mode != SPARSE_ATTN_DENSE) return fail(SPARSE_ATTN_ERR_PARAMS, "params must not be NULL in a sparse mode");
    const int def_tile = (D == 64) ? 64 : 128;
    r->tile_q = r->tile_k = def_tile;
    r->scale = 1.0f / std::sqrt(static_cast<float>(D));
    r->lambda = -INFINITY;
    r->stream = nullptr;
    r->skip_mask = nullptr;
    r->margin = nullptr;
    r->mask_in = nullptr;
    r->cycles = nullptr;
    if (p) {
        if (p->struct_size != sizeof(sparse_attn_params))
            return fail(SPARSE_ATTN_ERR_PARAMS, "params->struct_size = %u, expected %zu", p->struct_size, sizeof(sparse_attn_params));
        if (std::isnan(p->lambda)) return fail(SPARSE_ATTN_ERR_PARAMS, "lambda is NaN");
        if (mode == SPARSE_ATTN_FIXED && p->lambda > 0.f)
            return fail(SPARSE_ATTN_ERR_PARAMS, "lambda = %g > 0 is unsupported in FIXED mode (DESIGN.md R6)", p->lambda);
        if (!(p->softmax_scale >= 0.f) || std::isinf(p->softmax_scale))
            return fail(SPARSE_ATTN_ERR_PARAMS, "softmax_scale must be finite and >= 0 (0 = 1/sqrt(D))");
        const int tq = p->tile_q ? p->tile_q : def_tile;
        const int tk = p->tile_k ? p->tile_k : tq;
        // D = 128 also takes decision tiles of 128 x 64 and 128 x 32 keys (block size 32 for the 5B model)
        const bool sub_ok = D == 128 && tq == 128 && (tk == 64 || tk == 32) && mode != SPARSE_ATTN_DENSE;
        if ((tq != def_tile || tk != def_tile) && !sub_ok)
            return fail(SPARSE_ATTN_ERR_TILE, "decision tile %dx%d unsupported for D = %d in mode %d (supported: %dx%d%s)", tq, tk, D,
                        mode, def_tile, def_tile, D == 128 ? ", and 128x64 / 128x32 in the sparse modes" : "");
        if (sub_ok && tk != def_tile && p->lambda > 0.f)
            return fail(SPARSE_ATTN_ERR_PARAMS, "lambda = %g > 0 is unsupported with %dx%d decision tiles (the stabiliser follows the "
                        "max of the whole 128-key MMA tile, which a positive threshold may skip)", p->lambda, tq, tk);
        r->tile_k = tk;
        if (p->softmax_scale > 0.f) r->scale = p->softmax_scale;
        r->lambda = p->lambda;
        r->stream = static_cast<cudaStream_t>(p->stream);
        r->skip_mask = p->skip_mask_out;
        r->margin = p->margin_out;
        if (mode == SPARSE_ATTN_MASK) {
            if (!p->skip_mask_in) return fail(SPARSE_ATTN_ERR_PARAMS, "MASK mode needs params->skip_mask_in");
            if (tq != def_tile || tk != def_tile)
                return fail(SPARSE_ATTN_ERR_TILE, "MASK mode takes the default %dx%d decision tiles only", def_tile, def_tile);
        } else if (p->skip_mask_in) {
            return fail(SPARSE_ATTN_ERR_PARAMS, "skip_mask_in is set but mode %d is not MASK", mode);
        }
        r->mask_in = p->skip_mask_in;
        r->cycles = p->cycles_out;
    }
    return 0;
}

int check_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(SPARSE_ATTN_ERR_DEVICE, "no CUDA device available (this library has no CPU fallback)");
    }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
        cudaGetLastError();
        return fail(SPARSE_ATTN_ERR_DEVICE, "device %d has compute capability major %d; sm_100 (B200) is required", dev, major);
    }
    return 0;
}

int sm_count(int* n_sm) {                                    // per call: the current device may differ between calls
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(n_sm, cudaDevAttrMultiProcessorCount, dev));
    return 0;
}

// ---- device scratch of sparse_attn_fwd_host: a pool of the library's own, one per device, so that neither the release
// threshold nor the retained memory touches the device's default pool (which the host application may be using).
constexpr int kMaxPoolDevices = 64;
std::mutex g_host_mu;
cudaMemPool_t g_scratch_pool[kMaxPoolDevices] = {};

int scratch_pool(int dev, cudaMemPool_t* pool) {
    if (dev < 0 || dev >= kMaxPoolDevices) return fail(SPARSE_ATTN_ERR_DEVICE, "device ordinal %d outside [0, %d)", dev, kMaxPoolDevices);
    std::lock_guard<std::mutex> lock(g_host_mu);
    if (!g_scratch_pool[dev]) {
        cudaMemPoolProps props;
        std::memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t created = nullptr;
        CUDA_TRY(cudaMemPoolCreate(&created, &props));
        uint64_t keep = UINT64_MAX;                          // freed scratch stays in THIS pool until sparse_attn_release_scratch
        cudaError_t err = cudaMemPoolSetAttribute(created, cudaMemPoolAttrReleaseThreshold, &keep);
        if (err != cudaSuccess) {
            cudaMemPoolDestroy(created);
            return fail(SPARSE_ATTN_ERR_CUDA, "cudaMemPoolSetAttribute failed: %s", cudaGetErrorString(err));
        }
        g_scratch_pool[dev] = created;
    }
    *pool = g_scratch_pool[dev];
    return 0;
}

// ---- the internal streams and events of one sparse_attn_fwd_host call; sets are recycled across calls (a call takes a
// free set of its device or creates one, and hands it back), so that a steady caller creates them once.
constexpr int kMaxChunks = 20;      // (config 3: 2 heads = 4 whole waves per chunk; 8 chunks left 3 ms of copy head and tail exposed)
struct HostSet {
    int dev = -1;
    cudaStream_t s_in = nullptr, s_out = nullptr, s_k[2] = {nullptr, nullptr};
    cudaEvent_t ev_start = nullptr, ev_in[kMaxChunks] = {}, ev_done[kMaxChunks] = {}, ev_end[4] = {};
};
std::vector<HostSet*> g_host_sets;                           // free sets, any device (guarded by g_host_mu)

void destroy_host_set(HostSet* h) {
    for (cudaStream_t s : {h->s_in, h->s_out, h->s_k[0], h->s_k[1]}) if (s) cudaStreamDestroy(s);
    if (h->ev_start) cudaEventDestroy(h->ev_start);
    for (int c = 0; c < kMaxChunks; ++c) { if (h->ev_in[c]) cudaEventDestroy(h->ev_in[c]); if (h->ev_done[c]) cudaEventDestroy(h->ev_done[c]); }
    for (cudaEvent_t e : h->ev_end) if (e) cudaEventDestroy(e);
    delete h;
}

int acquire_host_set(int dev, HostSet** out) {
    {
        std::lock_guard<std::mutex> lock(g_host_mu);
        for (size_t i = 0; i < g_host_sets.size(); ++i)
            if (g_host_sets[i]->dev == dev) {
                *out = g_host_sets[i];
                g_host_sets.erase(g_host_sets.begin() + i);
                return 0;
            }
    }
    HostSet* h = new HostSet;
    h->dev = dev;
    cudaError_t err = cudaSuccess;
    auto ok = [&](cudaError_t e) { if (err == cudaSuccess) err = e; return err == cudaSuccess; };
    for (cudaStream_t* s : {&h->s_in, &h->s_out, &h->s_k[0], &h->s_k[1]}) ok(cudaStreamCreateWithFlags(s, cudaStreamNonBlocking));
    ok(cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming));
    for (int c = 0; c < kMaxChunks; ++c) {
        ok(cudaEventCreateWithFlags(&h->ev_in[c], cudaEventDisableTiming));
        ok(cudaEventCreateWithFlags(&h->ev_done[c], cudaEventDisableTiming));
    }
    for (cudaEvent_t& e : h->ev_end) ok(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    if (err != cudaSuccess) {
        destroy_host_set(h);
        return fail(SPARSE_ATTN_ERR_CUDA, "creating the internal streams / events failed: %s", cudaGetErrorString(err));
    }
    *out = h;
    return 0;
}

void release_host_set(HostSet* h) {
    std::lock_guard<std::mutex> lock(g_host_mu);
    g_host_sets.push_back(h);
}

}  // namespace

extern "C" {

int sparse_attn_fwd(const void* q, const void* k, const void* v, void* out, float* lse, int B, int H, int N, int D,
                    const sparse_attn_params* params, int mode, int64_t* stats_out) {
    Resolved r;
    int rc = validate(q, k, v, out, B, H, N, D, params, mode, &r);
    if (rc) return rc;
    const uintptr_t align_or = reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k) |
                               reinterpret_cast<uintptr_t>(v) | reinterpret_cast<uintptr_t>(out);
    if (align_or & 15u) return fail(SPARSE_ATTN_ERR_ALIGNMENT, "q, k, v and out must be 16-byte aligned");
    if ((rc = check_device())) return rc;

    EncodeTiledFn enc = nullptr;
    if ((rc = get_encode_fn(&enc))) return rc;
    const int BH = B * H;
    CUtensorMap tq, tk, tv;
    if ((rc = make_tmap(enc, &tq, q, BH, N, D, 128))) return rc;
    const int mma_k = (D == 64) ? 64 : 128;                 // keys per MMA tile (the decision tile may be narrower)
    if ((rc = make_tmap(enc, &tk, k, BH, N, D, mma_k))) return rc;
    if ((rc = make_tmap(enc, &tv, v, BH, N, D, mma_k))) return rc;

    dsa::FwdArgs a;
    std::memset(&a, 0, sizeof a);
    a.out = static_cast<__nv_bfloat16*>(out);
    a.lse = lse;
    a.stats = reinterpret_cast<unsigned long long*>(stats_out);
    a.skip_mask = r.skip_mask;
    a.margin = r.margin;
    a.mask_in = r.mask_in;
    a.cycles = reinterpret_cast<unsigned long long*>(r.cycles);
    a.N = N;
    a.T_r = (N + r.tile_q - 1) / r.tile_q;
    a.T_c = (N + mma_k - 1) / mma_k;
    a.T_c_dec = (N + r.tile_k - 1) / r.tile_k;
    a.n_mma_tiles = (N + 127) / 128;
    a.mode = mode;
    a.scale_log2 = r.scale * dsa::kLog2e;
    a.lambda_log2 = r.lambda * dsa::kLog2e;

    if (stats_out) CUDA_TRY(cudaMemsetAsync(stats_out, 0, sizeof(int64_t) * 2 * BH, r.stream));
    if (r.cycles) CUDA_TRY(cudaMemsetAsync(r.cycles, 0, sizeof(uint64_t) * 2, r.stream));
    const bool sparse = mode != SPARSE_ATTN_DENSE;
    const bool debug = r.skip_mask || r.margin || r.cycles;
    if (D == 128) {
        if (!sparse && !debug) return launch<128, 128, 1, DSA_NK, DSA_NV, false, false>(tq, tk, tv, a, BH, r.stream);
        if (!sparse) return launch<128, 128, 1, DSA_NK, DSA_NV, false, true>(tq, tk, tv, a, BH, r.stream);
        if (r.tile_k == 64) {
            if (!debug) return launch<128, 128, 1, DSA_NK, DSA_NV, true, false, 2>(tq, tk, tv, a, BH, r.stream);
            return launch<128, 128, 1, DSA_NK, DSA_NV, true, true, 2>(tq, tk, tv, a, BH, r.stream);
        }
        if (r.tile_k == 32) {
            if (!debug) return launch<128, 128, 1, DSA_NK, DSA_NV, true, false, 4>(tq, tk, tv, a, BH, r.stream);
            return launch<128, 128, 1, DSA_NK, DSA_NV, true, true, 4>(tq, tk, tv, a, BH, r.stream);
        }
        if (!debug) return launch<128, 128, 1, DSA_NK, DSA_NV, true, false>(tq, tk, tv, a, BH, r.stream);
        return launch<128, 128, 1, DSA_NK, DSA_NV, true, true>(tq, tk, tv, a, BH, r.stream);
    }
    if (!sparse && !debug) return launch<64, 64, 2, 3, 2, false, false>(tq, tk, tv, a, BH, r.stream);
    if (!sparse) return launch<64, 64, 2, 3, 2, false, true>(tq, tk, tv, a, BH, r.stream);
    if (!debug) return launch<64, 64, 2, 3, 2, true, false>(tq, tk, tv, a, BH, r.stream);
    return launch<64, 64, 2, 3, 2, true, true>(tq, tk, tv, a, BH, r.stream);
}

// Host-buffer entry: the B*H heads are independent units, so they are cut into chunks and pipelined over four internal
// streams -- H2D of chunk c+1 (s_in) and D2H of chunk c-1 (s_out) run under the kernel of chunk c (PCIe is full duplex),
// and the kernels of consecutive chunks alternate between two streams (s_k[0..1]) so that the next chunk's CTAs fill the
// last wave of the previous one.  Device scratch comes from the library's own stream-ordered pool (one allocation per
// tensor and call; freed memory stays in that pool until sparse_attn_release_scratch); the streams and events are
// recycled across calls.
int sparse_attn_fwd_host(const void* q, const void* k, const void* v, void* out, float* lse, int B, int H, int N, int D,
                         const sparse_attn_params* params, int mode, int64_t* stats_out) {
    Resolved r;
    int rc = validate(q, k, v, out, B, H, N, D, params, mode, &r);
    if (rc) return rc;
    if ((rc = check_device())) return rc;
    if (r.cycles) return fail(SPARSE_ATTN_ERR_PARAMS, "params->cycles_out is not supported by the host-buffer entry");
    const size_t BH = static_cast<size_t>(B) * H;
    const size_t head_elems = static_cast<size_t>(N) * D;
    const size_t T_r = (N + r.tile_q - 1) / r.tile_q, T_c = (N + r.tile_k - 1) / r.tile_k;
    const size_t head_tiles = T_r * T_c;
    const int n_chunks = static_cast<int>(std::min<size_t>(BH, kMaxChunks));
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaMemPool_t pool = nullptr;
    if ((rc = scratch_pool(dev, &pool))) return rc;
    HostSet* hs = nullptr;
    if ((rc = acquire_host_set(dev, &hs))) return rc;
    cudaStream_t st = r.stream;
    void *dq = nullptr, *dk = nullptr, *dv = nullptr, *dout = nullptr;
    float *dlse = nullptr, *dmargin = nullptr;
    int64_t* dstats = nullptr;
    uint8_t *dmask = nullptr, *dmask_in = nullptr;
    auto cleanup = [&]() {
        void* bufs[] = {dq, dk, dv, dout, dlse, dstats, dmask, dmargin, dmask_in};
        for (void* b : bufs) if (b) cudaFreeAsync(b, st);
        cudaStreamSynchronize(st);
        release_host_set(hs);
    };
#define HOST_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t err__ = (expr);                                                                      \
        if (err__ != cudaSuccess) {                                                                      \
            cudaDeviceSynchronize();                                                                     \
            cleanup();                                                                                   \
            return fail(SPARSE_ATTN_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(err__));        \
        }                                                                                                \
    } while (0)
    HOST_TRY(cudaMallocFromPoolAsync(&dq, BH * head_elems * 2, pool, st));
    HOST_TRY(cudaMallocFromPoolAsync(&dk, BH * head_elems * 2, pool, st));
    HOST_TRY(cudaMallocFromPoolAsync(&dv, BH * head_elems * 2, pool, st));
    HOST_TRY(cudaMallocFromPoolAsync(&dout, BH * head_elems * 2, pool, st));
    if (lse) HOST_TRY(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&dlse), BH * N * sizeof(float), pool, st));
    if (stats_out) HOST_TRY(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&dstats), BH * 2 * sizeof(int64_t), pool, st));
    if (r.skip_mask) HOST_TRY(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&dmask), BH * head_tiles, pool, st));
    if (r.margin) HOST_TRY(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&dmargin), BH * head_tiles * sizeof(float), pool, st));
    if (r.mask_in) HOST_TRY(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&dmask_in), BH * head_tiles, pool, st));
    cudaStream_t s_in = hs->s_in, s_out = hs->s_out, s_k[2] = {hs->s_k[0], hs->s_k[1]};
    // the scratch allocations (and whatever the caller enqueued before) are ordered on `st`
    HOST_TRY(cudaEventRecord(hs->ev_start, st));
    for (cudaStream_t s : {s_in, s_out, s_k[0], s_k[1]}) HOST_TRY(cudaStreamWaitEvent(s, hs->ev_start, 0));

    sparse_attn_params dp;
    std::memset(&dp, 0, sizeof dp);
    if (params) dp = *params;
    dp.struct_size = sizeof dp;
    if (!params) dp.lambda = -INFINITY;
    auto at = [](const void* p, size_t bytes) { return static_cast<const char*>(p) + bytes; };
    auto atw = [](void* p, size_t bytes) { return static_cast<char*>(p) + bytes; };
    for (int c = 0; c < n_chunks; ++c) {
        const size_t h0 = BH * c / n_chunks, h1 = BH * (c + 1) / n_chunks, nh = h1 - h0;
        const size_t eoff = h0 * head_elems * 2, ebytes = nh * head_elems * 2;
        if (r.mask_in)
            HOST_TRY(cudaMemcpyAsync(dmask_in + h0 * head_tiles, r.mask_in + h0 * head_tiles, nh * head_tiles, cudaMemcpyHostToDevice, s_in));
        HOST_TRY(cudaMemcpyAsync(atw(dq, eoff), at(q, eoff), ebytes, cudaMemcpyHostToDevice, s_in));
        HOST_TRY(cudaMemcpyAsync(atw(dk, eoff), at(k, eoff), ebytes, cudaMemcpyHostToDevice, s_in));
        HOST_TRY(cudaMemcpyAsync(atw(dv, eoff), at(v, eoff), ebytes, cudaMemcpyHostToDevice, s_in));
        HOST_TRY(cudaEventRecord(hs->ev_in[c], s_in));
        cudaStream_t sk = s_k[c & 1];
        HOST_TRY(cudaStreamWaitEvent(sk, hs->ev_in[c], 0));
        dp.stream = sk;
        dp.skip_mask_out = dmask ? dmask + h0 * head_tiles : nullptr;
        dp.margin_out = dmargin ? dmargin + h0 * head_tiles : nullptr;
        dp.skip_mask_in = dmask_in ? dmask_in + h0 * head_tiles : nullptr;
        rc = sparse_attn_fwd(atw(dq, eoff), atw(dk, eoff), atw(dv, eoff), atw(dout, eoff), dlse ? dlse + h0 * N : nullptr, 1,
                             static_cast<int>(nh), N, D, &dp, mode, dstats ? dstats + h0 * 2 : nullptr);
        if (rc) { cudaDeviceSynchronize(); cleanup(); return rc; }
        HOST_TRY(cudaEventRecord(hs->ev_done[c], sk));
        HOST_TRY(cudaStreamWaitEvent(s_out, hs->ev_done[c], 0));
        HOST_TRY(cudaMemcpyAsync(atw(out, eoff), at(dout, eoff), ebytes, cudaMemcpyDeviceToHost, s_out));
        if (lse) HOST_TRY(cudaMemcpyAsync(lse + h0 * N, dlse + h0 * N, nh * N * sizeof(float), cudaMemcpyDeviceToHost, s_out));
        if (stats_out) HOST_TRY(cudaMemcpyAsync(stats_out + h0 * 2, dstats + h0 * 2, nh * 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, s_out));
        if (r.skip_mask) HOST_TRY(cudaMemcpyAsync(r.skip_mask + h0 * head_tiles, dmask + h0 * head_tiles, nh * head_tiles, cudaMemcpyDeviceToHost, s_out));
        if (r.margin)
            HOST_TRY(cudaMemcpyAsync(r.margin + h0 * head_tiles, dmargin + h0 * head_tiles, nh * head_tiles * sizeof(float), cudaMemcpyDeviceToHost, s_out));
    }
    // join everything back into `st`, then wait: the call is synchronous
    cudaStream_t joins[4] = {s_in, s_out, s_k[0], s_k[1]};
    for (int i = 0; i < 4; ++i) {
        HOST_TRY(cudaEventRecord(hs->ev_end[i], joins[i]));
        HOST_TRY(cudaStreamWaitEvent(st, hs->ev_end[i], 0));
    }
    HOST_TRY(cudaStreamSynchronize(st));
    cleanup();
#undef HOST_TRY
    return 0;
}

// Hands the memory sparse_attn_fwd_host keeps in the library's scratch pool of the current device back to the driver,
// and drops the recycled stream / event sets of that device.
int sparse_attn_release_scratch(void) {
    g_last_error[0] = '\0';
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    std::vector<HostSet*> mine;
    cudaMemPool_t pool = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_host_mu);
        for (size_t i = 0; i < g_host_sets.size();)
            if (g_host_sets[i]->dev == dev) { mine.push_back(g_host_sets[i]); g_host_sets.erase(g_host_sets.begin() + i); }
            else ++i;
        if (dev >= 0 && dev < kMaxPoolDevices) pool = g_scratch_pool[dev];
    }
    for (HostSet* h : mine) destroy_host_set(h);
    if (pool) CUDA_TRY(cudaMemPoolTrimTo(pool, 0));
    return 0;
}

int sparse_attn_block_stats(const void* q, const void* k, const float* lse, float* mass_out, float* sqmass_out, int B, int H,
                            int N, int D, float softmax_scale, void* stream) {
    g_last_error[0] = '\0';
    if (!q || !k || !lse || !mass_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "q, k, lse and mass_out must not be NULL");
    if (B <= 0 || H <= 0 || N <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N must be positive (got %d, %d, %d)", B, H, N);
    if (static_cast<long long>(B) * H > 65535) return fail(SPARSE_ATTN_ERR_SHAPE, "B*H = %lld exceeds 65535", (long long)B * H);
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %d exceeds 2^24", N);
    if (D != 64 && D != 128) return fail(SPARSE_ATTN_ERR_HEAD_DIM, "D = %d not in {64, 128}", D);
    if (!(softmax_scale >= 0.f) || std::isinf(softmax_scale))
        return fail(SPARSE_ATTN_ERR_PARAMS, "softmax_scale must be finite and >= 0 (0 = 1/sqrt(D))");
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k)) & 15u)
        return fail(SPARSE_ATTN_ERR_ALIGNMENT, "q and k must be 16-byte aligned");
    int rc = check_device();
    if (rc) return rc;
    EncodeTiledFn enc = nullptr;
    if ((rc = get_encode_fn(&enc))) return rc;
    const int BH = B * H;
    const int tile = (D == 64) ? 64 : 128;
    CUtensorMap tq, tk;
    if ((rc = make_tmap(enc, &tq, q, BH, N, D, 128))) return rc;
    if ((rc = make_tmap(enc, &tk, k, BH, N, D, tile))) return rc;
    dsa::FwdArgs a;
    std::memset(&a, 0, sizeof a);
    a.N = N;
    a.T_r = (N + tile - 1) / tile;
    a.T_c = a.T_c_dec = (N + tile - 1) / tile;
    a.n_mma_tiles = (N + 127) / 128;
    a.mode = dsa::kModeMass;
    a.scale_log2 = (softmax_scale > 0.f ? softmax_scale : 1.0f / std::sqrt(static_cast<float>(D))) * dsa::kLog2e;
    a.lambda_log2 = -INFINITY;
    a.lse_in = lse;
    a.mass_out = mass_out;
    a.sqmass_out = sqmass_out;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CUDA_TRY(cudaMemsetAsync(mass_out, 0, sizeof(float) * static_cast<size_t>(BH) * a.T_r * a.T_c, st));
    if (sqmass_out) CUDA_TRY(cudaMemsetAsync(sqmass_out, 0, sizeof(float) * static_cast<size_t>(BH) * a.T_r * a.T_c, st));
    // V is never read in this mode (every tile is voted skipped and the V warp fetches nothing); the V map aliases K only
    // because the kernel's signature wants one
    if (D == 128) return launch<128, 128, 1, DSA_NK, DSA_NV, true, false, 0>(tq, tk, tk, a, BH, st);
    return launch<64, 64, 2, 3, 2, true, false, 0>(tq, tk, tk, a, BH, st);
}

int sparse_attn_block_mass(const void* q, const void* k, const float* lse, float* mass_out, int B, int H, int N, int D,
                           float softmax_scale, void* stream) {
    return sparse_attn_block_stats(q, k, lse, mass_out, nullptr, B, H, N, D, softmax_scale, stream);
}

int sparse_attn_select_blocks_greedy(const float* mass, const float* sqmass, uint8_t* skip_mask_out, int B, int H, int N,
                                     int tile_q, int T_c, double theta, void* stream) {
    g_last_error[0] = '\0';
    if (!mass || !sqmass || !skip_mask_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "mass, sqmass and skip_mask_out must not be NULL");
    if (B <= 0 || H <= 0 || N <= 0 || T_c <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N, T_c must be positive");
    if (tile_q != 64 && tile_q != 128) return fail(SPARSE_ATTN_ERR_TILE, "tile_q = %d not in {64, 128}", tile_q);
    if (static_cast<long long>(B) * H > 65535) return fail(SPARSE_ATTN_ERR_SHAPE, "B*H = %lld exceeds 65535", (long long)B * H);
    if (T_c > dsa::kSelectMaxTc) return fail(SPARSE_ATTN_ERR_SHAPE, "T_c = %d exceeds %d", T_c, dsa::kSelectMaxTc);
    if (!(theta >= 0.0)) return fail(SPARSE_ATTN_ERR_PARAMS, "theta = %g must be >= 0", theta);
    int rc = check_device();
    if (rc) return rc;
    const int T_r = (N + tile_q - 1) / tile_q;
    dim3 grid(T_r, B * H, 1);
    dsa::select_blocks_greedy_kernel<<<grid, 256, sizeof(float) * 3 * T_c, static_cast<cudaStream_t>(stream)>>>(
        mass, sqmass, skip_mask_out, T_c, N, tile_q, theta);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(1);
    return 0;
}

int sparse_attn_select_blocks(const float* mass, uint8_t* skip_mask_out, int B, int H, int T_r, int T_c, int kind,
                              double param, void* stream) {
    g_last_error[0] = '\0';
    if (!mass || !skip_mask_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "mass and skip_mask_out must not be NULL");
    if (B <= 0 || H <= 0 || T_r <= 0 || T_c <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, T_r, T_c must be positive");
    if (static_cast<long long>(B) * H > 65535) return fail(SPARSE_ATTN_ERR_SHAPE, "B*H = %lld exceeds 65535", (long long)B * H);
    if (T_c > dsa::kSelectMaxTc) return fail(SPARSE_ATTN_ERR_SHAPE, "T_c = %d exceeds %d", T_c, dsa::kSelectMaxTc);
    if (kind != SPARSE_ATTN_SELECT_TOPK && kind != SPARSE_ATTN_SELECT_TOPP)
        return fail(SPARSE_ATTN_ERR_MODE, "kind %d not in {0 (Top-K), 1 (Top-P)}", kind);
    if (!(param > 0.0) || param > 1.0) return fail(SPARSE_ATTN_ERR_PARAMS, "param = %g not in (0, 1]", param);
    int rc = check_device();
    if (rc) return rc;
    int n_keep = static_cast<int>(std::ceil(param * T_c));
    n_keep = std::max(1, std::min(T_c, n_keep));
    dim3 grid(T_r, B * H, 1);
    dsa::select_blocks_kernel<<<grid, 256, sizeof(float) * T_c, static_cast<cudaStream_t>(stream)>>>(
        mass, skip_mask_out, T_c, kind, n_keep, param);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(1);
    return 0;
}

int sparse_attn_brick_permutation(int grid_t, int grid_h, int grid_w, int brick_t, int brick_h, int brick_w,
                                  int32_t* perm_out) {
    g_last_error[0] = '\0';
    if (!perm_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "perm_out must not be NULL");
    if (grid_t <= 0 || grid_h <= 0 || grid_w <= 0 || brick_t <= 0 || brick_h <= 0 || brick_w <= 0)
        return fail(SPARSE_ATTN_ERR_SHAPE, "grid and brick dimensions must be positive");
    const long long N = static_cast<long long>(grid_t) * grid_h * grid_w;
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %lld exceeds 2^24", N);
    int32_t* p = perm_out;
    for (int t0 = 0; t0 < grid_t; t0 += brick_t)
        for (int h0 = 0; h0 < grid_h; h0 += brick_h)
            for (int w0 = 0; w0 < grid_w; w0 += brick_w)
                for (int t = t0; t < t0 + brick_t && t < grid_t; ++t)
                    for (int h = h0; h < h0 + brick_h && h < grid_h; ++h)
                        for (int w = w0; w < w0 + brick_w && w < grid_w; ++w)
                            *p++ = (t * grid_h + h) * grid_w + w;
    return 0;
}

int sparse_attn_reorder_tokens(const void* src, void* dst, int B, int H, int N, int D, const int32_t* perm,
                               int inverse, void* stream) {
    g_last_error[0] = '\0';
    if (!src || !dst || !perm) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "src, dst and perm must not be NULL");
    if (B <= 0 || H <= 0 || N <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N must be positive (got %d, %d, %d)", B, H, N);
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %d exceeds 2^24", N);
    if (D != 64 && D != 128) return fail(SPARSE_ATTN_ERR_HEAD_DIM, "D = %d not in {64, 128}", D);
    const size_t bytes = static_cast<size_t>(B) * H * N * D * 2;
    const uintptr_t s0 = reinterpret_cast<uintptr_t>(src), d0 = reinterpret_cast<uintptr_t>(dst);
    if ((s0 | d0) & 15u) return fail(SPARSE_ATTN_ERR_ALIGNMENT, "src and dst must be 16-byte aligned");
    if (s0 < d0 + bytes && d0 < s0 + bytes) return fail(SPARSE_ATTN_ERR_PARAMS, "src and dst overlap");
    int rc = check_device();
    if (rc) return rc;
    int n_sm = 0;
    if ((rc = sm_count(&n_sm))) return rc;
    const long long rows = static_cast<long long>(B) * H * N;
    const int lanes = D / 8;                                 // 16 bytes per thread
    const long long blocks_needed = (rows + (256 / lanes) * 4 - 1) / ((256 / lanes) * 4);
    const int grid = static_cast<int>(std::min<long long>(blocks_needed, static_cast<long long>(n_sm) * 8));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (lanes == 16)
        dsa::reorder_tokens_kernel<16><<<grid, 256, 0, st>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst), perm, rows, N, inverse ? 1 : 0);
    else
        dsa::reorder_tokens_kernel<8><<<grid, 256, 0, st>>>(static_cast<const uint4*>(src), static_cast<uint4*>(dst), perm, rows, N, inverse ? 1 : 0);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(1);
    return 0;
}

int sparse_attn_recall_stats(const float* lse_retained, const float* lse_dense, int64_t n_rows, double* stats_out, void* stream) {
    g_last_error[0] = '\0';
    if (!lse_retained || !lse_dense || !stats_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "lse_retained, lse_dense and stats_out must not be NULL");
    if (n_rows <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "n_rows must be positive");
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int n_sm = 0;
    if ((rc = sm_count(&n_sm))) return rc;
    const int grid = static_cast<int>(std::min<int64_t>((n_rows + 255) / 256, static_cast<int64_t>(n_sm) * 8));   // 8 CTAs of 256 threads per SM
    dsa::stats_init_kernel<<<1, 1, 0, st>>>(stats_out, INFINITY, 0.0);
    dsa::recall_stats_kernel<<<grid, 256, 0, st>>>(lse_retained, lse_dense, n_rows, stats_out);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(2);
    return 0;
}

int sparse_attn_output_error(const void* out_a, const void* out_b, int64_t n_elems, double* stats_out, void* stream) {
    g_last_error[0] = '\0';
    if (!out_a || !out_b || !stats_out) return fail(SPARSE_ATTN_ERR_NULL_POINTER, "out_a, out_b and stats_out must not be NULL");
    if (n_elems <= 0 || (n_elems & 1)) return fail(SPARSE_ATTN_ERR_SHAPE, "n_elems must be positive and even");
    if ((reinterpret_cast<uintptr_t>(out_a) | reinterpret_cast<uintptr_t>(out_b)) & 3u)
        return fail(SPARSE_ATTN_ERR_ALIGNMENT, "out_a and out_b must be 4-byte aligned");
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int64_t n2 = n_elems / 2;
    int n_sm = 0;
    if ((rc = sm_count(&n_sm))) return rc;
    const int grid = static_cast<int>(std::min<int64_t>((n2 + 255) / 256, static_cast<int64_t>(n_sm) * 8));
    dsa::stats_init_kernel<<<1, 1, 0, st>>>(stats_out, 0.0, 0.0);
    dsa::output_error_kernel<<<grid, 256, 0, st>>>(static_cast<const __nv_bfloat162*>(out_a), static_cast<const __nv_bfloat162*>(out_b), n2, stats_out);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(2);
    return 0;
}

int sparse_attn_row_topk_curve(const void* q, const void* k, const void* v, int B, int H, int N, int D, float softmax_scale,
                               const int32_t* rows, int n_rows, const int32_t* keep_counts, int n_keep,
                               double* kurtosis_out, double* recall_out, double* mae_out, void* stream) {
    g_last_error[0] = '\0';
    if (!q || !k || !v || !rows || !keep_counts || !kurtosis_out || !recall_out || !mae_out)
        return fail(SPARSE_ATTN_ERR_NULL_POINTER, "q, k, v, rows, keep_counts and the three outputs must not be NULL");
    if (B <= 0 || H <= 0 || N <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N must be positive (got %d, %d, %d)", B, H, N);
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %d exceeds 2^24", N);
    if (D != 64 && D != 128) return fail(SPARSE_ATTN_ERR_HEAD_DIM, "D = %d not in {64, 128}", D);
    if (n_rows <= 0 || n_rows > (1 << 20) || n_keep <= 0 || n_keep > 4096)
        return fail(SPARSE_ATTN_ERR_SHAPE, "n_rows must be in [1, 2^20] and n_keep in [1, 4096] (got %d, %d)", n_rows, n_keep);
    if (!(softmax_scale >= 0.f) || std::isinf(softmax_scale))
        return fail(SPARSE_ATTN_ERR_PARAMS, "softmax_scale must be finite and >= 0 (0 = 1/sqrt(D))");
    for (int i = 0; i < n_rows; ++i)
        if (rows[2 * i] < 0 || rows[2 * i] >= B * H || rows[2 * i + 1] < 0 || rows[2 * i + 1] >= N)
            return fail(SPARSE_ATTN_ERR_PARAMS, "rows[%d] = (%d, %d) outside [0, B*H) x [0, N)", i, rows[2 * i], rows[2 * i + 1]);
    for (int i = 0; i < n_keep; ++i)
        if (keep_counts[i] < 1 || keep_counts[i] > N)
            return fail(SPARSE_ATTN_ERR_PARAMS, "keep_counts[%d] = %d outside [1, N]", i, keep_counts[i]);
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k) | reinterpret_cast<uintptr_t>(v)) & 15u)
        return fail(SPARSE_ATTN_ERR_ALIGNMENT, "q, k and v must be 16-byte aligned");
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int32_t *d_rows = nullptr, *d_keep = nullptr;
    float* scratch = nullptr;
    auto release = [&]() {                                   // stream-ordered: safe whether or not the kernel was enqueued
        cudaError_t first = cudaSuccess;
        for (void* b : {static_cast<void*>(scratch), static_cast<void*>(d_keep), static_cast<void*>(d_rows)})
            if (b) { cudaError_t e = cudaFreeAsync(b, st); if (first == cudaSuccess) first = e; }
        return first;
    };
#define CURVE_TRY(expr)                                                                                  \
    do {                                                                                                 \
        cudaError_t err__ = (expr);                                                                      \
        if (err__ != cudaSuccess) {                                                                      \
            release();                                                                                   \
            return fail(SPARSE_ATTN_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(err__));        \
        }                                                                                                \
    } while (0)
    CURVE_TRY(cudaMallocAsync(reinterpret_cast<void**>(&d_rows), sizeof(int32_t) * 2 * n_rows, st));
    CURVE_TRY(cudaMallocAsync(reinterpret_cast<void**>(&d_keep), sizeof(int32_t) * n_keep, st));
    CURVE_TRY(cudaMallocAsync(reinterpret_cast<void**>(&scratch), sizeof(float) * static_cast<size_t>(n_rows) * N, st));
    CURVE_TRY(cudaMemcpyAsync(d_rows, rows, sizeof(int32_t) * 2 * n_rows, cudaMemcpyHostToDevice, st));
    CURVE_TRY(cudaMemcpyAsync(d_keep, keep_counts, sizeof(int32_t) * n_keep, cudaMemcpyHostToDevice, st));
    CURVE_TRY(cudaStreamSynchronize(st));                    // rows / keep_counts may be pageable: the caller may reuse them now
    const float scale = softmax_scale > 0.f ? softmax_scale : 1.0f / std::sqrt(static_cast<float>(D));
    auto qp = static_cast<const __nv_bfloat16*>(q), kp = static_cast<const __nv_bfloat16*>(k), vp = static_cast<const __nv_bfloat16*>(v);
    if (D == 128)
        dsa::row_topk_curve_kernel<128><<<n_rows, dsa::kRowCurveThreads, 0, st>>>(qp, kp, vp, N, scale, d_rows, d_keep, n_keep, scratch,
                                                                                  kurtosis_out, recall_out, mae_out);
    else
        dsa::row_topk_curve_kernel<64><<<n_rows, dsa::kRowCurveThreads, 0, st>>>(qp, kp, vp, N, scale, d_rows, d_keep, n_keep, scratch,
                                                                                 kurtosis_out, recall_out, mae_out);
    CURVE_TRY(cudaGetLastError());
#undef CURVE_TRY
    g_reorder_launches.fetch_add(1);
    CUDA_TRY(release());
    return 0;
}

// ---- sparse_attn_row_topk_curve without any allocation ---------------------------------------------------------------
// Working memory of row_topk_curve_kernel for callers that cannot allocate on the device (a host that has handed all
// of HBM to another allocator, or whose request path must stay away from cudaMalloc / cudaFree): a fixed array in this
// translation unit's device image.  Layout: [0, 16 MiB) fp32 lines of exponentials, then the (bh, r) pairs, then the K list.
// g_curve_static is a HOST-side stand-in in host code -- never pass it to a kernel or a memcpy; the device address comes
// from cudaGetSymbolAddress (curve_static_base below), once per device.
constexpr size_t kCurveStaticLineBytes = sizeof(float) * static_cast<size_t>(SPARSE_ATTN_STATIC_SCRATCH_FLOATS);
constexpr size_t kCurveStaticRowBytes = sizeof(int32_t) * 2 * SPARSE_ATTN_STATIC_MAX_ROWS;
constexpr size_t kCurveStaticKeepBytes = sizeof(int32_t) * SPARSE_ATTN_STATIC_MAX_KEEP;
static __device__ __align__(256) unsigned char g_curve_static[kCurveStaticLineBytes + kCurveStaticRowBytes + kCurveStaticKeepBytes];

namespace {
constexpr int kCurveStaticMaxDevices = 64;
std::atomic<unsigned char*> g_curve_static_base[kCurveStaticMaxDevices];

// Device address of g_curve_static on the CURRENT device: looked up on the first call per device, remembered afterwards
// (two threads racing through the first call both store the same address).
int curve_static_base(unsigned char** base) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    const bool cacheable = dev >= 0 && dev < kCurveStaticMaxDevices;
    if (cacheable) {
        unsigned char* known = g_curve_static_base[dev].load(std::memory_order_acquire);
        if (known) { *base = known; return 0; }
    }
    void* ptr = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&ptr, g_curve_static));
    if (!ptr) return fail(SPARSE_ATTN_ERR_CUDA, "cudaGetSymbolAddress returned a NULL address for the static scratch array");
    if (cacheable) g_curve_static_base[dev].store(static_cast<unsigned char*>(ptr), std::memory_order_release);
    *base = static_cast<unsigned char*>(ptr);
    return 0;
}
}  // namespace

int sparse_attn_row_topk_curve_static(const void* q, const void* k, const void* v, int B, int H, int N, int D,
                                      float softmax_scale, const int32_t* rows, int n_rows, const int32_t* keep_counts,
                                      int n_keep, double* kurtosis_out, double* recall_out, double* mae_out, void* stream) {
    g_last_error[0] = '\0';
    if (!q || !k || !v || !rows || !keep_counts || !kurtosis_out || !recall_out || !mae_out)
        return fail(SPARSE_ATTN_ERR_NULL_POINTER, "q, k, v, rows, keep_counts and the three outputs must not be NULL");
    if (B <= 0 || H <= 0 || N <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "B, H, N must be positive (got %d, %d, %d)", B, H, N);
    if (N > (1 << 24)) return fail(SPARSE_ATTN_ERR_SHAPE, "N = %d exceeds 2^24", N);
    if (D != 64 && D != 128) return fail(SPARSE_ATTN_ERR_HEAD_DIM, "D = %d not in {64, 128}", D);
    if (n_rows <= 0 || n_keep <= 0) return fail(SPARSE_ATTN_ERR_SHAPE, "n_rows and n_keep must be positive (got %d, %d)", n_rows, n_keep);
    if (n_rows > SPARSE_ATTN_STATIC_MAX_ROWS || n_keep > SPARSE_ATTN_STATIC_MAX_KEEP)
        return fail(SPARSE_ATTN_ERR_SHAPE, "n_rows = %d / n_keep = %d exceed the static limits of %d rows and %d K values per call",
                    n_rows, n_keep, SPARSE_ATTN_STATIC_MAX_ROWS, SPARSE_ATTN_STATIC_MAX_KEEP);
    if (static_cast<long long>(n_rows) * N > static_cast<long long>(SPARSE_ATTN_STATIC_SCRATCH_FLOATS))
        return fail(SPARSE_ATTN_ERR_SHAPE, "n_rows * N = %lld exceeds the static scratch of %u floats (16 MiB): at N = %d pass at most "
                    "%d rows per call, or use sparse_attn_row_topk_curve, which allocates",
                    static_cast<long long>(n_rows) * N, SPARSE_ATTN_STATIC_SCRATCH_FLOATS, N,
                    static_cast<int>(SPARSE_ATTN_STATIC_SCRATCH_FLOATS / static_cast<unsigned>(N)));
    if (!(softmax_scale >= 0.f) || std::isinf(softmax_scale))
        return fail(SPARSE_ATTN_ERR_PARAMS, "softmax_scale must be finite and >= 0 (0 = 1/sqrt(D))");
    for (int i = 0; i < n_rows; ++i)
        if (rows[2 * i] < 0 || rows[2 * i] >= B * H || rows[2 * i + 1] < 0 || rows[2 * i + 1] >= N)
            return fail(SPARSE_ATTN_ERR_PARAMS, "rows[%d] = (%d, %d) outside [0, B*H) x [0, N)", i, rows[2 * i], rows[2 * i + 1]);
    for (int i = 0; i < n_keep; ++i)
        if (keep_counts[i] < 1 || keep_counts[i] > N)
            return fail(SPARSE_ATTN_ERR_PARAMS, "keep_counts[%d] = %d outside [1, N]", i, keep_counts[i]);
    if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k) | reinterpret_cast<uintptr_t>(v)) & 15u)
        return fail(SPARSE_ATTN_ERR_ALIGNMENT, "q, k and v must be 16-byte aligned");
    int rc = check_device();
    if (rc) return rc;
    unsigned char* base = nullptr;                           // (first call on this device: the one-time address look-up)
    if ((rc = curve_static_base(&base))) return rc;
    float* lines = reinterpret_cast<float*>(base);
    int32_t* d_rows = reinterpret_cast<int32_t*>(base + kCurveStaticLineBytes);
    int32_t* d_keep = reinterpret_cast<int32_t*>(base + kCurveStaticLineBytes + kCurveStaticRowBytes);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // Nothing in the array has to start at zero: the two lists are overwritten here, and the kernel stores all N logits of
    // a row's line before it reads any of them.  What the previous call left behind is never looked at.
    CUDA_TRY(cudaMemcpyAsync(d_rows, rows, sizeof(int32_t) * 2 * n_rows, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_keep, keep_counts, sizeof(int32_t) * n_keep, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));                     // rows / keep_counts may be pageable: the caller may reuse them now
    const float scale = softmax_scale > 0.f ? softmax_scale : 1.0f / std::sqrt(static_cast<float>(D));
    auto qp = static_cast<const __nv_bfloat16*>(q), kp = static_cast<const __nv_bfloat16*>(k), vp = static_cast<const __nv_bfloat16*>(v);
    if (D == 128)
        dsa::row_topk_curve_kernel<128><<<n_rows, dsa::kRowCurveThreads, 0, st>>>(qp, kp, vp, N, scale, d_rows, d_keep, n_keep, lines,
                                                                                  kurtosis_out, recall_out, mae_out);
    else
        dsa::row_topk_curve_kernel<64><<<n_rows, dsa::kRowCurveThreads, 0, st>>>(qp, kp, vp, N, scale, d_rows, d_keep, n_keep, lines,
                                                                                 kurtosis_out, recall_out, mae_out);
    CUDA_TRY(cudaGetLastError());
    g_reorder_launches.fetch_add(1);
    return 0;
}

double sparse_attn_lambda_from_recall(double recall, int N) { return std::log((1.0 - recall) / N); }

double sparse_attn_lambda_from_preal(double p_real, int tile_k, int N) {
    return std::log(p_real) + std::log(static_cast<double>(tile_k) / N);
}

const char* sparse_attn_status_string(int status) {
    switch (status) {
        case SPARSE_ATTN_OK: return "ok";
        case SPARSE_ATTN_ERR_NULL_POINTER: return "required pointer is NULL";
        case SPARSE_ATTN_ERR_SHAPE: return "bad shape";
        case SPARSE_ATTN_ERR_HEAD_DIM: return "unsupported head dim";
        case SPARSE_ATTN_ERR_TILE: return "unsupported decision tile";
        case SPARSE_ATTN_ERR_MODE: return "bad mode";
        case SPARSE_ATTN_ERR_PARAMS: return "bad params";
        case SPARSE_ATTN_ERR_ALIGNMENT: return "misaligned pointer";
        case SPARSE_ATTN_ERR_DEVICE: return "no sm_100 device";
        case SPARSE_ATTN_ERR_CUDA: return "CUDA error";
        default: return "unknown status";
    }
}

const char* sparse_attn_last_error(void) { return g_last_error; }

int sparse_attn_version(void) { return SPARSE_ATTN_VERSION; }

int64_t sparse_attn_launch_count(void) { return g_launches.load() + g_reorder_launches.load(); }

}  // extern "C"
