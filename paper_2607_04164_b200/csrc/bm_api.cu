// bm_api.cu -- the C-ABI entry points of include/bm.h: argument checking, workspace carving, path
// dispatch.  No compute happens on the host and there is no CPU fallback.
#include <atomic>
#include <cstdlib>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "bm_common.cuh"

namespace bm {

static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// bm_profile_*: g_prof_kernel = the kind being recorded (BM_KERNEL_ALL: every kind), one event pair per launch
static int g_prof_kernel = 0, g_prof_max = 0, g_prof_n = 0;
static cudaEvent_t *g_prof_start = nullptr, *g_prof_stop = nullptr;
static int *g_prof_kind = nullptr;

void profile_begin(int kernel, cudaStream_t stream) {
    if ((kernel == g_prof_kernel || g_prof_kernel == BM_KERNEL_ALL) && g_prof_n < g_prof_max)
        cudaEventRecord(g_prof_start[g_prof_n], stream);
}
void profile_end(int kernel, cudaStream_t stream) {
    if ((kernel == g_prof_kernel || g_prof_kernel == BM_KERNEL_ALL) && g_prof_n < g_prof_max) {
        g_prof_kind[g_prof_n] = kernel;
        cudaEventRecord(g_prof_stop[g_prof_n++], stream);
    }
}

// ---- options (bm_set_option / bm_get_option) ---------------------------------------------------------------
struct OptDef { const char *name; int dflt; };
static const OptDef kOptDefs[OPT_COUNT] = {
    {"PDL", 1}, {"DECODE_MAX_T", BM_DECODE_MAX_T}, {"DECODE_MID_T", 192}, {"DECODE_ROWS", 44}, {"DECODE_MID_ROWS", 128},
    {"GEMV_ROWS", 1}, {"GEMV_MAX_T", 2}, {"GEMV_FUSE", 1}, {"DC_RMAX", 128}, {"DC_KS_FORCE", 0}, {"DC_STAGES", 12},
    {"PF_STAGES", 12}, {"DC_R1", 0}, {"DC_R2", 0}, {"DC_KS2", 1}, {"PF_PAIR", -1}, {"PF_GATHER", 1},
    {"COMBINE_WARPS", 64}, {"PERM_SMALL_WARPS", 0}, {"ROUTER_WE", 0}, {"ROUTER_TP_MIN_T", kSplitRouterMaxT},
    {"ROUTER_SPLIT_MAX_T", 16}, {"FUSED_COMBINE", -1}, {"PF_G1_BC", -1}, {"PF_G2_BC", -1}, {"PF_G2_BW", -1}, {"PF_G1_HINTS", -1}, {"PF_G2_HINTS", -1}, {"DC_DENSE_MAX_T", kDenseMaxT}, {"DC_PREFETCH_MB", 48}, {"DC_KPACK", 2}, {"ROUTER_FILTER", 1}, {"HOST_CHUNK_T", -1}, {"LAYER_SMALL", 1}, {"PERM_CLUSTER", 1}, {"DC_SPEC_US", 12}, {"DC_SPEC_MIN_ROWS", 1}, {"PF_SPEC", 1},
};
static int g_opt[OPT_COUNT];
static bool init_options() {
    for (int i = 0; i < OPT_COUNT; ++i) {
        g_opt[i] = kOptDefs[i].dflt;
        char env[64];
        std::snprintf(env, sizeof(env), "BM_%s", kOptDefs[i].name);
        const char *v = std::getenv(env);          // once, at first use of the library
        if (v && *v) {
            char *end = nullptr;
            const long r = std::strtol(v, &end, 10);
            if (end && *end == '\0') g_opt[i] = (int)r;
        }
    }
    return true;
}
static void options_ready() { static const bool done = init_options(); (void)done; }
int opt(Opt o) { options_ready(); return g_opt[o]; }

// PDL is off while bm_profile_* records (events between launches would time overlapped kernels) and when option
// "PDL" is 0.
bool pdl_enabled() { return opt(OPT_PDL) != 0 && g_prof_kernel == 0; }

// ---- per-device facts --------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
struct DeviceInfo { int state = 0; int sms = 0; int cc_major = 0; };      // state: 0 = not queried, 1 = queried
static DeviceInfo g_dev[kMaxDevices];
static std::mutex g_dev_mutex;

static const DeviceInfo *device_info(int *ordinal = nullptr) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    if (ordinal) *ordinal = dev;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceInfo &d = g_dev[dev];
    if (d.state == 0) {
        int v = 0, major = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess)
            return nullptr;
        d.sms = v > 0 ? v : kNumSMsFallback;
        d.cc_major = major;
        d.state = 1;
    }
    return &d;
}

int num_sms() {
    const DeviceInfo *d = device_info();
    return d ? d->sms : kNumSMsFallback;
}

// 1 = the current device is sm_100, -1 = it is not (or there is none)
static int device_ok() {
    const DeviceInfo *d = device_info();
    return d && d->cc_major == 10 ? 1 : -1;
}

// dynamic shared memory opt-in, remembered per (device, kernel)
struct SmemGrant { const void *fn; size_t bytes; };
static SmemGrant g_smem[kMaxDevices][64];
cudaError_t ensure_dyn_smem(const void *fn, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    SmemGrant *slot = nullptr;
    for (SmemGrant &g : g_smem[dev]) {
        if (g.fn == fn) { slot = &g; break; }
        if (!g.fn) { slot = &g; break; }
    }
    if (slot && slot->fn == fn && slot->bytes >= bytes) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && slot) { slot->fn = fn; slot->bytes = bytes; }
    return e;
}

static inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_shapes(int T, int D, int F, int E, int K, int G, int S, bool with_f) {
    if (T < 0 || D < 8 || D % 8 != 0) return BM_ERR_SHAPE;
    if (E < 1 || E > BM_MAX_E || K < 1 || K > E || K > BM_MAX_K) return BM_ERR_SHAPE;
    if (G < 1 || G > BM_MAX_G) return BM_ERR_SHAPE;
    if (with_f && (F < 8 || F % 8 != 0 || S < 0 || S > kMaxShared)) return BM_ERR_SHAPE;
    if ((long long)T * K > 0x3fffffffLL) return BM_ERR_SHAPE;
    return BM_OK;
}

}  // namespace bm

using namespace bm;

extern "C" {

size_t bm_workspace_bytes(int T_max, int D, int F, int E, int K, int G, int S) {
    (void)E;
    if (T_max < 0 || D < 1 || F < 1 || K < 1 || G < 1 || S < 0 || S > BM_MAX_S) return 0;
    return workspace_layout(T_max, D, F, K, G, S).total;
}

int bm_workspace_init(void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    if (!workspace) return BM_ERR_NULL;
    if (device_ok() != 1) return BM_ERR_CUDA;
    return cudaMemsetAsync(workspace, 0, workspace_bytes, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

// shared body of bm_route (cold_mask == nullptr) and bm_route_partial
static int route_common(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E,
                        int K, const int32_t *group_map, int G, const int32_t *cold_mask, bool partial,
                        bm_routing *routing, void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    if (!routing) return BM_ERR_NULL;
    int rc = check_shapes(T, D, 8, E, K, G, 0, false);
    if (rc != BM_OK) return rc;
    const int NS = partial ? G + E : G;            // weight sets the routing arrays range over
    if (NS > BM_MAX_G) return BM_ERR_SHAPE;
    routing->T = T; routing->E = E; routing->K = K; routing->G = NS;
    if (!W_router || !group_map || !workspace || !routing->counts || !routing->offsets) return BM_ERR_NULL;
    if (partial && !cold_mask) return BM_ERR_NULL;
    if (T > 0 && (!x || !routing->expert_ids || !routing->group_ids || !routing->gate_w || !routing->n_slots ||
                  !routing->row_token || !routing->row_slot || !routing->slot_row))
        return BM_ERR_NULL;
    if (!aligned16(x) || !aligned16(W_router) || !aligned16(workspace)) return BM_ERR_ALIGN;
    // only the routing part of the workspace is needed here (F = 8, S = 0 gives its lower bound)
    const Workspace full = workspace_layout(T, D, 8, K, NS, 0);
    if (workspace_bytes < full.sched) return BM_ERR_WORKSPACE;
    if (device_ok() != 1) return BM_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    uint8_t *ws = static_cast<uint8_t *>(workspace);
    int32_t *status = reinterpret_cast<int32_t *>(ws + full.status);
    if (T == 0) {
        // empty batch: counts = 0, offsets = 0
        if (cudaMemsetAsync(routing->counts, 0, sizeof(int32_t) * NS, st) != cudaSuccess ||
            cudaMemsetAsync(routing->offsets, 0, sizeof(int32_t) * (NS + 1), st) != cudaSuccess)
            return BM_ERR_CUDA;
        return BM_OK;
    }
    profile_begin(BM_KERNEL_ROUTER, st);
    bool fused_permute = false;
    if (launch_router(x, T, D, W_router, router_bias, E, K, GroupMap{group_map, partial ? cold_mask : nullptr, G},
                      *routing, status, reinterpret_cast<float *>(ws + full.route_logits), &fused_permute, st) != cudaSuccess)
        return BM_ERR_CUDA;
    profile_end(BM_KERNEL_ROUTER, st);
    profile_begin(BM_KERNEL_PERMUTE, st);
    if (!fused_permute &&
        launch_permute(T, K, NS, *routing, reinterpret_cast<int32_t *>(ws + full.block_hist), status, st) != cudaSuccess)
        return BM_ERR_CUDA;
    profile_end(BM_KERNEL_PERMUTE, st);
    return BM_OK;
}

int bm_route(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
             const int32_t *group_map, int G, bm_routing *routing, void *workspace, size_t workspace_bytes,
             bm_stream_t stream) {
    return route_common(x, T, D, W_router, router_bias, E, K, group_map, G, nullptr, false, routing, workspace,
                        workspace_bytes, stream);
}

int bm_route_partial(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
                     const int32_t *group_map, int G, const int32_t *cold_mask, bm_routing *routing, void *workspace,
                     size_t workspace_bytes, bm_stream_t stream) {
    return route_common(x, T, D, W_router, router_bias, E, K, group_map, G, cold_mask, true, routing, workspace,
                        workspace_bytes, stream);
}

// -------------------------------------------------------------------------------------------------
// bm_route_static: bm_route for callers that may not allocate (CUDA graph capture, serving loops, harnesses without
// cudaMalloc).  Its scratch -- the routing part of a workspace: status word and arrival counters, per-block histograms of
// the permutation, logits / row norms / candidate masks of the router -- is the file-scope device array below, which every
// GPU that loads the library holds until the process exits.  In host code the array's NAME is a host-side stand-in, not a
// device address: its device address is looked up once per device with cudaGetSymbolAddress (that device current) and
// that pointer is what the kernels get.
// -------------------------------------------------------------------------------------------------
constexpr size_t kStaticRouteBytes = (size_t)BM_STATIC_ROUTE_BYTES;
static __device__ __align__(256) unsigned char g_static_route_scratch[kStaticRouteBytes];
static void *g_static_route_ptr[kMaxDevices];       // device address of the array on device i, nullptr = not looked up yet

static void *static_route_scratch() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (!g_static_route_ptr[dev]) {
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_static_route_scratch) != cudaSuccess || !ptr) {
            cudaGetLastError();
            return nullptr;
        }
        g_static_route_ptr[dev] = ptr;
    }
    return g_static_route_ptr[dev];
}

int bm_route_static(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
                    const int32_t *group_map, int G, bm_routing *routing, bm_stream_t stream) {
    if (!routing) return BM_ERR_NULL;
    int rc = check_shapes(T, D, 8, E, K, G, 0, false);
    if (rc != BM_OK) return rc;
    // the limit, checked on the host before anything else: the routing scratch of this (T, K, G) must fit the array
    if (T > BM_STATIC_ROUTE_MAX_T || workspace_layout(T, D, 8, K, G, 0).sched > kStaticRouteBytes) return BM_ERR_LIMIT;
    if (device_ok() != 1) return BM_ERR_CUDA;
    void *scratch = static_route_scratch();
    if (!scratch) return BM_ERR_CUDA;
    // The array keeps what the last call left.  What a call needs to find zero is the 4096-byte head (status word, arrival
    // counters): cleared here, on `stream`, ahead of the kernels -- so the status word afterwards holds THIS call's bits.
    if (T > 0 && cudaMemsetAsync(scratch, 0, kStatusInts * sizeof(int32_t), reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
        return BM_ERR_CUDA;
    return route_common(x, T, D, W_router, router_bias, E, K, group_map, G, nullptr, false, routing, scratch,
                        kStaticRouteBytes, stream);
}

int bm_route_static_status(int32_t *host_out, bm_stream_t stream) {
    if (!host_out) return BM_ERR_NULL;
    if (device_ok() != 1) return BM_ERR_CUDA;
    void *scratch = static_route_scratch();
    if (!scratch) return BM_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (cudaMemcpyAsync(host_out, scratch, sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BM_ERR_CUDA;
    return BM_OK;
}

int bm_unite_weights(const bm_bf16 *W, int E, size_t n, const int32_t *group_map, int G, bm_bf16 *out,
                     bm_stream_t stream) {
    if (E < 1 || E > BM_MAX_E || G < 1 || G > BM_MAX_G || n % 8 != 0) return BM_ERR_SHAPE;
    if (n == 0) return BM_OK;
    if (!W || !group_map || !out) return BM_ERR_NULL;
    if (!aligned16(W) || !aligned16(out)) return BM_ERR_ALIGN;
    if (device_ok() != 1) return BM_ERR_CUDA;
    return launch_unite(W, E, n, group_map, G, out, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

int bm_expert_histogram(const int32_t *expert_ids, int T, int K, int E, int32_t *w, bm_stream_t stream) {
    if (T < 0 || K < 1 || E < 1 || E > BM_MAX_E || (long long)T * K > 0x3fffffffLL) return BM_ERR_SHAPE;
    if (!w || (T > 0 && !expert_ids)) return BM_ERR_NULL;
    if (device_ok() != 1) return BM_ERR_CUDA;
    return launch_expert_hist(expert_ids, (long long)T * K, E, w, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

size_t bm_expert_outputs_workspace_bytes(int T, int D, int F, int E) {
    if (T < 0 || D < 1 || F < 1 || E < 1 || E > BM_MAX_G) return 0;
    return workspace_layout(T, D, F, 1, 1, E).front_end;
}

int bm_expert_outputs(const bm_bf16 *x, int T, int D, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int E,
                      int F, bm_bf16 *y, void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    if (T < 0 || D < 8 || D % 8 != 0 || F < 8 || F % 8 != 0 || E < 1 || E > BM_MAX_G) return BM_ERR_SHAPE;
    if ((long long)T * E > 0x3fffffffLL) return BM_ERR_SHAPE;
    if (T == 0) return BM_OK;
    if (!x || !W1 || !W3 || !W2 || !y || !workspace) return BM_ERR_NULL;
    if (!aligned16(x) || !aligned16(W1) || !aligned16(W3) || !aligned16(W2) || !aligned16(y) || !aligned16(workspace))
        return BM_ERR_ALIGN;
    const Workspace w = workspace_layout(T, D, F, 1, 1, E);
    if (workspace_bytes < w.front_end) return BM_ERR_WORKSPACE;
    if (device_ok() != 1) return BM_ERR_CUDA;
    uint8_t *ws = static_cast<uint8_t *>(workspace);
    return launch_expert_outputs(x, T, D, W1, W3, W2, E, F, y, reinterpret_cast<bm_bf16 *>(ws + w.h),
                                 reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

size_t bm_gram_workspace_bytes(int E) {
    if (E < 1 || E > 128) return 0;
    return (size_t)256 * E * E * sizeof(float);          // one partial tile per CTA, any SM count up to 256
}

int bm_cosine_gram(const bm_bf16 *Y, int E, int T, int D, float *gram, float *cosine, void *workspace,
                   size_t workspace_bytes, bm_stream_t stream) {
    if (E < 1 || E > 128 || T < 1 || D < 8 || D % 8 != 0 || (long long)T * ((D + 63) / 64) > 0x7fffff00LL) return BM_ERR_SHAPE;
    if (!Y || !gram || !workspace) return BM_ERR_NULL;
    if (!aligned16(Y) || !aligned16(workspace)) return BM_ERR_ALIGN;
    if (workspace_bytes < bm_gram_workspace_bytes(E)) return BM_ERR_WORKSPACE;
    if (device_ok() != 1) return BM_ERR_CUDA;
    if (num_sms() > 256) return BM_ERR_CUDA;
    return launch_gram(Y, E, T, D, gram, cosine, static_cast<float *>(workspace), reinterpret_cast<cudaStream_t>(stream)) ==
                   cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

size_t bm_mse_workspace_bytes(int G) {
    if (G < 1 || G > BM_MAX_G) return 0;
    return ((size_t)256 * 8 + (size_t)G) * sizeof(float) * 2;   // >= G * blocks-per-group partial sums (see launch_group_mse)
}

int bm_group_mse(const bm_bf16 *Y, const bm_bf16 *U, int T, int D, const int32_t *w, const int32_t *group_map, int E,
                 int G, float *mse, float *mse_total, void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    if (T < 1 || D < 8 || D % 8 != 0 || E < 1 || E > BM_MAX_E || G < 1 || G > BM_MAX_G) return BM_ERR_SHAPE;
    if (!Y || !U || !w || !group_map || !mse || !mse_total || !workspace) return BM_ERR_NULL;
    if (!aligned16(Y) || !aligned16(U)) return BM_ERR_ALIGN;
    if (workspace_bytes < bm_mse_workspace_bytes(G)) return BM_ERR_WORKSPACE;
    if (device_ok() != 1) return BM_ERR_CUDA;
    if ((size_t)(mse_blocks() / G + 1) * G * sizeof(float) > workspace_bytes) return BM_ERR_WORKSPACE;
    return launch_group_mse(Y, U, T, D, w, group_map, E, G, mse, mse_total, static_cast<float *>(workspace),
                            reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess
               ? BM_OK : BM_ERR_CUDA;
}

// BM_PATH_AUTO -> the path a batch of these host-side sizes takes
static int resolve_auto_path(int T, int K, int G, int D, int F) {

    // decode (swap-AB weight streaming) for small batches: always up to 64 tokens; up to DECODE_MID_T = 192 tokens (256
    // where a weight set has >= 64 MB: long items) while a group expects at most one 128-row chunk (the weights then
    // stream once); up to DECODE_MAX_T = 320 tokens while a group expects at most ~44 rows.  Measured, forward only,
    // decode / prefill kernels (us; cold weights):
    //   D = 2048, F = 1408, E = 60, top-4:
    //     G = 8:   T = 128 48 / 56,   T = 192 51 / 52,    T = 256 55 / 50,    T = 320 59 / 49
    //     G = 15:  T = 128 58 / 71,   T = 192 64 / 69,    T = 256 75 / 70,    T = 320 77 / 68
    //     G = 30:  T = 192 97 / 113,  T = 256 111 / 115,  T = 320 112 / 113,  T = 384 115 / 110
    //     G = 60:  T = 192 170 / 193, T = 256 194 / 191,  T = 320 195 / 197,  T = 384 202 / 192
    //   D = 4096, F = 14336, E = 8, top-2, G = 4:  T = 128 240 / 301, T = 192 300 / 375, T = 256 334 / 359, T = 320 423 / 397
    const int max_t = opt(OPT_DECODE_MAX_T);
    int mid_t = opt(OPT_DECODE_MID_T);
    if (mid_t == 192 && (long long)D * F * 2 >= (64LL << 20)) mid_t = 256;
    const bool few_rows = (long long)T * K <= (long long)opt(OPT_DECODE_ROWS) * G;
    const bool one_chunk = (long long)T * K <= (long long)opt(OPT_DECODE_MID_ROWS) * G;
    int path = (T <= 64 || (T <= mid_t && one_chunk) || (T <= max_t && few_rows)) ? BM_PATH_DECODE : BM_PATH_PREFILL;
    // matrix-vector streaming for one or two tokens whose sets expect at most ~1 row (single-token decode above
    // all): the tcgen05 k-block loop has a latency floor that such a step never fills (see bm_gemv.cu).
    // Measured (D = 2048, F = 1408, E = 60, top-4; matrix-vector / tensor path): T = 1: 29-30 / 36-39 us,
    // T = 2: 42-44 / 43-45 us, T = 3: 53-55 / 51-53 us, T = 8 at G = 60: 93 / 77 us -- beyond two tokens the
    // token-major W2 stage re-reads weight rows per (token, source) and the equal unit ranges lose balance.
    const int gemv_rows = opt(OPT_GEMV_ROWS);
    const int gemv_max_t = opt(OPT_GEMV_MAX_T);
    if (T <= gemv_max_t && (long long)T * K <= (long long)gemv_rows * G) path = BM_PATH_GEMV;
    return path;
}

static int forward_common(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1,
                          const bm_bf16 *W3, const bm_bf16 *W2, int F, int S, bm_bf16 *out, float *out_f32,
                          void *workspace, size_t workspace_bytes, bm_stream_t stream, int path, bool after_router = false) {
    if (!routing) return BM_ERR_NULL;
    const int K = routing->K, G = routing->G;
    int rc = check_shapes(T, D, F, routing->E, K, G, S, true);
    if (rc != BM_OK) return rc;
    if (routing->T != T) return BM_ERR_SHAPE;
    if (path < BM_PATH_AUTO || path > BM_PATH_GEMV) return BM_ERR_PATH;
    if (out_f32 && path == BM_PATH_SIMT) return BM_ERR_PATH;
    if (T == 0) return BM_OK;
    if (!x || !W1 || !W3 || !W2 || (!out && !out_f32) || !workspace || !routing->group_ids || !routing->gate_w ||
        !routing->n_slots || !routing->counts || !routing->offsets || !routing->row_token || !routing->row_slot ||
        !routing->slot_row)
        return BM_ERR_NULL;
    if (!aligned16(x) || !aligned16(W1) || !aligned16(W3) || !aligned16(W2) || !aligned16(out) || !aligned16(out_f32) ||
        !aligned16(workspace))
        return BM_ERR_ALIGN;
    const Workspace w = workspace_layout(T, D, F, K, G, S);
    if (workspace_bytes < w.total) return BM_ERR_WORKSPACE;
    if (device_ok() != 1) return BM_ERR_CUDA;

    if (path == BM_PATH_AUTO) path = resolve_auto_path(T, K, G, D, F);

    uint8_t *ws = static_cast<uint8_t *>(workspace);
    ForwardArgs a{};
    a.x = x; a.T = T; a.D = D; a.F = F; a.K = K; a.G = G; a.S = S;
    a.r = *routing;
    a.W1 = W1; a.W3 = W3; a.W2 = W2; a.out = out; a.out_f32 = out_f32;
    a.after_router = after_router;
    a.status = reinterpret_cast<int32_t *>(ws + w.status);
    a.xs = reinterpret_cast<bm_bf16 *>(ws + w.xs);
    a.h = reinterpret_cast<bm_bf16 *>(ws + w.h);
    const size_t zbase = zero_region_base(workspace_bytes, w);
    a.out_acc = reinterpret_cast<float *>(ws + zbase + w.z_acc);
    a.tickets = reinterpret_cast<int32_t *>(ws + zbase + w.z_tickets);
    a.y = reinterpret_cast<bm_bf16 *>(ws + w.y);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (path == BM_PATH_SIMT) e = launch_forward_simt(a, st);
    else if (path == BM_PATH_GEMV) e = launch_forward_gemv(a, st);
    else e = launch_forward_tc(a, path == BM_PATH_DECODE, st);
    return e == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

int bm_moe_forward_path(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1,
                        const bm_bf16 *W3, const bm_bf16 *W2, int F, int S, bm_bf16 *out, void *workspace,
                        size_t workspace_bytes, bm_stream_t stream, int path) {
    if (!out && T > 0) return BM_ERR_NULL;
    return forward_common(x, T, D, routing, W1, W3, W2, F, S, out, nullptr, workspace, workspace_bytes, stream, path);
}

int bm_moe_forward_f32(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1, const bm_bf16 *W3,
                       const bm_bf16 *W2, int F, int S, float *out_f32, void *workspace, size_t workspace_bytes,
                       bm_stream_t stream) {
    if (!out_f32 && T > 0) return BM_ERR_NULL;
    return forward_common(x, T, D, routing, W1, W3, W2, F, S, nullptr, out_f32, workspace, workspace_bytes, stream,
                          BM_PATH_AUTO);
}

int bm_round_bf16(const float *in, size_t n, bm_bf16 *out, bm_stream_t stream) {
    if (n % 8 != 0) return BM_ERR_SHAPE;
    if (n == 0) return BM_OK;
    if (!in || !out) return BM_ERR_NULL;
    if (!aligned16(in) || !aligned16(out)) return BM_ERR_ALIGN;
    if (device_ok() != 1) return BM_ERR_CUDA;
    return launch_round_bf16(in, n, out, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

int bm_moe_forward(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1, const bm_bf16 *W3,
                   const bm_bf16 *W2, int F, int S, bm_bf16 *out, void *workspace, size_t workspace_bytes,
                   bm_stream_t stream) {
    return bm_moe_forward_path(x, T, D, routing, W1, W3, W2, F, S, out, workspace, workspace_bytes, stream,
                               BM_PATH_AUTO);
}

int bm_moe_layer(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
                 const int32_t *group_map, int G, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int F, int S,
                 bm_bf16 *out, bm_routing *routing, void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    // one or two tokens whose sets expect at most one row (the matrix-vector rule of BM_PATH_AUTO): one persistent kernel
    if (routing && T >= 1 && T <= 2 && opt(OPT_LAYER_SMALL) != 0 && resolve_auto_path(T, K, G, D, F) == BM_PATH_GEMV) {
        int rc = check_shapes(T, D, F, E, K, G, S, true);
        if (rc != BM_OK) return rc;
        if (!x || !W_router || !group_map || !W1 || !W3 || !W2 || !out || !workspace || !routing->expert_ids ||
            !routing->group_ids || !routing->gate_w || !routing->n_slots || !routing->counts || !routing->offsets ||
            !routing->row_token || !routing->row_slot || !routing->slot_row)
            return BM_ERR_NULL;
        if (!aligned16(x) || !aligned16(W_router) || !aligned16(W1) || !aligned16(W3) || !aligned16(W2) || !aligned16(out) ||
            !aligned16(workspace))
            return BM_ERR_ALIGN;
        const Workspace w = workspace_layout(T, D, F, K, G, S);
        if (workspace_bytes < w.total) return BM_ERR_WORKSPACE;
        if (device_ok() != 1) return BM_ERR_CUDA;
        routing->T = T; routing->E = E; routing->K = K; routing->G = G;
        uint8_t *ws = static_cast<uint8_t *>(workspace);
        bool handled = false;
        const cudaError_t e = launch_layer_small(x, T, D, W_router, router_bias, E, K, group_map, G, W1, W3, W2, F, S, out, *routing,
                                                 reinterpret_cast<bm_bf16 *>(ws + w.h), reinterpret_cast<float *>(ws + w.route_logits),
                                                 reinterpret_cast<int32_t *>(ws + w.status), &handled,
                                                 reinterpret_cast<cudaStream_t>(stream));
        if (e != cudaSuccess) return BM_ERR_CUDA;
        if (handled) return BM_OK;
    }
    int rc = bm_route(x, T, D, W_router, router_bias, E, K, group_map, G, routing, workspace, workspace_bytes, stream);
    if (rc != BM_OK) return rc;
    if (!out && T > 0) return BM_ERR_NULL;
    // the forward kernels know that the routing kernels run directly before them (speculative dense decode, bm_gemm.cu)
    return forward_common(x, T, D, routing, W1, W3, W2, F, S, out, nullptr, workspace, workspace_bytes, stream, BM_PATH_AUTO, true);
}

// Copy streams and events of bm_moe_layer_host's chunk pipeline, created on first use, one set per device.
constexpr int kHostMaxChunks = 16;
struct HostPipe { bool ready = false; cudaStream_t in = nullptr, out = nullptr; cudaEvent_t ev_in[kHostMaxChunks], ev_cmp[kHostMaxChunks], ev_done; };
static HostPipe g_pipe[kMaxDevices];

static HostPipe *host_pipe() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    HostPipe &p = g_pipe[dev];
    if (!p.ready) {
        if (cudaStreamCreateWithFlags(&p.in, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&p.out, cudaStreamNonBlocking) != cudaSuccess)
            return nullptr;
        for (int i = 0; i < kHostMaxChunks; ++i)
            if (cudaEventCreateWithFlags(&p.ev_in[i], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&p.ev_cmp[i], cudaEventDisableTiming) != cudaSuccess)
                return nullptr;
        if (cudaEventCreateWithFlags(&p.ev_done, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        p.ready = true;
    }
    return &p;
}

// Token chunks of bm_moe_layer_host: equal chunks of whole 128-row tiles, about HOST_CHUNK_T tokens each, from two chunks on.
// The pipeline hides every copy except the first chunk's way in and the last chunk's way out, but every chunk streams the
// layer's weights once more -- BJ:configs[2]'s layer takes 0.51 us per token plus ~210 us per call (1.4 GB of weights): 0.53
// us per token at T = 8192, 0.55 at 4096, 0.63 at 2048, 1.03 at 512.  Measured there, end to end (ms, two boxes): one piece
// 6.12 / 6.08, 8 x 1024 6.34 / 6.25, 4 x 2048 5.36 / 5.26, 3 x 2816 - / 5.01, 2 x 4096 5.21 / 5.11; chunks growing from a small
// first one towards the middle and shrinking again (512, 1536, 4096, 1536, 512: the exposed copies shrink 4x) 5.54 -- small
// chunks cost more than their copies save.  So: 2816 tokens (22 tiles) where a token computes at least twice as long as it
// copies (6 D F (K + S) flops at ~1.3 PFLOP/s against 2 D bytes at ~50 GB/s: F (K + S) >= 17400), 2048 elsewhere (Qwen-like
// shapes: copies as long as compute).  Returns the number of chunks.
static int host_chunk_plan(int T, int F, int K, int S, int *sizes) {
    int chunk_t = opt(OPT_HOST_CHUNK_T);
    if (chunk_t < 0) chunk_t = (long long)F * (K + S) >= 17400 ? 2816 : 2048;
    sizes[0] = T;
    if (chunk_t == 0 || T < 2 * chunk_t) return 1;
    int pieces = (T + chunk_t - 1) / chunk_t;
    if (pieces > kHostMaxChunks) pieces = kHostMaxChunks;
    const int per = ((T + pieces - 1) / pieces + 127) & ~127;
    int n = 0;
    for (int t0 = 0; t0 < T; t0 += per) sizes[n++] = T - t0 < per ? T - t0 : per;
    return n;
}

int bm_host_chunks(int T, int F, int K, int S, int *sizes, int cap) {
    if (T < 0 || F < 1 || K < 1 || S < 0 || cap < 0) return BM_ERR_SHAPE;
    if (cap > 0 && !sizes) return BM_ERR_NULL;
    int plan[kHostMaxChunks];
    const int n = host_chunk_plan(T, F, K, S, plan);
    for (int i = 0; i < n && i < cap; ++i) sizes[i] = plan[i];
    return n;
}

int bm_moe_layer_host(const bm_bf16 *x_host, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E,
                      int K, const int32_t *group_map, int G, const bm_bf16 *W1, const bm_bf16 *W3,
                      const bm_bf16 *W2, int F, int S, bm_bf16 *out_host, bm_bf16 *x_dev, bm_bf16 *out_dev,
                      bm_routing *routing, void *workspace, size_t workspace_bytes, bm_stream_t stream) {
    if (T < 0 || K < 1 || D < 8) return BM_ERR_SHAPE;
    if (!routing) return BM_ERR_NULL;
    if (T > 0 && (!x_host || !out_host || !x_dev || !out_dev)) return BM_ERR_NULL;
    if (device_ok() != 1) return BM_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const size_t row_bytes = (size_t)D * sizeof(bm_bf16);
    // Large batches go through in token chunks (tokens are independent: the layer on a chunk is the layer on its tokens):
    // the host->device copy of chunk c+1 and the device->host copy of chunk c-1 run on two copy streams while chunk c
    // computes, so a PCIe-bound step (BJ:configs[2]: 67 MB each way) costs its compute time plus one chunk of copies.
    int sizes[kHostMaxChunks];
    int n_chunks = host_chunk_plan(T, F, K, S, sizes);
    HostPipe *pipe = n_chunks > 1 ? host_pipe() : nullptr;
    if (!pipe) n_chunks = 1;
    if (n_chunks == 1) {
        if (T > 0 && cudaMemcpyAsync(x_dev, x_host, (size_t)T * row_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return BM_ERR_CUDA;
        int rc = bm_moe_layer(x_dev, T, D, W_router, router_bias, E, K, group_map, G, W1, W3, W2, F, S, out_dev, routing, workspace,
                              workspace_bytes, stream);
        if (rc != BM_OK) return rc;
        if (T > 0 && cudaMemcpyAsync(out_host, out_dev, (size_t)T * row_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess)
            return BM_ERR_CUDA;
        return cudaStreamSynchronize(st) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
    }
    // the copy streams start after whatever the caller queued on `stream` before this call
    if (cudaEventRecord(pipe->ev_done, st) != cudaSuccess || cudaStreamWaitEvent(pipe->in, pipe->ev_done, 0) != cudaSuccess ||
        cudaStreamWaitEvent(pipe->out, pipe->ev_done, 0) != cudaSuccess)
        return BM_ERR_CUDA;
    const bm_routing whole = *routing;
    for (int c = 0, t0 = 0; c < n_chunks; t0 += sizes[c], ++c) {
        const int tc = sizes[c];
        if (cudaMemcpyAsync(x_dev + (size_t)t0 * D, x_host + (size_t)t0 * D, (size_t)tc * row_bytes, cudaMemcpyHostToDevice, pipe->in) != cudaSuccess ||
            cudaEventRecord(pipe->ev_in[c], pipe->in) != cudaSuccess || cudaStreamWaitEvent(st, pipe->ev_in[c], 0) != cudaSuccess)
            return BM_ERR_CUDA;
        bm_routing r = whole;          // the chunk's slices of the caller's arrays; counts / offsets are reused chunk after chunk
        r.expert_ids += (size_t)t0 * K; r.group_ids += (size_t)t0 * K; r.gate_w += (size_t)t0 * K; r.n_slots += t0;
        r.row_token += (size_t)t0 * K; r.row_slot += (size_t)t0 * K; r.slot_row += (size_t)t0 * K;
        int rc = bm_route(x_dev + (size_t)t0 * D, tc, D, W_router, router_bias, E, K, group_map, G, &r, workspace, workspace_bytes, stream);
        if (rc != BM_OK) return rc;
        rc = bm_moe_forward(x_dev + (size_t)t0 * D, tc, D, &r, W1, W3, W2, F, S, out_dev + (size_t)t0 * D, workspace, workspace_bytes, stream);
        if (rc != BM_OK) return rc;
        if (cudaEventRecord(pipe->ev_cmp[c], st) != cudaSuccess || cudaStreamWaitEvent(pipe->out, pipe->ev_cmp[c], 0) != cudaSuccess ||
            cudaMemcpyAsync(out_host + (size_t)t0 * D, out_dev + (size_t)t0 * D, (size_t)tc * row_bytes, cudaMemcpyDeviceToHost, pipe->out) != cudaSuccess)
            return BM_ERR_CUDA;
        routing->T = r.T; routing->E = r.E; routing->K = r.K; routing->G = r.G;
    }
    if (cudaEventRecord(pipe->ev_done, pipe->out) != cudaSuccess || cudaStreamWaitEvent(st, pipe->ev_done, 0) != cudaSuccess)
        return BM_ERR_CUDA;
    return cudaStreamSynchronize(st) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

int bm_device_status(void *workspace, int32_t *host_out, bm_stream_t stream) {
    if (!workspace || !host_out) return BM_ERR_NULL;
    if (device_ok() != 1) return BM_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (cudaMemcpyAsync(host_out, workspace, sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemsetAsync(workspace, 0, sizeof(int32_t), st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BM_ERR_CUDA;
    return BM_OK;
}

int bm_profile_enable(int kernel, int max_records) {
    for (int i = 0; i < g_prof_max; ++i) { cudaEventDestroy(g_prof_start[i]); cudaEventDestroy(g_prof_stop[i]); }
    delete[] g_prof_start; delete[] g_prof_stop; delete[] g_prof_kind;
    g_prof_start = g_prof_stop = nullptr;
    g_prof_kind = nullptr;
    g_prof_kernel = 0; g_prof_max = 0; g_prof_n = 0;
    if (kernel == BM_KERNEL_NONE || max_records <= 0) return BM_OK;
    if (kernel < BM_KERNEL_ROUTER || kernel > BM_KERNEL_ALL) return BM_ERR_SHAPE;
    if (device_ok() != 1) return BM_ERR_CUDA;
    g_prof_start = new cudaEvent_t[max_records];
    g_prof_stop = new cudaEvent_t[max_records];
    g_prof_kind = new int[max_records];
    for (int i = 0; i < max_records; ++i)
        if (cudaEventCreate(&g_prof_start[i]) != cudaSuccess || cudaEventCreate(&g_prof_stop[i]) != cudaSuccess)
            return BM_ERR_CUDA;
    g_prof_kernel = kernel; g_prof_max = max_records;
    return BM_OK;
}

int bm_profile_read_kinds(float *ms_by_kind, int *n_by_kind) {
    if (!ms_by_kind || !n_by_kind) return BM_ERR_NULL;
    for (int k = 0; k < BM_KERNEL_ALL; ++k) { ms_by_kind[k] = 0.f; n_by_kind[k] = 0; }
    for (int i = 0; i < g_prof_n; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(g_prof_stop[i]) != cudaSuccess ||
            cudaEventElapsedTime(&ms, g_prof_start[i], g_prof_stop[i]) != cudaSuccess)
            return BM_ERR_CUDA;
        const int k = g_prof_kind[i];
        if (k > 0 && k < BM_KERNEL_ALL) { ms_by_kind[k] += ms; n_by_kind[k] += 1; }
    }
    g_prof_n = 0;
    return BM_OK;
}

int bm_profile_read(float *total_ms, int *n_records) {
    if (!total_ms || !n_records) return BM_ERR_NULL;
    float ms[BM_KERNEL_ALL];
    int n[BM_KERNEL_ALL];
    const int rc = bm_profile_read_kinds(ms, n);
    if (rc != BM_OK) return rc;
    *total_ms = 0.f; *n_records = 0;
    for (int k = 1; k < BM_KERNEL_ALL; ++k) { *total_ms += ms[k]; *n_records += n[k]; }
    return BM_OK;
}

int bm_forward_info(int T, int K, int G, int S, int D, int F, int *path, int *deterministic) {
    if (T < 0 || K < 1 || K > BM_MAX_K || G < 1 || G > BM_MAX_G || S < 0 || S > BM_MAX_S || D < 8 || F < 8) return BM_ERR_SHAPE;
    const int pth = resolve_auto_path(T, K, G, D, F);
    int det = 1;
    if (pth == BM_PATH_PREFILL) {
        const int fc = opt(OPT_FUSED_COMBINE);
        const bool fused = fc < 0 ? F >= 4096 : fc != 0;          // as launch_forward_tc
        det = (!fused || K + S <= 2) ? 1 : 0;
    }
    else if (pth == BM_PATH_DECODE) det = ((K + S) * decode_ksplit(T, D, F, K, G, S) <= 2) ? 1 : 0;   // fp32 reds either way
    if (path) *path = pth;
    if (deterministic) *deterministic = det;
    return BM_OK;
}

int bm_set_option(const char *name, int value) {
    if (!name) return BM_ERR_NULL;
    options_ready();
    for (int i = 0; i < OPT_COUNT; ++i)
        if (std::strcmp(name, kOptDefs[i].name) == 0) { g_opt[i] = value; return BM_OK; }
    return BM_ERR_SHAPE;
}

int bm_get_option(const char *name, int *value) {
    if (!name || !value) return BM_ERR_NULL;
    options_ready();
    for (int i = 0; i < OPT_COUNT; ++i)
        if (std::strcmp(name, kOptDefs[i].name) == 0) { *value = g_opt[i]; return BM_OK; }
    return BM_ERR_SHAPE;
}

long long bm_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char *bm_status_string(int code) {
    switch (code) {
        case BM_OK: return "BM_OK";
        case BM_ERR_NULL: return "BM_ERR_NULL: a required pointer is NULL";
        case BM_ERR_SHAPE: return "BM_ERR_SHAPE: unsupported or inconsistent shape";
        case BM_ERR_ALIGN: return "BM_ERR_ALIGN: a device pointer is not 16-byte aligned";
        case BM_ERR_WORKSPACE: return "BM_ERR_WORKSPACE: workspace too small";
        case BM_ERR_CUDA: return "BM_ERR_CUDA: no sm_100 device or a CUDA call failed";
        case BM_ERR_PATH: return "BM_ERR_PATH: the forced path cannot run this shape";
        case BM_ERR_LIMIT: return "BM_ERR_LIMIT: sizes beyond the fixed scratch of an entry point that allocates nothing";
        default: return "unknown bm_status";
    }
}

}  // extern "C"
