// bm_common.cuh -- shared declarations of the CUDA path (internal; the public boundary is include/bm.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bm.h"

namespace bm {

constexpr int kNumSMsFallback = 148;
constexpr unsigned kFullMask = 0xffffffffu;

// ---------------------------------------------------------------------------------------------
// Workspace layout (host-computed; all sections 1024-byte aligned).  Shapes only, never data.
// ---------------------------------------------------------------------------------------------
constexpr int kPermItemsPerBlock = 512;    // (token, slot) items per CTA of the three-kernel permutation
constexpr int kPermSmallItems = 2048;      // up to this many items one CTA does the whole permutation in one launch
constexpr int kMaxSchedTiles = 1 << 20;

struct Workspace {
    // byte offsets from the workspace base ("front": scratch that every call writes before it reads)
    size_t status;       // int32[1024]: [0] device status bits, [1] A (copy of offsets[G]), [2] tokens routed (split
                         // router), [64..64+512) expert slices done per token (split router); zeroed once by the caller,
                         // the counters are put back to zero by the kernel that used them
    size_t block_hist;   // int32[nb * G]   per-block group histograms / bases of the permutation
    size_t route_logits; // router scratch: logits of the split router (T < 512) / row norms and candidate masks of the filter router
    size_t sched;        // int32[kSchedInts] tile-schedule scratch of the forward pass
    size_t xs;           // bf16[T*K, D]    token rows gathered in permuted order (CTA-pair prefill and decode kernels)
    size_t h;            // bf16[T*K + S*T, F]  SwiGLU intermediate
    size_t y;            // bf16[T*K + S*T, D]  per-row expert outputs (two-pass combine only: option FUSED_COMBINE = 0, GEMV fallback)
    size_t front_end;
    // "zero region": anchored at the END of the caller's buffer (see zero_region_base), all-zero between calls -- the
    // kernels that use it put every word back to zero (fused combine: the last arriver of an output piece rounds it,
    // stores it and clears accumulator and ticket).  Offsets are relative to the region's start.
    size_t z_acc;        // f32[T, D]       fp32 accumulation of the gate-weighted combine (GEMM2 epilogues add into it)
    size_t z_tickets;    // int32[T * ceil(D/32) * 4]  arrivals per (token, output piece)
    size_t z_total;
    size_t total;        // front_end + z_total (+ alignment slack)
};

constexpr int kStatusInts = 1024;                               // the zero-once head of the workspace (4096 bytes)
constexpr int kSplitRouterMaxT = 512;                           // the split (latency) router serves T < 512
constexpr int kStatusTokCnt = 64;                               // status[64 + t]: expert slices of token t done
constexpr int kStatusDone = 2;                                  // status[2]: tokens routed
constexpr int kMaxShared = BM_MAX_S;                            // S <= 16 always-on shared experts
constexpr int kSchedInts = 4 + 5 * (BM_MAX_G + kMaxShared) + 8;

__host__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Rows of the SwiGLU intermediate H: one per (token, slot) assignment and per (shared expert, token); the dense decode
// kernels (T <= kDenseMaxT) instead keep a row per (active weight set, token).  Monotone in T.
constexpr int kDenseMaxT = 64;
__host__ inline size_t h_rows_needed(int T, int K, int G, int S) {
    const size_t items = (size_t)T * K;
    const size_t td = T < kDenseMaxT ? T : kDenseMaxT;
    const size_t sets = (size_t)G < td * K ? (size_t)G : td * K;
    const size_t plain = items + (size_t)S * T, dense = (sets + S) * td;
    return plain > dense ? plain : dense;
}

__host__ inline size_t ticket_ints(int T, int D) { return (size_t)T * (size_t)((D + 31) / 32) * 4; }

__host__ inline Workspace workspace_layout(int T, int D, int F, int K, int G, int S) {
    Workspace w{};
    size_t off = 0;
    const size_t items = (size_t)T * K;
    const size_t nb = (items + kPermItemsPerBlock - 1) / kPermItemsPerBlock;
    w.status = off;      off = align_up(off + kStatusInts * sizeof(int32_t), 1024);
    w.block_hist = off;  off = align_up(off + (nb > 0 ? nb : 1) * (size_t)G * sizeof(int32_t), 1024);
    {   // split router (T < 512): logits [T][E]; filter router (T >= 512): row norms [T + E] and candidate masks [T][8]
        const size_t split = (size_t)(T < kSplitRouterMaxT ? T : kSplitRouterMaxT) * BM_MAX_E * sizeof(float);
        const size_t filter = ((size_t)T + BM_MAX_E + 4) * sizeof(float) + (size_t)T * 8 * sizeof(uint32_t);
        w.route_logits = off; off = align_up(off + (split > filter ? split : filter), 1024);
    }
    w.sched = off;       off = align_up(off + kSchedInts * sizeof(int32_t), 1024);
    w.xs = off;          off = align_up(off + items * D * sizeof(bm_bf16), 1024);
    w.h = off;           off = align_up(off + h_rows_needed(T, K, G, S) * F * sizeof(bm_bf16), 1024);
    w.y = off;           off = align_up(off + (items + (size_t)S * T) * D * sizeof(bm_bf16), 1024);
    w.front_end = off;
    size_t z = 0;
    w.z_acc = z;         z = align_up(z + (size_t)T * D * sizeof(float), 1024);
    w.z_tickets = z;     z = align_up(z + ticket_ints(T, D) * sizeof(int32_t), 1024);
    w.z_total = z;
    w.total = w.front_end + w.z_total + 1024;
    return w;
}

// Start of the zero region inside a caller buffer of `workspace_bytes` bytes: anchored at the buffer's end, so that
// the regions of calls with different T (<= T_max) all lie inside [end - z_total(T_max), end), which the front
// sections of no call reach (front_end(T) <= front_end(T_max) <= end - z_total(T_max) - slack).
__host__ inline size_t zero_region_base(size_t workspace_bytes, const Workspace &w) {
    return (workspace_bytes - w.z_total) & ~(size_t)1023;
}

// ---------------------------------------------------------------------------------------------
// Launch bookkeeping (host)
// ---------------------------------------------------------------------------------------------
void count_launch(int n = 1);
// SM count / compute capability of the CURRENT device (cudaGetDevice), cached per device ordinal, so one process
// can drive several GPUs.
int num_sms();
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: raises the opt-in of `fn` on the current device
// to at least `bytes` (no-op below 48 KB or when already granted there).
cudaError_t ensure_dyn_smem(const void *fn, size_t bytes);
// bm_profile_*: record an event pair around the launches of one kernel kind (no-ops unless enabled)
void profile_begin(int kernel, cudaStream_t stream);
void profile_end(int kernel, cudaStream_t stream);

// Programmatic dependent launch (PDL).  Every kernel of the path is launched with
// cudaLaunchAttributeProgrammaticStreamSerialization (unless bm_profile_* is recording or option "PDL" is 0), so
// its prologue overlaps the tail of its predecessor.  Contract for every kernel launched this way:
// all threads call grid_dep_wait() before touching anything a predecessor wrote (or will overwrite)
// and before exiting -- it returns once ALL prerequisite grids have completed and flushed, so the chain
// of launches stays transitively ordered -- and grid_dep_launch() only AFTER that wait.
bool pdl_enabled();

// Tuning / test switches (include/bm.h: bm_set_option).  A plain int table: initialised once from the environment
// (BM_<NAME>) when the library is first used, changed only through bm_set_option -- no getenv on the call path.
enum Opt {
    OPT_PDL, OPT_DECODE_MAX_T, OPT_DECODE_MID_T, OPT_DECODE_ROWS, OPT_DECODE_MID_ROWS, OPT_GEMV_ROWS, OPT_GEMV_MAX_T,
    OPT_GEMV_FUSE, OPT_DC_RMAX, OPT_DC_KS_FORCE, OPT_DC_STAGES, OPT_PF_STAGES, OPT_DC_R1, OPT_DC_R2, OPT_DC_KS2,
    OPT_PF_PAIR, OPT_PF_GATHER, OPT_COMBINE_WARPS, OPT_PERM_SMALL_WARPS, OPT_ROUTER_WE, OPT_ROUTER_TP_MIN_T,
    OPT_ROUTER_SPLIT_MAX_T, OPT_FUSED_COMBINE, OPT_PF_G1_BC, OPT_PF_G2_BC, OPT_PF_G2_BW, OPT_PF_G1_HINTS, OPT_PF_G2_HINTS, OPT_DC_DENSE_MAX_T, OPT_DC_PREFETCH_MB, OPT_DC_KPACK, OPT_ROUTER_FILTER, OPT_HOST_CHUNK_T, OPT_LAYER_SMALL, OPT_PERM_CLUSTER, OPT_DC_SPEC_US, OPT_DC_SPEC_MIN_ROWS, OPT_PF_SPEC, OPT_COUNT
};
int opt(Opt o);

template <typename... KArgs, typename... Args>
cudaError_t launch_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                          Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    count_launch();
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// ---------------------------------------------------------------------------------------------
// Internal kernel launchers (defined in the .cu files, called from bm_api.cu)
// ---------------------------------------------------------------------------------------------
// group map of a routing call: gmap [E] with values in [0,G); cold [E] or nullptr.  nullptr = full brownout
// (every expert e -> set gmap[e]); otherwise partial brownout: cold[e] != 0 -> set gmap[e], else set G + e.
struct GroupMap {
    const int32_t *gmap;
    const int32_t *cold;
    int G;
};

// *fused_permute is set when the router kernel also ran the permutation (small batches: its last CTA does it)
cudaError_t launch_router(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E,
                          int K, GroupMap gm, const bm_routing &r, int32_t *status, float *route_logits,
                          bool *fused_permute, cudaStream_t stream);

cudaError_t launch_permute(int T, int K, int G, const bm_routing &r, int32_t *block_hist, int32_t *status,
                           cudaStream_t stream);

struct ForwardArgs {
    const bm_bf16 *x;
    int T, D, F, K, G, S;
    bm_routing r;
    const bm_bf16 *W1, *W3, *W2;
    bm_bf16 *out;
    // workspace sections
    int32_t *status;
    bm_bf16 *xs;
    bm_bf16 *h;
    float *out_acc;      // zero region: fp32 accumulator of the fused combine
    int32_t *tickets;    // zero region: arrival counters of the fused combine
    bm_bf16 *y;
    float *out_f32;      // non-null: leave the fp32 sums here instead of writing bf16 `out` (tensor-parallel partial)
    bool after_router;   // bm_moe_layer: the routing kernels of the same call are this call's direct predecessors in the stream
};

cudaError_t launch_unite(const bm_bf16 *W, int E, size_t n, const int32_t *gmap, int G, bm_bf16 *out,
                         cudaStream_t stream);

cudaError_t launch_expert_outputs(const bm_bf16 *x, int T, int D, const bm_bf16 *W1, const bm_bf16 *W3,
                                  const bm_bf16 *W2, int E, int F, bm_bf16 *y, bm_bf16 *h, cudaStream_t stream);

cudaError_t launch_expert_hist(const int32_t *expert_ids, long long items, int E, int32_t *w, cudaStream_t stream);
size_t gram_workspace_bytes(int E);
cudaError_t launch_gram(const bm_bf16 *Y, int E, int T, int D, float *gram, float *cosine, float *partial,
                        cudaStream_t stream);
int mse_blocks();
cudaError_t launch_group_mse(const bm_bf16 *Y, const bm_bf16 *U, int T, int D, const int32_t *w, const int32_t *gmap,
                             int E, int G, float *mse, float *mse_total, float *part, cudaStream_t stream);

cudaError_t launch_round_bf16(const float *in, size_t n, bm_bf16 *out, cudaStream_t stream);

cudaError_t launch_forward_simt(const ForwardArgs &a, cudaStream_t stream);
cudaError_t launch_forward_tc(const ForwardArgs &a, bool decode, cudaStream_t stream);
cudaError_t launch_forward_gemv(const ForwardArgs &a, cudaStream_t stream);
int decode_ksplit(int T, int D, int F, int K, int G, int S);     // K splits the decode GEMM2 would use
cudaError_t launch_combine(const ForwardArgs &a, cudaStream_t stream);
cudaError_t launch_layer_small(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                               const int32_t *gmap, int G, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int F, int S,
                               bm_bf16 *out, const bm_routing &r, bm_bf16 *h, float *logits, int32_t *status, bool *handled,
                               cudaStream_t stream);

// ---------------------------------------------------------------------------------------------
// Device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// fp32 -> bf16 bits, round to nearest even (finite inputs; NaN stays NaN)
__device__ __forceinline__ uint32_t f32_to_bf16_bits(float f) {
    uint32_t u = __float_as_uint(f);
    if ((u & 0x7fffffffu) > 0x7f800000u) return (u >> 16) | 0x40u;   // quiet NaN
    u += 0x7fffu + ((u >> 16) & 1u);
    return u >> 16;
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    return f32_to_bf16_bits(lo) | (f32_to_bf16_bits(hi) << 16);
}

}  // namespace bm
