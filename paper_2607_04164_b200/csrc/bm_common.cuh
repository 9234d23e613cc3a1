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
    // byte offsets from the workspace base
    size_t status;       // int32[1024]: [0] device status bits, [1] A (copy of offsets[G]), [2] tokens routed (split
                         // router), [64..64+512) expert slices done per token (split router); zeroed once by the caller,
                         // the counters are put back to zero by the kernel that used them
    size_t block_hist;   // int32[nb * G]   per-block group histograms / bases of the permutation
    size_t route_logits; // f32[min(T, 512) * BM_MAX_E]  logits of the split router (T < 512), gathered by a token's last CTA
    size_t sched;        // int32[kSchedInts] tile-schedule scratch of the forward pass
    size_t xs;           // bf16[T*K, D]    token rows gathered in permuted order (prefill path)
    size_t h;            // bf16[T*K + S*T, F]  SwiGLU intermediate
    size_t out_acc;      // f32[T, D]       fp32 accumulation of the combine (decode path: split-K partials)
    size_t y;            // bf16[T*K + S*T, D]  per-row expert outputs (prefill path), combined by combine_kernel
    size_t total;
};

constexpr int kStatusInts = 1024;                               // the zero-once head of the workspace (4096 bytes)
constexpr int kSplitRouterMaxT = 512;                           // the split (latency) router serves T < 512
constexpr int kStatusTokCnt = 64;                               // status[64 + t]: expert slices of token t done
constexpr int kStatusDone = 2;                                  // status[2]: tokens routed
constexpr int kMaxShared = 16;                                  // S <= 16 always-on shared experts
constexpr int kSchedInts = 4 + 5 * (BM_MAX_G + kMaxShared) + 8;

__host__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

__host__ inline Workspace workspace_layout(int T, int D, int F, int K, int G, int S) {
    Workspace w{};
    size_t off = 0;
    const size_t items = (size_t)T * K;
    const size_t nb = (items + kPermItemsPerBlock - 1) / kPermItemsPerBlock;
    w.status = off;      off = align_up(off + kStatusInts * sizeof(int32_t), 1024);
    w.block_hist = off;  off = align_up(off + (nb > 0 ? nb : 1) * (size_t)G * sizeof(int32_t), 1024);
    w.route_logits = off; off = align_up(off + (size_t)(T < kSplitRouterMaxT ? T : kSplitRouterMaxT) * BM_MAX_E * sizeof(float), 1024);
    w.sched = off;       off = align_up(off + kSchedInts * sizeof(int32_t), 1024);
    w.xs = off;          off = align_up(off + items * D * sizeof(bm_bf16), 1024);
    w.h = off;           off = align_up(off + (items + (size_t)S * T) * F * sizeof(bm_bf16), 1024);
    w.out_acc = off;     off = align_up(off + (size_t)T * D * sizeof(float), 1024);
    w.y = off;           off = align_up(off + (items + (size_t)S * T) * D * sizeof(bm_bf16), 1024);
    w.total = off;
    return w;
}

// ---------------------------------------------------------------------------------------------
// Launch bookkeeping (host)
// ---------------------------------------------------------------------------------------------
void count_launch(int n = 1);
int num_sms();
// bm_profile_*: record an event pair around the launches of one kernel kind (no-ops unless enabled)
void profile_begin(int kernel, cudaStream_t stream);
void profile_end(int kernel, cudaStream_t stream);

// Programmatic dependent launch (PDL).  Every kernel of the path is launched with
// cudaLaunchAttributeProgrammaticStreamSerialization (unless bm_profile_* is recording or BM_PDL=0), so
// its prologue overlaps the tail of its predecessor.  Contract for every kernel launched this way:
// all threads call grid_dep_wait() before touching anything a predecessor wrote (or will overwrite)
// and before exiting -- it returns once ALL prerequisite grids have completed and flushed, so the chain
// of launches stays transitively ordered -- and grid_dep_launch() only AFTER that wait.
bool pdl_enabled();
int tune_int(const char *env_name, int dflt);      // integer tuning override from the environment

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
    int32_t *sched;
    bm_bf16 *xs;
    bm_bf16 *h;
    float *out_acc;
    bm_bf16 *y;
    float *out_f32;      // non-null: leave the fp32 sums here instead of writing bf16 `out` (tensor-parallel partial)
};

cudaError_t launch_unite(const bm_bf16 *W, int E, size_t n, const int32_t *gmap, int G, bm_bf16 *out,
                         cudaStream_t stream);

cudaError_t launch_expert_outputs(const bm_bf16 *x, int T, int D, const bm_bf16 *W1, const bm_bf16 *W3,
                                  const bm_bf16 *W2, int E, int F, bm_bf16 *y, int32_t *sched, bm_bf16 *h,
                                  cudaStream_t stream);

cudaError_t launch_expert_hist(const int32_t *expert_ids, long long items, int E, int32_t *w, cudaStream_t stream);
size_t gram_workspace_bytes(int E);
cudaError_t launch_gram(const bm_bf16 *Y, int E, size_t n, float *gram, float *cosine, float *partial,
                        cudaStream_t stream);
int mse_blocks();
cudaError_t launch_group_mse(const bm_bf16 *Y, const bm_bf16 *U, int T, int D, const int32_t *w, const int32_t *gmap,
                             int E, int G, float *mse, float *mse_total, float *part, cudaStream_t stream);

cudaError_t launch_round_bf16(const float *in, size_t n, bm_bf16 *out, cudaStream_t stream);

cudaError_t launch_forward_simt(const ForwardArgs &a, cudaStream_t stream);
cudaError_t launch_forward_tc(const ForwardArgs &a, bool decode, cudaStream_t stream);
cudaError_t launch_forward_gemv(const ForwardArgs &a, cudaStream_t stream);
cudaError_t launch_combine(const ForwardArgs &a, cudaStream_t stream);

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
