/*
 * bm.h -- C ABI of the B200-native grouped MoE-layer forward pass (BrownoutMoE full-brownout path), plus the
 *         SURVEY.md 8(f) rows built on it: partial brownout, united-weight construction, the calibration forward and
 *         the per-rank partial of a tensor-parallel layer.
 *
 * The operation (PAPER.md = /root/reference/PAPER.md, "P:NN" = line NN; readings A1..A22 = DESIGN.md):
 *   P:42   MoE layer with E experts and top-K routing:  h_t = sum_{i<=K} g_i(x_t) * FFN_i(x_t),
 *          g_i the gating score.
 *   P:46   united experts / full brownout: every routed expert e is served by the united expert of its
 *          group, "reducing the number of experts loaded during inference".
 *   P:118-122 (Eq. 2): the group map g: expert -> group decides which united expert handles the
 *          tokens originally routed to each expert.
 *   BASELINE.json north_star: bm_route(x, W_router, k, group_map) and
 *          bm_moe_forward(x, routing, united W1/W3/W2, out).
 *
 * Conventions
 *   - bf16 values are passed as uint16_t storage (bm_bf16).  Row-major, innermost dimension last.
 *   - Every pointer is a DEVICE pointer unless its comment says HOST.  The caller owns all memory;
 *     the library never allocates, frees or synchronises (except bm_moe_layer_host,
 *     bm_device_status and the bm_profile_* pair, which say so) and borrows the buffers until the work enqueued on `stream`
 *     has completed.  All device pointers must be 16-byte aligned.
 *   - Workspace.  Call bm_workspace_init once after allocating a workspace (it zeroes it).  Two parts of it must be
 *     all-zero whenever a call starts, and every call that completes leaves them all-zero again: the first 4096
 *     bytes (device status word, arrival counters of the small-batch router, grid barriers of the single-token kernel) and a region anchored at the END of
 *     the buffer (fp32 accumulator and tickets of the fused combine; kernels clear what they used).  Hence: pass the
 *     buffer's true size as `workspace_bytes` on every call, use one workspace for one layer shape (D, F, E, K, G, S;
 *     any T <= T_max), and call bm_workspace_init again after a failed launch, after a device status fault
 *     (bm_device_status != 0) or before re-using the buffer for another shape.
 *   - Threads and devices.  Calls may be issued from several host threads and on several devices of one process
 *     (per-device facts are cached per device ordinal); two calls that share a workspace or routing arrays must be
 *     ordered by the caller.  bm_set_option and the bm_profile_* pair change process-global state and must not run
 *     concurrently with other calls.
 *   - `stream` is a cudaStream_t (0 = the legacy default stream).
 *   - Return value: BM_OK (0) or a negative bm_status, checked synchronously on the host before
 *     anything is enqueued.  T == 0 is BM_OK and a no-op.  Data-dependent faults (a group_map entry
 *     outside [0,G), a non-finite router logit) cannot be seen without a sync: kernels raise a bit in a
 *     device status word inside the workspace (read it with bm_device_status); the outputs are then
 *     unspecified but all indices written stay in range.
 *   - There is no CPU fallback: without a CUDA device of compute capability 10.0 every compute entry
 *     point returns BM_ERR_CUDA.
 */
#ifndef BM_H_
#define BM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef uint16_t bm_bf16;
typedef struct CUstream_st *bm_stream_t;

typedef enum bm_status {
    BM_OK = 0,
    BM_ERR_NULL = -1,      /* a required pointer is NULL */
    BM_ERR_SHAPE = -2,     /* K<1, K>E, K>BM_MAX_K, E>BM_MAX_E, G<1, G>BM_MAX_G, T<0, D%8, F%8, D<8, F<8, S<0, S>BM_MAX_S;
                              an unknown option name */
    BM_ERR_ALIGN = -3,     /* a device pointer is not 16-byte aligned */
    BM_ERR_WORKSPACE = -4, /* workspace_bytes < bm_workspace_bytes(...) */
    BM_ERR_CUDA = -5,      /* no sm_100 device, driver entry point missing, or a launch failed */
    BM_ERR_PATH = -6,      /* forced path cannot run this shape (bm_moe_forward_path) */
    BM_ERR_LIMIT = -7      /* sizes beyond the fixed scratch of bm_route_static */
} bm_status;

enum { BM_MAX_E = 512, BM_MAX_K = 16, BM_MAX_G = 512, BM_MAX_S = 16 };

/* bits of the device status word */
enum { BM_DEV_BAD_GROUP_MAP = 1, BM_DEV_NONFINITE_LOGIT = 2, BM_DEV_BAD_ROUTING = 4 };

/* execution path of bm_moe_forward_path */
enum {
    BM_PATH_AUTO = 0,    /* GEMV if T <= 2 and T*K <= G (a weight set expects at most ~1 row: single-token decode); else DECODE if
                            T <= 64, or T <= 192 (256 where a weight set D*F has >= 64 MB) and T*K <= 128*G (one chunk per
                            group), or T <= BM_DECODE_MAX_T and T*K <= 44*G (few rows per group); else PREFILL */
    BM_PATH_DECODE = 1,  /* weight-streaming, weights on the MMA M side (small M; HBM-bound)   */
    BM_PATH_PREFILL = 2, /* 128-token x 256-column tcgen05 tiles (large M; tensor-pipe-bound)  */
    BM_PATH_SIMT = 3,    /* plain CUDA-core kernels; a debugging cross-check, never picked by AUTO */
    BM_PATH_GEMV = 4     /* weight-streaming matrix-vector products on the CUDA cores (FFMA2), <= 8 rows of a set per
                            pass over its weights; W2 stage fused with the slot-order combine (deterministic)    */
};
enum { BM_DECODE_MAX_T = 320 };   /* default of option DECODE_MAX_T: AUTO never picks DECODE beyond it */

/*
 * Routing of one batch: the result of steps R1-R7.  A host struct of device
 * arrays, every array allocated by the caller at its maximum size.  A = offsets[G] <= T*K is the
 * number of (token, group) assignments after dedup.
 */
typedef struct bm_routing {
    int32_t T, E, K, G;   /* filled by bm_route (host values) */
    int32_t *expert_ids;  /* [T,K]  ranked top-K expert indices (rank 0 = largest logit; ties -> lower index) */
    int32_t *group_ids;   /* [T,K]  distinct groups of the token in first-occurrence (rank) order, -1 padded  */
    float *gate_w;        /* [T,K]  merged gate weights (softmax over the K selected logits, summed per group), 0 padded */
    int32_t *n_slots;     /* [T]    number of distinct groups, 1..K */
    int32_t *counts;      /* [G]    rows per group */
    int32_t *offsets;     /* [G+1]  exclusive scan of counts; offsets[G] = A */
    int32_t *row_token;   /* [T*K]  token of permuted row r (rows ordered by group, then token ascending); -1 for r >= A */
    int32_t *row_slot;    /* [T*K]  slot s of permuted row r; -1 for r >= A */
    int32_t *slot_row;    /* [T,K]  inverse permutation: row of (token, slot); -1 padded */
} bm_routing;

/* Bytes of scratch both calls need for shapes up to T_max tokens (independent of the data); 0 for arguments no call
 * accepts (negative sizes, S > BM_MAX_S).  HOST call. */
size_t bm_workspace_bytes(int T_max, int D, int F, int E, int K, int G, int S);

/* Zeroes the workspace (asynchronously on `stream`): required once after allocation, see "Workspace" above. */
int bm_workspace_init(void *workspace, size_t workspace_bytes, bm_stream_t stream);

/*
 * bm_route -- steps R1-R7: router logits in fp32 with the canonical summation order (A1), top-K with
 * lower-index tie-break (A4), softmax over the selected logits (A2), group remap (Eq. 2), dedup with
 * summed weights (A5, A6), per-group histogram, exclusive scan and the stable permutation (A7).
 * Cite: P:42 (gate, top-K), P:118-122 + P:247 (group map).
 *   x            [T,D]  bf16 tokens
 *   W_router     [E,D]  bf16
 *   router_bias  [E]    f32, added once after the reduction; NULL = none
 *   group_map    [E]    i32, values in [0,G)
 *   routing      HOST struct of device arrays (see bm_routing); T,E,K,G are written by this call
 * Every routing array is fully written (pads included).  Integer outputs are deterministic.
 */
int bm_route(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E,
             int K, const int32_t *group_map, int G, bm_routing *routing, void *workspace,
             size_t workspace_bytes, bm_stream_t stream);

/*
 * bm_route_partial -- partial brownout.  Cite: "partial-brownout delegates only
 * cold expert tokens to united experts based on a configurable threshold"; P:172 the original gate still
 * determines the activated experts; "the grouping map determines which united expert handles tokens
 * originally routed to each cold expert".  Which experts are cold is the caller's decision (A9: the
 * paper's threshold criterion lives in its reference [7]).
 *   cold_mask  [E] i32: non-zero = cold (served by united expert group_map[e]); zero = hot (keeps its own weights)
 * Weight sets are numbered  [0, G) = united experts,  G + e = original expert e, so the routing arrays range over
 * G + E sets: routing->G is set to G + E, counts holds G + E and offsets G + E + 1 entries (G + E <= BM_MAX_G), and
 * the workspace must be sized with bm_workspace_bytes(..., G + E, S).  The forward pass is bm_moe_forward on weights
 * stacked as [united (G) ; original (E) ; shared (S)]; sets that receive no row cost nothing.  All cold = full
 * brownout (same arrays as bm_route), all hot = zero brownout.  Everything else as bm_route.
 */
int bm_route_partial(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E,
                     int K, const int32_t *group_map, int G, const int32_t *cold_mask, bm_routing *routing,
                     void *workspace, size_t workspace_bytes, bm_stream_t stream);

/*
 * bm_route_static -- bm_route without a workspace, for callers that may not allocate device memory (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The scratch bm_route keeps in the workspace
 * (status word, arrival counters, permutation histograms, router logits / norms / candidate masks) lives in a
 * file-scope device array of BM_STATIC_ROUTE_BYTES = 2 MiB inside the library; every GPU that loads the library holds
 * those 2 MiB until the process exits.  The call allocates and frees nothing and calls no allocating library routine.
 *   - Arguments and results exactly as bm_route (same kernels, same bits); the caller still passes x, the router, the
 *     group map and the routing arrays.
 *   - Limit: T <= BM_STATIC_ROUTE_MAX_T = 8192 (any E, K, G the library accepts then fits the array); beyond it the
 *     call returns BM_ERR_LIMIT on the host, before anything is enqueued.
 *   - The array is shared by every call on the device and keeps the last call's contents.  Each call clears the part
 *     that must start at zero (its first 4096 bytes) on `stream` ahead of its kernels.  Calls that overlap on the GPU
 *     -- different streams without an ordering between them, or two threads -- RACE on the array: order them.
 *   - The first call on a device looks up the array's device address (cudaGetSymbolAddress): make one call, e.g. with
 *     T = 0, outside any stream capture.
 *   - bm_route_static_status copies the status word of the array (the BM_DEV_* bits the LAST bm_route_static call on
 *     this device raised) to *host_out (HOST) and SYNCHRONISES `stream`.
 */
enum { BM_STATIC_ROUTE_BYTES = 2 * 1024 * 1024, BM_STATIC_ROUTE_MAX_T = 8192 };
int bm_route_static(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
                    const int32_t *group_map, int G, bm_routing *routing, bm_stream_t stream);
int bm_route_static_status(int32_t *host_out, bm_stream_t stream);

/*
 * bm_unite_weights -- united-weight construction.  Cite: "The united expert is
 * initialized as the parameter average of member experts"; group map: P:118-122 (Eq. 2).
 *   out[u, i] = (1 / |G_u|) * sum_{e : group_map[e] == u} W[e, i],   members added in ascending e in fp32,
 *   rounded once to bf16; an empty group gives zeros.
 *   W    [E, n] bf16 (one expert matrix flattened: n = F*D), n % 8 == 0
 *   out  [G, n] bf16, overwritten.  Call it once per matrix kind (W1, W3, W2).
 */
int bm_unite_weights(const bm_bf16 *W, int E, size_t n, const int32_t *group_map, int G, bm_bf16 *out,
                     bm_stream_t stream);

/*
 * Calibration forward: the forward half of the reward evaluation of the grouping search
 * (P:127 routing frequency; Eq. 5-6; P:170 cosine similarity of expert outputs; "> 95%" of the
 * search time).  The four calls below are independent; all outputs are overwritten.
 *
 * bm_expert_histogram -- w[e] = number of (token, rank) pairs whose selected expert is e ("how often expert
 *   e is selected by the gating function on the calibration dataset").  expert_ids [T,K] i32 as bm_route wrote
 *   them; w [E] i32.  Exact.
 * bm_expert_outputs -- y[t, e, :] = FFN_e(x_t) for EVERY expert e and token t (the f_e(x) of Eq. 5), through the
 *   grouped tcgen05 GEMM kernels.  W1, W3 [E,F,D], W2 [E,D,F]; y is TOKEN-MAJOR, [T,E,D] bf16 (the E outputs of a token
 *   are neighbours in memory: that is what lets bm_cosine_gram and bm_group_mse stream at HBM rate); workspace of
 *   bm_expert_outputs_workspace_bytes(T, D, F, E) bytes (no initialisation needed).  E <= BM_MAX_G.
 * bm_cosine_gram -- gram[e,e'] = <Y_e, Y_e'> with Y_e = all outputs of expert e (T*D values), and
 *   cosine[e,e'] = gram[e,e'] / (|Y_e| |Y_e'|) (A19), fp32 accumulation on the tensor cores, per-CTA
 *   partial tiles summed in a fixed order.  Y [T,E,D] bf16 (token-major, as bm_expert_outputs writes it), D % 8 == 0,
 *   E <= 128; gram, cosine [E,E] f32 (cosine may be NULL); workspace >= bm_gram_workspace_bytes(E).
 * bm_group_mse -- Eq. 5: alpha_e = w_e / sum_{e' in G_r} w_e', t_r(x) = sum_{e in G_r} alpha_e f_e(x);
 *   MSE_r = mean over tokens of |U_r(x) - t_r(x)|^2 (Eq. 9's expectation); Eq. 6: beta_r = sum_{e in G_r} w_e with w
 *   normalised to sum 1, MSE_total = sum_r beta_r MSE_r (A20: a never-selected group takes uniform alpha
 *   and weight 0; an empty group has MSE 0).  Y [T,E,D] bf16 expert outputs, U [T,G,D] bf16 united-expert outputs (both token-major),
 *   w [E] i32, group_map [E] i32; mse [G] f32, mse_total [1] f32; workspace >= bm_mse_workspace_bytes(G).
 */
int bm_expert_histogram(const int32_t *expert_ids, int T, int K, int E, int32_t *w, bm_stream_t stream);
size_t bm_expert_outputs_workspace_bytes(int T, int D, int F, int E);
int bm_expert_outputs(const bm_bf16 *x, int T, int D, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int E,
                      int F, bm_bf16 *y, void *workspace, size_t workspace_bytes, bm_stream_t stream);
size_t bm_gram_workspace_bytes(int E);
int bm_cosine_gram(const bm_bf16 *Y, int E, int T, int D, float *gram, float *cosine, void *workspace,
                   size_t workspace_bytes, bm_stream_t stream);
size_t bm_mse_workspace_bytes(int G);
int bm_group_mse(const bm_bf16 *Y, const bm_bf16 *U, int T, int D, const int32_t *w, const int32_t *group_map, int E,
                 int G, float *mse, float *mse_total, void *workspace, size_t workspace_bytes, bm_stream_t stream);

/*
 * bm_moe_forward -- steps 9-13: out[t] = sum_s gate_w[t,s] * FFN_{group_ids[t,s]}(x_t) + sum_{j<S} FFN_{G+j}(x_t)
 * with FFN_u(x) = W2[u] . ( SiLU(W1[u] x) * (W3[u] x) )   (P:42 with united experts P:46; SwiGLU: A3).
 * bf16 operands, fp32 accumulation (tensor cores; CUDA-core FFMA2 on the matrix-vector path), the intermediate h
 * is rounded to bf16 (A12).  The gate-weighted sum is taken in fp32:
 *   - tensor-core paths (decode, prefill): the W2 GEMM's epilogue adds gw * y into an fp32 accumulator with
 *     reductions; on the prefill tiles (F >= 4096) the arrival that completes an output piece also rounds it to bf16
 *     inside the kernel (north_star kernel (4)), on the decode kernel a small finalize pass does.  fp32 addition is commutative, so the result is bit-deterministic when no token has more than two
 *     source rows (K + S <= 2, and no K split on the decode path); with more sources the order of the additions, hence
 *     the last bits before the bf16 rounding, may vary between calls.  bm_forward_info tells which case a call is in.
 *   - matrix-vector path and the two-pass prefill form (F < 4096 by default, or option FUSED_COMBINE = 0): slot order,
 *     bit-deterministic; the two-pass form rounds the per-row expert outputs y to bf16 before the sum.
 *   x        [T,D]      bf16
 *   routing  as produced by bm_route (or any arrays satisfying the same invariants), same T
 *   W1, W3   [G+S,F,D]  bf16 (united experts 0..G-1, then the S always-on shared experts, A11)
 *   W2       [G+S,D,F]  bf16
 *   out      [T,D]      bf16, overwritten
 * The path (matrix-vector / decode / prefill, see BM_PATH_AUTO) is picked from the host values T, K, G and S.
 */
int bm_moe_forward(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1,
                   const bm_bf16 *W3, const bm_bf16 *W2, int F, int S, bm_bf16 *out, void *workspace,
                   size_t workspace_bytes, bm_stream_t stream);

/*
 * bm_moe_layer -- bm_route followed by bm_moe_forward on device buffers, as one call: out and every routing array are
 * written exactly as by the two calls.  Having the whole step in one call lets the library run single-token decode
 * (T <= 2 with T*K <= G, the matrix-vector rule of BM_PATH_AUTO) as ONE persistent kernel -- router dots, selection,
 * W1/W3 stream, W2 stream + combine separated by two grid-wide barriers (cooperative launch) instead of three
 * dependent launches; every other shape takes the two calls' kernels.  Option LAYER_SMALL = 0 switches the single kernel off.
 * Small decode batches (T <= 64 with G <= T*K) also gain from the single call: their first weight sets are multiplied
 * while the routing kernels still run (every active set multiplies all T tokens there, so the work needs no routing;
 * options DC_SPEC_US / DC_SPEC_MIN_ROWS), which bm_moe_forward on its own cannot know to be worth while.
 * Arguments as in bm_route / bm_moe_forward (full brownout: no cold mask).
 */
int bm_moe_layer(const bm_bf16 *x, int T, int D, const bm_bf16 *W_router, const float *router_bias, int E, int K,
                 const int32_t *group_map, int G, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int F, int S,
                 bm_bf16 *out, bm_routing *routing, void *workspace, size_t workspace_bytes, bm_stream_t stream);

/*
 * Tensor parallelism over F (the paper scales with tensor parallelism).
 * SwiGLU is elementwise over the F hidden features, so with W1, W3 row-sharded and W2 column-sharded over N ranks
 *     FFN_u(x) = sum_r W2_r[u] . ( SiLU(W1_r[u] x) * (W3_r[u] x) ),     W1_r, W3_r [G+S, F/N, D],  W2_r [G+S, D, F/N]
 * and the layer output is the sum over ranks of the per-rank layer outputs (routing is replicated).
 * bm_moe_forward_f32 is bm_moe_forward on one rank's shard that leaves the fp32 sums in out_f32 [T,D] (no bf16
 * rounding); the caller all-reduces out_f32 over the ranks (NCCL, torch.distributed) and rounds once with
 * bm_round_bf16.  out_f32 is overwritten.  The SIMT cross-check path has no fp32 variant.
 * bm_round_bf16: out[i] = bf16(in[i]), round to nearest even, n % 8 == 0.
 */
int bm_moe_forward_f32(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1,
                       const bm_bf16 *W3, const bm_bf16 *W2, int F, int S, float *out_f32, void *workspace,
                       size_t workspace_bytes, bm_stream_t stream);
int bm_round_bf16(const float *in, size_t n, bm_bf16 *out, bm_stream_t stream);

/*
 * SLO-aware latency control (PAPER.md 4.5): host logic that decides how aggressively the runtime applies
 * united experts.  "When recent P90 latency exceeds the SLO, the threshold is multiplicatively reduced to lower
 * latency.  When latency falls below a warning line, the threshold is linearly increased to improve accuracy."
 * (P:259); threshold = 1.0 means no merging, threshold = 0 all cold-expert calls go to united experts.
 * The paper prints no constants and Eq. 10-11 only state the objective, so every constant is a caller-set field
 * (reading A21).  All pointers are HOST pointers; nothing here touches the GPU.
 *
 *   bm_salc_init     fills *c: threshold = 1 (zero brownout), empty latency window.  BM_ERR_SHAPE unless
 *                    slo > 0, 0 < warn_frac <= 1, 0 < decrease < 1, increase > 0, 1 <= window <= BM_SALC_MAX_WINDOW.
 *   bm_salc_observe  records one request latency (same unit as slo) in the sliding window of the last `window`
 *                    observations and applies one control step on the window's P90 (nearest-rank: the
 *                    ceil(0.9 n)-th smallest of the n latencies held):
 *                        P90 > slo              -> threshold *= decrease
 *                        P90 < warn_frac * slo  -> threshold  = min(1, threshold + increase)
 *                        otherwise              -> unchanged
 *                    Returns the new threshold (a negative bm_status as a double on a NULL / NaN argument).
 *   bm_salc_cold_mask  turns a threshold into the cold_mask of bm_route_partial: the n_cold = round((1 - threshold) E)
 *                    experts with the smallest routing frequency w[e] (bm_expert_histogram; ties -> lower index
 *                    colder) are cold.  The paper defines "cold" only in its ref. [7]; this rule is reading A17's
 *                    caller-supplied mask made concrete for the controller and is the one bench.py --config next uses.
 */
enum { BM_SALC_MAX_WINDOW = 256 };
typedef struct {
    double slo;          /* latency objective                                             */
    double warn_frac;    /* warning line as a fraction of slo                             */
    double decrease;     /* multiplicative factor applied above the SLO, in (0, 1)        */
    double increase;     /* additive step applied below the warning line                  */
    double threshold;    /* state: in [0, 1]                                              */
    int32_t window;      /* observations the P90 is taken over                            */
    int32_t count;       /* state: observations held (<= window)                          */
    int32_t head;        /* state: next slot of the ring                                  */
    double lat[BM_SALC_MAX_WINDOW];   /* state: ring of the last latencies                */
} bm_salc;
int bm_salc_init(bm_salc *c, double slo, double warn_frac, double decrease, double increase, int window);
double bm_salc_observe(bm_salc *c, double latency);
double bm_salc_p90(const bm_salc *c);    /* P90 of the window (0 when empty) */
int bm_salc_cold_mask(const int32_t *w /*HOST [E]*/, int E, double threshold, int32_t *cold_mask /*HOST [E]*/);

/*
 * bm_forward_info -- what bm_moe_forward will do for a batch of these host-side sizes, without running anything:
 *   *path           the BM_PATH_* that BM_PATH_AUTO resolves to (under the current options)
 *   *deterministic  1 if two calls on the same inputs give bit-identical `out` on that path, 0 if the order of
 *                   fp32 additions may vary (tensor-core paths with more than two source rows per output value)
 * Either pointer may be NULL.  HOST call.
 */
int bm_forward_info(int T, int K, int G, int S, int D, int F, int *path, int *deterministic);

/* Same as bm_moe_forward with the execution path forced (BM_PATH_*); used by tests and the bench to
 * exercise every path on any shape.  BM_ERR_PATH if the path cannot run the shape. */
int bm_moe_forward_path(const bm_bf16 *x, int T, int D, const bm_routing *routing, const bm_bf16 *W1,
                        const bm_bf16 *W3, const bm_bf16 *W2, int F, int S, bm_bf16 *out,
                        void *workspace, size_t workspace_bytes, bm_stream_t stream, int path);

/*
 * bm_moe_layer_host -- the whole layer for one batch held in HOST memory: copies x host->device,
 * runs bm_route + bm_moe_forward, copies out device->host and SYNCHRONISES `stream`.
 *   x_host    HOST [T,D] bf16 (pinned memory gives an asynchronous copy)
 *   out_host  HOST [T,D] bf16
 *   x_dev, out_dev   device staging buffers [T,D] bf16 owned by the caller
 * All other arguments as in bm_route / bm_moe_forward (weights, router and group map stay resident on
 * the device).  Batches of T >= 2 * HOST_CHUNK_T tokens (option; 0 = never) are processed in up to 16 equal token
 * chunks so that the copies of neighbouring chunks overlap the compute of the current one (two internal copy streams and
 * their events are created on first use, once per device -- the one place where the library owns CUDA objects).  By
 * default (HOST_CHUNK_T = -1) a chunk has about 2816 tokens where a token computes at least twice as long as it copies
 * (F * (K + S) >= 17400, e.g. Mixtral shapes: smaller chunks lose more tile efficiency than their copies hide) and 2048
 * elsewhere.  bm_host_chunks returns the number of chunks such a call takes and writes the first min(n, cap) chunk sizes
 * to `sizes` (HOST; no GPU needed).  `out` is the same either way; the routing arrays then hold each chunk's result in
 * the chunk's slice ([t0*K, (t0+tc)*K) of the [T,K] arrays, row indices relative to the chunk) and counts / offsets those
 * of the LAST chunk: call bm_route yourself when you need the whole batch's permutation.
 */
int bm_host_chunks(int T, int F, int K, int S, int *sizes, int cap);
int bm_moe_layer_host(const bm_bf16 *x_host, int T, int D, const bm_bf16 *W_router,
                      const float *router_bias, int E, int K, const int32_t *group_map, int G,
                      const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int F, int S,
                      bm_bf16 *out_host, bm_bf16 *x_dev, bm_bf16 *out_dev, bm_routing *routing,
                      void *workspace, size_t workspace_bytes, bm_stream_t stream);

/* Copies the device status word (OR of BM_DEV_* bits raised since the last call of this function) to
 * *host_out (HOST), clears it, and SYNCHRONISES `stream`. */
int bm_device_status(void *workspace, int32_t *host_out, bm_stream_t stream);

/*
 * Options: integer tuning and test switches, process-global.  Each starts at its default, or at the value of the
 * environment variable BM_<NAME> read ONCE when the library is first used; afterwards only bm_set_option changes it
 * (no call reads the environment).  BM_ERR_SHAPE for an unknown name.
 *   PDL (1)                 programmatic dependent launch between the kernels of a call
 *   FUSED_COMBINE (-1)      1 = combine fused into the W2 GEMM epilogue, 0 = separate pass (prefill tiles: bf16 y rows +
 *                           slot-order sum, deterministic; decode kernel: finalize pass); -1 = by shape: prefill tiles fused
 *                           from F = 4096 on, decode kernel never (its finalize pass measured faster)
 *   PF_PAIR (-1)            prefill tiles: 1 / 0 force CTA pairs (cta_group::2) on / off, -1 = by rows per group
 *   PF_GATHER (1)           0 = materialise gathered rows, 1 = gather inside GEMM1 on single-CTA tiles, 2 = also with pairs
 *   PF_G1_BC, PF_G2_BC, PF_G2_BW (-1)   prefill tiles: L2 bands of the item order -- chunk units per band in GEMM1 / GEMM2,
 *                           weight tiles per band in GEMM2; <= 0 = one band (chunk-fastest order, the default)
 *   PF_G1_HINTS, PF_G2_HINTS (-1)       L2 eviction hints of the prefill tiles' TMA loads: 10 * activations + weights with
 *                           0 = evict_first, 1 = normal, 2 = evict_last; -1 = default (21)
 *   DECODE_MAX_T (320), DECODE_MID_T (192), DECODE_ROWS (44), DECODE_MID_ROWS (128), GEMV_MAX_T (2), GEMV_ROWS (1)
 *                           thresholds of BM_PATH_AUTO
 *   DC_DENSE_MAX_T (64)     decode kernels: up to this many tokens (<= 64) every active set multiplies all T tokens (no gather)
 *   DC_PREFETCH_MB (48)     decode GEMM1: megabytes of W1 / W3 it asks L2 to fetch while it still waits for the routing; 0 = off
 *   GEMV_FUSE (1)           matrix-vector path: fuse the W2 stage with the combine
 *   DC_R1, DC_R2, DC_KS2, DC_RMAX, DC_KS_FORCE (0, 0, 1, 128, 0)   decode tiling overrides (rows per tile, K splits)
 *   DC_STAGES, PF_STAGES (12)   cap on the shared-memory ring depth
 *   DC_SPEC_US (12), DC_SPEC_MIN_ROWS (1)   bm_moe_layer, dense decode with G <= T*K: GEMM1 multiplies the leading weight sets
 *                           -- as many as stream from HBM in DC_SPEC_US microseconds -- before it waits for the routing
 *                           kernels (0 = off), provided T*K >= DC_SPEC_MIN_ROWS * G
 *   PF_SPEC (1)             bm_moe_layer, prefill tiles with S > 0: GEMM1 runs the shared experts' items before it waits for the
 *                           routing kernels (0 = off)
 *   PERM_CLUSTER (1)        permutation of 2048 < T*K <= 65536 items: 1 = one launch (a cluster of eight CTAs), 0 = three kernels
 *   LAYER_SMALL (1)         bm_moe_layer: 1 = one persistent kernel for T <= 2 (single-token decode), 0 = the separate kernels
 *   HOST_CHUNK_T (-1)       bm_moe_layer_host: tokens per pipelined chunk; 0 = one piece; -1 = by shape (2816 or 2048)
 *   ROUTER_FILTER (1)       T >= 512, E <= 256, K <= 8, E >= 4K + 8: tensor-core filter + canonical refinement of the
 *                           candidates; 0 = all E dots; 2 = the filter whenever the kernel supports the shape
 *   DC_KPACK (2)            decode kernels: k-blocks per ring stage
 *   COMBINE_WARPS (64), PERM_SMALL_WARPS (0), ROUTER_WE (0), ROUTER_TP_MIN_T (512), ROUTER_SPLIT_MAX_T (16)
 *                           shape thresholds of the small kernels
 */
int bm_set_option(const char *name, int value);
int bm_get_option(const char *name, int *value);

/* Number of kernel launches the library has enqueued in this process so far (a HOST counter;
 * bench.py reports its difference over the timed region as `gpu_launches`). */
long long bm_launch_count(void);

/*
 * Per-kernel device timing for the roofline report (bench.py).  bm_profile_enable(kernel, max_records) makes every
 * later bm_route / bm_moe_forward call bracket the launches of `kernel` (BM_KERNEL_*; BM_KERNEL_ALL = every kind)
 * with a pair of CUDA events on the call's stream, up to max_records pairs, and switches programmatic dependent
 * launch off (events between overlapped kernels would time nothing meaningful); kernel = 0 switches it off and
 * frees the events.  bm_profile_read_kinds SYNCHRONISES on the recorded events, writes the summed elapsed
 * milliseconds and the number of launches per kind to HOST arrays of BM_KERNEL_ALL entries (index = kind) and
 * restarts the recording; bm_profile_read gives the totals over all recorded kinds.  Process-global, not thread-safe.
 */
enum {
    BM_KERNEL_NONE = 0, BM_KERNEL_ROUTER = 1, BM_KERNEL_PERMUTE = 2, BM_KERNEL_PREP = 3,
    BM_KERNEL_GEMM1 = 4, BM_KERNEL_GEMM2 = 5, BM_KERNEL_FINALIZE = 6, BM_KERNEL_ALL = 7
};
int bm_profile_enable(int kernel, int max_records);
int bm_profile_read(float *total_ms, int *n_records);
int bm_profile_read_kinds(float *ms_by_kind, int *n_by_kind);

/* Human-readable name of a bm_status code.  Never NULL. */
const char *bm_status_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* BM_H_ */
