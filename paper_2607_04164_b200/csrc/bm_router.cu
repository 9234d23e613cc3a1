// bm_router.cu -- steps R1-R5 in one kernel: canonical fp32 router logits, top-K with lower-index
// tie-break, softmax over the K selected logits, group remap, dedup with summed gate weights.
//
// Cite: PAPER.md:42 (gating function, top-K routing, gating score g_i), Eq. 2 and
// PAPER.md:247 (group map g: expert -> united group), readings A1, A2, A4, A5, A6.
//
// Canonical dot product (A1).  A warp owns one (token, expert) dot product: lane l accumulates the
// 8-element chunks c = l, l+32, l+64, ... (chunk c = elements 8c..8c+7, one 128-bit load) in ascending
// order with __fmaf_rn from 0, then the five-step xor butterfly (16, 8, 4, 2, 1) adds the 32 partials.
// That is exactly the association tree the oracle spells out, so the logits are bit-identical and the
// integer outputs (expert_ids, group_ids, n_slots) are too.  No fast-math, no FTZ in this file.
//
// Work split inside a CTA of 8 warps: WT token-slices x WE expert-slices (WT*WE = 8).  Each warp
// keeps a register tile acc[TOK][ET] (TOK tokens x ET experts) and walks D once per expert tile.
// Small T (decode): TOK = 1, warps split the experts, one CTA per token -> latency-bound, ~2 us.
// Large T (prefill): TOK = 4, ET = 8, warps split the tokens -> each W_router chunk feeds 32 FMAs.
#include <algorithm>

#include "bm_common.cuh"
#include "bm_permute.cuh"
#include "bm_ptx.cuh"
#include "bm_router.cuh"

namespace bm {

namespace {

constexpr int kWarps = 8;

template <int TOK, int ET>
__global__ void __launch_bounds__(kWarps * 32)
router_kernel(const bm_bf16 *__restrict__ x, int T, int D, const bm_bf16 *__restrict__ Wr,
              const float *__restrict__ bias, int E, int K, GroupMap gm,
              int WT, int WE, int32_t *__restrict__ expert_ids, int32_t *__restrict__ group_ids,
              float *__restrict__ gate_w, int32_t *__restrict__ n_slots, int32_t *__restrict__ status) {
    extern __shared__ float s_logits[];   // [TB][E], TB = WT * TOK
    grid_dep_wait();      // x may come from a predecessor; the routing arrays may still be read by one
    grid_dep_launch();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int TB = WT * TOK;
    const int t_block = blockIdx.x * TB;
    const int tw = warp % WT, ew = warp / WT;
    const int n_etiles = (E + ET - 1) / ET;

    // ---- R1: logits ---------------------------------------------------------------------
    const bm_bf16 *xrow[TOK];
#pragma unroll
    for (int i = 0; i < TOK; ++i) {
        int t = t_block + tw * TOK + i;
        xrow[i] = x + (size_t)(t < T ? t : T - 1) * D;     // clamp: rows past T are computed and dropped
    }
    for (int et = ew; et < n_etiles; et += WE) {
        const int e0 = et * ET;
        const bm_bf16 *wrow[ET];
#pragma unroll
        for (int j = 0; j < ET; ++j) wrow[j] = Wr + (size_t)(e0 + j < E ? e0 + j : E - 1) * D;
        float acc[TOK][ET];
#pragma unroll
        for (int i = 0; i < TOK; ++i)
#pragma unroll
            for (int j = 0; j < ET; ++j) acc[i][j] = 0.0f;

#pragma unroll 2
        for (int k = lane * 8; k < D; k += 256) {
            uint4 xv[TOK];
#pragma unroll
            for (int i = 0; i < TOK; ++i) xv[i] = __ldg(reinterpret_cast<const uint4 *>(xrow[i] + k));
#pragma unroll
            for (int j = 0; j < ET; ++j) {
                const uint4 wv = __ldg(reinterpret_cast<const uint4 *>(wrow[j] + k));
                const float w0 = bf16_lo(wv.x), w1 = bf16_hi(wv.x), w2 = bf16_lo(wv.y), w3 = bf16_hi(wv.y);
                const float w4 = bf16_lo(wv.z), w5 = bf16_hi(wv.z), w6 = bf16_lo(wv.w), w7 = bf16_hi(wv.w);
#pragma unroll
                for (int i = 0; i < TOK; ++i) {
                    float p = acc[i][j];                    // ascending element order inside the chunk
                    p = __fmaf_rn(bf16_lo(xv[i].x), w0, p);
                    p = __fmaf_rn(bf16_hi(xv[i].x), w1, p);
                    p = __fmaf_rn(bf16_lo(xv[i].y), w2, p);
                    p = __fmaf_rn(bf16_hi(xv[i].y), w3, p);
                    p = __fmaf_rn(bf16_lo(xv[i].z), w4, p);
                    p = __fmaf_rn(bf16_hi(xv[i].z), w5, p);
                    p = __fmaf_rn(bf16_lo(xv[i].w), w6, p);
                    p = __fmaf_rn(bf16_hi(xv[i].w), w7, p);
                    acc[i][j] = p;
                }
            }
        }
#pragma unroll
        for (int i = 0; i < TOK; ++i)
#pragma unroll
            for (int j = 0; j < ET; ++j) {
                float p = acc[i][j];
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) p = __fadd_rn(p, __shfl_xor_sync(kFullMask, p, o));
                if (lane == 0 && e0 + j < E) {
                    if (bias) p = __fadd_rn(p, bias[e0 + j]);
                    s_logits[(tw * TOK + i) * E + e0 + j] = p;
                }
            }
    }
    __syncthreads();

    // ---- R2-R5: one warp per token --------------------------------------------------------
    for (int tl = warp; tl < TB; tl += kWarps) {
        const int t = t_block + tl;
        if (t >= T) break;
        select_and_write(s_logits + tl * E, t, lane, E, K, gm, expert_ids, group_ids, gate_w, n_slots, status);
    }
}

// -------------------------------------------------------------------------------------------------
// Latency shape with the experts of a token spread over 32 warps and, for E > 64, over CTAs (T <= 16, E > 8).
// CTA (es, t) computes the logits of 32 * ET experts of token t -- a warp owns ET dot products in the canonical order -- and parks them
// in a global scratch row.  The CTA that completes a token (arrival counter) runs R2-R5 for it; the CTA that
// completes the batch runs the whole permutation R6-R8 when it fits one CTA (T*K <= 2048), which saves the
// launch of the permutation kernel.  Counters live in the zero-once head of the workspace and are put back
// to zero by the CTA that consumed them.  Writers fence before they signal (the threadFenceReduction
// pattern); the consumers read the other CTAs' results with ld.global.cg.
// One token on one CTA (router_kernel) streams all of W_router through a single SM: 7 us at E = 60, D = 2048.
// -------------------------------------------------------------------------------------------------
constexpr int kTinyPermItems = 128;    // up to this many (token, slot) items the fused permutation needs no scans
constexpr int kSplitWarps = 32;        // a CTA of 32 warps x ET experts: E <= 64 needs one CTA per token and no arrival counter

template <int ET>
__global__ void __launch_bounds__(kSplitWarps * 32)
router_split_kernel(const bm_bf16 *__restrict__ x, int T, int D, const bm_bf16 *__restrict__ Wr,
                    const float *__restrict__ bias, int E, int K, GroupMap gm, int ES, float *__restrict__ logits_ws,
                    int fuse_permute, int per_warp, bm_routing r, int32_t *__restrict__ status) {
    extern __shared__ int rs_dyn[];       // float [E] for the select, then the permutation's scratch
    __shared__ int s_flag, s_total;
    grid_dep_wait();      // x may come from a predecessor; the routing arrays may still be read by one
    grid_dep_launch();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int t = blockIdx.y;
    const int e0 = (blockIdx.x * kSplitWarps + warp) * ET;

    // ---- R1: ET logits per warp ---------------------------------------------------------------
    if (e0 < E) {
        const bm_bf16 *xrow = x + (size_t)t * D;
        const bm_bf16 *wrow[ET];
#pragma unroll
        for (int j = 0; j < ET; ++j) wrow[j] = Wr + (size_t)(e0 + j < E ? e0 + j : E - 1) * D;
        float acc[ET];
#pragma unroll
        for (int j = 0; j < ET; ++j) acc[j] = 0.0f;
#pragma unroll 4
        for (int k = lane * 8; k < D; k += 256) {
            const uint4 xv = __ldg(reinterpret_cast<const uint4 *>(xrow + k));
            uint4 wv[ET];
#pragma unroll
            for (int j = 0; j < ET; ++j) wv[j] = __ldg(reinterpret_cast<const uint4 *>(wrow[j] + k));
#pragma unroll
            for (int j = 0; j < ET; ++j) {
                float p = acc[j];                    // ascending element order inside the chunk
                p = __fmaf_rn(bf16_lo(xv.x), bf16_lo(wv[j].x), p);
                p = __fmaf_rn(bf16_hi(xv.x), bf16_hi(wv[j].x), p);
                p = __fmaf_rn(bf16_lo(xv.y), bf16_lo(wv[j].y), p);
                p = __fmaf_rn(bf16_hi(xv.y), bf16_hi(wv[j].y), p);
                p = __fmaf_rn(bf16_lo(xv.z), bf16_lo(wv[j].z), p);
                p = __fmaf_rn(bf16_hi(xv.z), bf16_hi(wv[j].z), p);
                p = __fmaf_rn(bf16_lo(xv.w), bf16_lo(wv[j].w), p);
                p = __fmaf_rn(bf16_hi(xv.w), bf16_hi(wv[j].w), p);
                acc[j] = p;
            }
        }
#pragma unroll
        for (int j = 0; j < ET; ++j) {
            float p = acc[j];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) p = __fadd_rn(p, __shfl_xor_sync(kFullMask, p, o));
            if (lane == 0 && e0 + j < E) {
                if (bias) p = __fadd_rn(p, bias[e0 + j]);
                if (ES > 1) __stcg(logits_ws + (size_t)t * E + e0 + j, p);
                else reinterpret_cast<float *>(rs_dyn)[e0 + j] = p;      // one CTA per token: the logits stay on chip
            }
        }
        if (lane == 0 && ES > 1) __threadfence();
    }
    __syncthreads();
    if (ES > 1) {                          // several CTAs share the token: the last one to arrive goes on
        if (threadIdx.x == 0) s_flag = atomicAdd(status + kStatusTokCnt + t, 1) == ES - 1;   // (the writers fenced above)
        __syncthreads();
        if (!s_flag) return;
    }

    // ---- R2-R5: this CTA completed token t -------------------------------------------------------
    if (warp == 0) {
        float *s_l = reinterpret_cast<float *>(rs_dyn);
        if (ES > 1) {
            __threadfence();
            for (int e = lane; e < E; e += 32) s_l[e] = __ldcg(logits_ws + (size_t)t * E + e);
            __syncwarp();
        }
        select_and_write(s_l, t, lane, E, K, gm, r.expert_ids, r.group_ids, r.gate_w, r.n_slots, status);
        if (lane == 0 && ES > 1) status[kStatusTokCnt + t] = 0;
        __threadfence();
    }
    if (!fuse_permute) return;
    __syncthreads();
    if (T > 1) {                           // the CTA that completes the batch goes on
        if (threadIdx.x == 0) {            // (warp 0 fenced its routing rows above)
            s_flag = atomicAdd(status + kStatusDone, 1) == T - 1;
            if (s_flag) status[kStatusDone] = 0;
        }
        __syncthreads();
        if (!s_flag) return;
    }

    // ---- R6-R8: this CTA completed the batch ---------------------------------------------------------
    __threadfence();
    const int items = T * K;
    if (items <= kTinyPermItems) {
        // at most 128 (token, slot) items: no histograms or scans -- every thread counts the keys below / equal to
        // its group from the keys in shared memory; item i's row = #(keys < key_i) + #(j < i with key_j = key_i),
        // the stable order of R7
        __shared__ int s_keys[kTinyPermItems];
        if (threadIdx.x < kTinyPermItems) s_keys[threadIdx.x] = (int)threadIdx.x < items ? __ldcg(r.group_ids + threadIdx.x) : -1;
        __syncthreads();
        const int G = r.G;
        for (int u = threadIdx.x; u <= G; u += blockDim.x) {
            int less = 0, eq = 0;
            for (int i = 0; i < items; ++i) {
                const int k = s_keys[i];
                less += (k >= 0 && k < u) ? 1 : 0;
                eq += (k == u) ? 1 : 0;
            }
            if (u < G) r.counts[u] = eq;
            r.offsets[u] = less;
            if (u == G) status[1] = less;
        }
        if ((int)threadIdx.x < items) {
            const int i = threadIdx.x, k = s_keys[i];
            int A = 0, row = 0;
            for (int j = 0; j < items; ++j) {
                const int kj = s_keys[j];
                A += kj >= 0 ? 1 : 0;
                row += (kj >= 0 && (kj < k || (kj == k && j < i))) ? 1 : 0;
            }
            if (k >= 0) {
                r.row_token[row] = i / K;
                r.row_slot[row] = i % K;
                r.slot_row[i] = row;
            } else {
                r.slot_row[i] = -1;
            }
            if (i >= A) { r.row_token[i] = -1; r.row_slot[i] = -1; }
        }
        return;
    }
    permute_block_small(r.group_ids, T, K, r.G, per_warp, r.counts, r.offsets, r.row_token, r.row_slot, r.slot_row,
                        status, rs_dyn, &s_total);
}

// -------------------------------------------------------------------------------------------------
// Throughput shape (T >= BM_ROUTER_TP_MIN_T): the same canonical dot products, operands staged through
// shared memory by TMA.  Persistent CTAs walk token blocks of TB = WT*8 tokens; per pass a block meets
// EB = WE*8 experts; compute warp (tw, ew) keeps the 8 x 8 register tile acc[token][expert] of its slice --
// lane l still owns partial l of every dot product and walks its chunks l, l+32, ... in ascending order, so
// the association tree is unchanged.  D is walked in slabs of 256 elements (one 16-byte chunk per lane and
// row).  A producer warp (one elected lane) fetches a slab with two tensor copies -- the x tile [TB, 256]
// and the W_router tile [EB, 256], rows past T or E zero-filled and never stored -- into a 4-stage ring
// guarded by full/empty mbarriers, three slabs ahead of the multiply and across passes and blocks, so
// neither the HBM read of x nor the L2 read of W_router is on the critical path and the compute warps
// never meet a CTA-wide barrier inside a pass.  (The first version copied row by row with per-lane
// cp.async.bulk: the copy instruction takes its operands from uniform registers, so the compiler serialises
// the lanes -- 16% of all executed instructions and a quarter of the stall samples in ncu.)
// The multiply is FFMA2 (two fp32 FMAs per instruction; the FMA pipe issues it at the rate of a scalar FFMA).
// E > EB takes ceil(E/EB) passes over the same tokens.
// -------------------------------------------------------------------------------------------------
constexpr int kTpStages = 4;
constexpr int kSlab = 256;                    // elements per slab row = 512 bytes
constexpr int kTpTok = 8;                     // tokens of a compute warp's register tile
constexpr int kTpComputeWarps = 8;
constexpr int kTpSelectWarps = 3;
constexpr int kTpThreads = (kTpComputeWarps + 1 + kTpSelectWarps) * 32;      // + the producer warp + the select warps

// Sum of the 32 lane partials of each of this lane's 32 accumulators: the xor butterfly (16, 8, 4, 2, 1)
// of reading A1, evaluated for all 32 accumulators at once.  At the step with offset o every lane hands
// over the half of its values whose index bit o differs from its own lane bit o, so a step costs n/2
// shuffles instead of n; each surviving value is p_l + p_{l xor o} exactly as in the per-accumulator
// butterfly (fp32 addition is commutative, so both partners of a pair would have computed the same
// bits).  On return lane l holds in v[0] the finished sum of accumulator index l.
__device__ __forceinline__ void butterfly32(float (&v)[32], int lane) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        const bool up = (lane & o) != 0;
#pragma unroll
        for (int a = 0; a < o; ++a) {
            const float keep = up ? v[a + o] : v[a];
            const float send = up ? v[a] : v[a + o];
            v[a] = __fadd_rn(keep, __shfl_xor_sync(kFullMask, send, o));
        }
    }
}

// Two fp32 fused multiply-adds in one instruction (FFMA2): d0 = fma(x, w0, d0), d1 = fma(x, w1, d1), each
// rounded to nearest exactly like __fmaf_rn, so the canonical order (A1) is untouched -- the two halves are
// the accumulators of two neighbouring experts.  ptxas folds the duplicated x into the scalar-broadcast
// operand form (FFMA2 Rd, Rx.F32, Rw.F32x2, Rd.F32x2), so no instruction is spent on it.
__device__ __forceinline__ void fma2(float &d0, float &d1, float x, float w0, float w1) {
    uint64_t a, b, c;
    asm("mov.b64 %0, {%1, %1};" : "=l"(a) : "f"(x));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(w0), "f"(w1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(d0), "f"(d1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(c));
}
// bf16 -> fp32 of the low half through PRMT, so that the unpack stays on the ALU pipe (the compiler turns a
// plain shift into IMAD.U32 half of the time, which competes with FFMA2 for the FMA pipe)
__device__ __forceinline__ float bf16_lo_alu(uint32_t u) { return __uint_as_float(__byte_perm(u, 0u, 0x1044)); }

// Wait of a helper role (producer lane, select warps): backs off between polls so that it does not take
// issue slots from the compute warps; bounded in time like ptx::mbar_wait (a protocol bug traps instead of hanging).
template <unsigned NS>
__device__ __forceinline__ void mbar_wait_sleep(uint64_t *bar, uint32_t parity) {
    uint32_t spins = 0;
    uint64_t t0 = 0;
    while (!ptx::mbar_try_wait(bar, parity)) {
        __nanosleep(NS);
        if ((++spins & 0xfffu) == 0) {
            const uint64_t now = ptx::globaltimer_ns();
            if (t0 == 0) t0 = now;
            else if (now - t0 > ptx::kWaitTimeoutNs) __trap();
        }
    }
}

__global__ void __launch_bounds__(kTpThreads, 1)
router_tp_kernel(const __grid_constant__ CUtensorMap tm_x,      // x [T, D], box 256 x TB
                 const __grid_constant__ CUtensorMap tm_w,      // W_router [E, D], box 256 x EB
                 int T, int D, const float *__restrict__ bias, int E, int K, GroupMap gm,
                 int WT, int WE, int n_blocks, int32_t *__restrict__ expert_ids, int32_t *__restrict__ group_ids,
                 float *__restrict__ gate_w, int32_t *__restrict__ n_slots, int32_t *__restrict__ status) {
    extern __shared__ __align__(128) uint8_t tp_smem[];
    const int TB = WT * kTpTok, EB = WE * 8;
    const int rows = TB + EB;
    const uint32_t stage_bytes = (uint32_t)rows * (kSlab * 2);
    uint64_t *full = reinterpret_cast<uint64_t *>(tp_smem + kTpStages * stage_bytes);
    uint64_t *empty = full + kTpStages;
    uint64_t *lfull = empty + kTpStages;                              // logits of a block parked / consumed
    uint64_t *lempty = lfull + 2;
    float *s_logits = reinterpret_cast<float *>(lempty + 2);          // [2][TB][E]
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int n_slabs = (D + kSlab - 1) / kSlab;
    const int n_pass = (E + EB - 1) / EB;

    if (tid == 0) {
        for (int i = 0; i < kTpStages; ++i) {
            ptx::mbar_init(&full[i], 1);
            ptx::mbar_init(&empty[i], kTpComputeWarps);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(&lfull[i], kTpComputeWarps);
            ptx::mbar_init(&lempty[i], kTpSelectWarps);
        }
        ptx::fence_barrier_init();
        ptx::prefetch_tmap(&tm_x);
        ptx::prefetch_tmap(&tm_w);
    }
    __syncthreads();
    grid_dep_wait();      // x may come from a predecessor; the routing arrays may still be read by one
    grid_dep_launch();

    if (warp == kTpComputeWarps) {
        // ---- producer: one lane, two tensor copies per slab -----------------------------------------
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x)
                for (int pass = 0; pass < n_pass; ++pass)
                    for (int slab = 0; slab < n_slabs; ++slab) {
                        mbar_wait_sleep<64>(&empty[stage], phase ^ 1);    // slab held before released by every compute warp
                        uint8_t *st = tp_smem + (size_t)stage * stage_bytes;
                        ptx::mbar_arrive_expect_tx(&full[stage], stage_bytes);
                        ptx::tma_load_2d(st, &tm_x, &full[stage], slab * kSlab, blk * TB, ptx::kEvictNormal);
                        ptx::tma_load_2d(st + (size_t)TB * (kSlab * 2), &tm_w, &full[stage], slab * kSlab, pass * EB,
                                         ptx::kEvictLast);
                        if (++stage == kTpStages) { stage = 0; phase ^= 1; }
                    }
        }
        return;
    }
    if (warp > kTpComputeWarps) {
        // ---- select warps: R2-R5 of block i while the compute warps multiply block i + 1 -----------------
        const int sw = warp - kTpComputeWarps - 1;
        int it = 0;
        for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x, ++it) {
            const int buf = it & 1;
            mbar_wait_sleep<400>(&lfull[buf], (it >> 1) & 1);     // a block takes microseconds: poll rarely
            const float *lg = s_logits + (size_t)buf * TB * E;
            // the CTA's last block: the compute warps have nothing left to multiply and take a share (below)
            const int stride = blk + (int)gridDim.x >= n_blocks ? kTpSelectWarps + kTpComputeWarps : kTpSelectWarps;
            for (int tl = sw; tl < TB; tl += stride) {
                const int t = blk * TB + tl;
                if (t >= T) break;
                select_and_write(lg + tl * E, t, lane, E, K, gm, expert_ids, group_ids, gate_w, n_slots, status);
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&lempty[buf]);
        }
        return;
    }

    const int tw = warp % WT, ew = warp / WT;
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x, ++it) {
        const int buf = it & 1;
        float *lg = s_logits + (size_t)buf * TB * E;
        for (int pass = 0; pass < n_pass; ++pass) {
            float acc[kTpTok * 8];              // index a = token * 8 + expert
#pragma unroll
            for (int a = 0; a < kTpTok * 8; ++a) acc[a] = 0.0f;
            for (int slab = 0; slab < n_slabs; ++slab) {
                ptx::mbar_wait(&full[stage], phase);
                const uint8_t *st = tp_smem + (size_t)stage * stage_bytes;
                if (slab * kSlab + lane * 8 < D) {
                    float xf[kTpTok][8];
#pragma unroll
                    for (int i = 0; i < kTpTok; ++i) {
                        const uint4 v = *reinterpret_cast<const uint4 *>(st + (tw * kTpTok + i) * (kSlab * 2) + lane * 16);
                        xf[i][0] = bf16_lo_alu(v.x); xf[i][1] = bf16_hi(v.x); xf[i][2] = bf16_lo_alu(v.y); xf[i][3] = bf16_hi(v.y);
                        xf[i][4] = bf16_lo_alu(v.z); xf[i][5] = bf16_hi(v.z); xf[i][6] = bf16_lo_alu(v.w); xf[i][7] = bf16_hi(v.w);
                    }
#pragma unroll
                    for (int j = 0; j < 8; j += 2) {        // experts j, j + 1 share one FFMA2
                        const uint8_t *wp = st + (TB + ew * 8 + j) * (kSlab * 2) + lane * 16;
                        const uint4 wa = *reinterpret_cast<const uint4 *>(wp);
                        const uint4 wb = *reinterpret_cast<const uint4 *>(wp + kSlab * 2);
                        const float a0 = bf16_lo_alu(wa.x), a1 = bf16_hi(wa.x), a2 = bf16_lo_alu(wa.y), a3 = bf16_hi(wa.y);
                        const float a4 = bf16_lo_alu(wa.z), a5 = bf16_hi(wa.z), a6 = bf16_lo_alu(wa.w), a7 = bf16_hi(wa.w);
                        const float b0 = bf16_lo_alu(wb.x), b1 = bf16_hi(wb.x), b2 = bf16_lo_alu(wb.y), b3 = bf16_hi(wb.y);
                        const float b4 = bf16_lo_alu(wb.z), b5 = bf16_hi(wb.z), b6 = bf16_lo_alu(wb.w), b7 = bf16_hi(wb.w);
#pragma unroll
                        for (int i = 0; i < kTpTok; ++i) {
                            float &p = acc[i * 8 + j], &q = acc[i * 8 + j + 1];   // ascending element order inside the chunk
                            fma2(p, q, xf[i][0], a0, b0);
                            fma2(p, q, xf[i][1], a1, b1);
                            fma2(p, q, xf[i][2], a2, b2);
                            fma2(p, q, xf[i][3], a3, b3);
                            fma2(p, q, xf[i][4], a4, b4);
                            fma2(p, q, xf[i][5], a5, b5);
                            fma2(p, q, xf[i][6], a6, b6);
                            fma2(p, q, xf[i][7], a7, b7);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(&empty[stage]);
                if (++stage == kTpStages) { stage = 0; phase ^= 1; }
            }
            // end of a pass: per group of 4 tokens, lane l finishes accumulator l = (token l/8, expert l%8),
            // adds the bias, parks it
            const int e = pass * EB + ew * 8 + (lane & 7);
            if (pass == 0) ptx::mbar_wait(&lempty[buf], ((it >> 1) & 1) ^ 1);   // the block parked here two blocks ago is consumed
#pragma unroll
            for (int h = 0; h < kTpTok / 4; ++h) {
                butterfly32(*reinterpret_cast<float(*)[32]>(&acc[h * 32]), lane);
                if (e < E) {
                    float v = acc[h * 32];
                    if (bias) v = __fadd_rn(v, bias[e]);
                    lg[(tw * kTpTok + h * 4 + (lane >> 3)) * E + e] = v;
                }
            }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&lfull[buf]);      // this warp's share of the block's logits is parked
    }
    if (it > 0) {
        // last block of this CTA: help the select warps (tokens kTpSelectWarps + warp, + 11, ...)
        const int li = it - 1, buf = li & 1;
        const int blk = blockIdx.x + li * (int)gridDim.x;
        ptx::mbar_wait(&lfull[buf], (li >> 1) & 1);
        const float *lg = s_logits + (size_t)buf * TB * E;
        for (int tl = kTpSelectWarps + warp; tl < TB; tl += kTpSelectWarps + kTpComputeWarps) {
            const int t = blk * TB + tl;
            if (t >= T) break;
            select_and_write(lg + tl * E, t, lane, E, K, gm, expert_ids, group_ids, gate_w, n_slots, status);
        }
    }
}

cudaError_t launch_tp(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                      GroupMap gm, const bm_routing &r, int32_t *status, cudaStream_t stream) {
    const int n_etiles = (E + 7) / 8;
    int WE = 1;
    while (WE < n_etiles && WE < kTpComputeWarps) WE *= 2;
    if (opt(OPT_ROUTER_WE) > 0) WE = opt(OPT_ROUTER_WE);
    const int WT = kTpComputeWarps / WE;
    const int TB = WT * kTpTok, EB = WE * 8;
    const size_t smem = (size_t)kTpStages * (TB + EB) * (kSlab * 2) + (2 * kTpStages + 4) * sizeof(uint64_t) +
                        2 * (size_t)TB * E * sizeof(float);
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(router_tp_kernel), smem); ea != cudaSuccess) return ea;
    CUtensorMap m_x, m_w;
    if (!make_map_2d_plain(&m_x, x, (uint64_t)T, (uint64_t)D, (uint32_t)TB, kSlab) ||
        !make_map_2d_plain(&m_w, Wr, (uint64_t)E, (uint64_t)D, (uint32_t)EB, kSlab))
        return cudaErrorInvalidValue;
    const int n_blocks = (T + TB - 1) / TB;
    const int grid = n_blocks < num_sms() ? n_blocks : num_sms();
    return launch_kernel(router_tp_kernel, dim3(grid), dim3(kTpThreads), smem, stream, m_x, m_w, T, D, bias, E, K,
                         gm, WT, WE, n_blocks, r.expert_ids, r.group_ids, r.gate_w, r.n_slots, status);
}

// -------------------------------------------------------------------------------------------------
// Filter + refine (T >= 512, E <= 256, K <= 8).  The canonical fp32 dot products decide the routing bit for bit, but
// only the K largest of a token's E logits matter, so:
//   1. row_norm_kernel    |x_t| and |Wr_e| (one warp per row)
//   2. router_filter_kernel   approximate logits a[t,e] = x_t . Wr_e on the tensor cores (tcgen05, bf16 products are exact,
//      fp32 accumulation in the hardware's order), tau_t = the K-th largest a[t,.] + bias, and the candidate set
//          C_t = { e : a[t,e] + bias_e >= tau_t - 2 beta[t,e] },   beta[t,e] = kappa |x_t| |Wr_e|
//      where beta bounds |a[t,e] - canonical logit|: both are fp32 evaluations of the same sum of exact products, each
//      within (number of additions) * 2^-23 * sum_i |x_i w_i| <= D 2^-23 |x_t| |Wr_e| of the real value (Cauchy-Schwarz);
//      kappa = 2 D 2^-23 + 2^-18 leaves a factor of two and room for the bias addition.
//      Every e outside C_t has canonical logit < tau_t - beta <= the canonical logit of each of the K experts with the
//      largest a[t,.], so it cannot be among the canonical top-K: the refinement over C_t alone is exact, ties included.
//      A token with a non-finite a[t,.] keeps all E experts.
//   3. router_refine_kernel   canonical dots (A1) for the candidates only -- K + ~0.1 of E = 60 -- then R2-R5 as everywhere.
// The FMA work falls from T E D to ~T K D (T = 4096, E = 60: 51 -> ~15 us for the whole routing step).
// -------------------------------------------------------------------------------------------------
constexpr int kFlThreads = 192;
constexpr int kFlMaxE = 256, kFlMaxK = 8;
constexpr int kFlXTile = 128 * 128;                 // bytes: 128 token rows x 64 bf16

__global__ void __launch_bounds__(256)
row_norm_kernel(const bm_bf16 *__restrict__ x, int T, const bm_bf16 *__restrict__ Wr, int E, int D, float *__restrict__ norms) {
    grid_dep_wait();
    grid_dep_launch();
    const int lane = threadIdx.x & 31;
    const int warps = (gridDim.x * blockDim.x) >> 5;
    for (int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; r < T + E; r += warps) {
        const uint4 *row = reinterpret_cast<const uint4 *>(r < T ? x + (size_t)r * D : Wr + (size_t)(r - T) * D);
        float s = 0.0f;
        for (int i = lane; i < D / 8; i += 32) {
            const uint4 v = __ldg(row + i);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) { const float a = bf16_lo(w[k]), b = bf16_hi(w[k]); s = fmaf(a, a, s); s = fmaf(b, b, s); }
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(kFullMask, s, o);
        if (lane == 0) norms[r] = sqrtf(s) * 1.0001f;          // rounded up a little: it feeds an upper bound
    }
}

__global__ void __launch_bounds__(kFlThreads, 1)
router_filter_kernel(const __grid_constant__ CUtensorMap tm_x,      // x [T, D], box 128 rows x 64, 128B swizzle
                     const __grid_constant__ CUtensorMap tm_w,      // W_router [E, D], box N rows x 64 (rows >= E: zeros)
                     int T, int D, int E, int K, int N, int BR, int n_blocks, int n_stages, const float *__restrict__ bias,
                     const float *__restrict__ norms, float kappa, int mask_words, uint32_t *__restrict__ mask) {
    extern __shared__ uint8_t fl_smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(fl_smem_raw) + 1023) & ~uintptr_t(1023));
    // a stage = two k-blocks (the single-thread issue loop costs ~0.3 us per barrier turn whatever the tiles hold), each
    // an x tile of BR token rows (the slot keeps 128 rows: the M = 128 MMA reads that much; rows >= BR are never used)
    // and a W_router tile of N rows
    const uint32_t x_bytes = (uint32_t)BR * 128u, w_bytes = (uint32_t)N * 128u;
    const uint32_t x_slot = (x_bytes + 1023u) & ~1023u;
    const uint32_t half_bytes = x_slot + ((w_bytes + 1023u) & ~1023u);
    const uint32_t stage_bytes = 2u * half_bytes;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)n_stages * stage_bytes + kFlXTile);   // (+ the MMA's 16 KB read window)
    uint64_t *empty = full + 16;
    uint64_t *tfull = empty + 16;        // [2]
    uint64_t *tempty = tfull + 2;        // [2]
    uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(tempty + 2);
    float *s_wn = reinterpret_cast<float *>(tmem_ptr + 2);          // [kFlMaxE] |Wr_e|
    float *s_bias = s_wn + kFlMaxE;                                 // [kFlMaxE]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nkb = ((D + 63) / 64 + 1) / 2;          // stages per block (columns past D arrive as zeros)

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tm_x);
        ptx::prefetch_tmap(&tm_w);
        for (int i = 0; i < n_stages; ++i) { ptx::mbar_init(&full[i], 1); ptx::mbar_init(&empty[i], 1); }
        for (int i = 0; i < 2; ++i) { ptx::mbar_init(&tfull[i], 1); ptx::mbar_init(&tempty[i], 4); }
        ptx::fence_barrier_init();
    }
    if (warp == 1) ptx::tmem_alloc(tmem_ptr, 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    // Only the epilogue needs row_norm_kernel's result.  x and W_router are ready for the producer as soon as this grid runs:
    // row_norm_kernel let it start only after its own grid-dependency wait had returned, i.e. after everything before this
    // call had completed -- so the main loop runs beside the norm pass instead of behind it.
    if (warp >= 2) grid_dep_wait();
    if (threadIdx.x == 0) grid_dep_launch();

    if (warp == 0) {
        int stage = 0;
        uint32_t phase = 0;
        for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x)
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(&empty[stage], phase ^ 1);
                if (ptx::elect_one()) {
                    uint8_t *st = smem + (size_t)stage * stage_bytes;
                    ptx::mbar_arrive_expect_tx(&full[stage], 2u * (x_bytes + w_bytes));
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        ptx::tma_load_2d(st + h * half_bytes, &tm_x, &full[stage], (2 * kb + h) * 64, blk * BR, ptx::kEvictNormal);
                        ptx::tma_load_2d(st + h * half_bytes + x_slot, &tm_w, &full[stage], (2 * kb + h) * 64, 0, ptx::kEvictLast);
                    }
                }
                __syncwarp();
                if (++stage == n_stages) { stage = 0; phase ^= 1; }
            }
    } else if (warp == 1) {
        const uint32_t idesc = ptx::make_idesc_bf16(128, N);
        const uint32_t a_lo0 = ptx::smem_desc_lo(ptx::smem_u32(smem));
        int stage = 0, acc = 0;
        uint32_t phase = 0, acc_phase = 0;
        for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
            ptx::mbar_wait(&tempty[acc], acc_phase ^ 1);
            ptx::tc_fence_after();
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(&full[stage], phase);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t a_lo = a_lo0 + stage * (stage_bytes >> 4) + h * (half_bytes >> 4);
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            ptx::mma_bf16_ss(tmem_base + acc * 256, ptx::smem_desc(a_lo + 2 * k),
                                             ptx::smem_desc(a_lo + (x_slot >> 4) + 2 * k), idesc, (kb | h | k) ? 1u : 0u);
                    }
                    ptx::mma_commit(&empty[stage]);
                    if (kb == nkb - 1) ptx::mma_commit(&tfull[acc]);
                }
                __syncwarp();
                if (++stage == n_stages) { stage = 0; phase ^= 1; }
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    } else {
        // epilogue: thread = token row of the block (TMEM lane); pass 1 finds tau (K-th largest of a + bias), pass 2 marks
        const int q = warp & 3;
        const int epi_tid = (warp - 2) * 32 + lane;
        for (int e = epi_tid; e < kFlMaxE; e += 128) {
            s_wn[e] = e < E ? norms[T + e] : 0.0f;
            s_bias[e] = (bias && e < E) ? bias[e] : 0.0f;
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
            const int row = q * 32 + lane;
            const int t = row < BR ? blk * BR + row : T;       // rows >= BR of the accumulator hold nothing
            const float xn = t < T ? norms[t] : 0.0f;
            ptx::mbar_wait(&tfull[acc], acc_phase);
            ptx::tc_fence_after();
            if (q * 32 >= BR) {                                // warp-uniform: just hand the accumulator back
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(&tempty[acc]);
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
                continue;
            }
            const uint32_t t_addr = tmem_base + acc * 256 + ((uint32_t)(q * 32) << 16);
            float top[kFlMaxK];
#pragma unroll
            for (int i = 0; i < kFlMaxK; ++i) top[i] = -INFINITY;
            bool finite = true;
            for (int c = 0; c < N; c += 16) {
                uint32_t v[16];
                ptx::tmem_ld_x16(t_addr + c, v);
                ptx::tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    if (c + i < E) {
                        float a = __uint_as_float(v[i]) + s_bias[c + i];
                        if (!(fabsf(a) <= 3.0e38f)) finite = false;
                        // insert into the descending top-K list (registers, fully unrolled)
#pragma unroll
                        for (int j = 0; j < kFlMaxK; ++j) {
                            const float hi = fmaxf(top[j], a);
                            a = fminf(top[j], a);
                            top[j] = hi;
                        }
                    }
                }
            }
            float tau = top[0];
#pragma unroll
            for (int j = 1; j < kFlMaxK; ++j) if (j < K) tau = top[j];
            const float slack = 2.0f * kappa * xn;
            for (int w = 0; w < mask_words; ++w) {
                uint32_t v[32];
                uint32_t bits = 0;
                if (w * 32 < N) {
                    ptx::tmem_ld_x16(t_addr + w * 32, *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
                    if (w * 32 + 16 < N) ptx::tmem_ld_x16(t_addr + w * 32 + 16, *reinterpret_cast<uint32_t(*)[16]>(&v[16]));
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        const int e = w * 32 + i;
                        if (e < E && (i < 16 || w * 32 + 16 < N)) {
                            const float a = __uint_as_float(v[i]) + s_bias[e];
                            if (!finite || a >= tau - slack * s_wn[e]) bits |= 1u << i;
                        }
                    }
                }
                if (t < T) mask[(size_t)t * mask_words + w] = bits;
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&tempty[acc]);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, 512);
    }
}

// NB canonical dot products (A1) of one token against candidates ce[0..NB): lane l owns the 8-element chunks l, l + 32, ...
// in ascending order with fmaf from 0, then the xor butterfly, then the bias -- bit for bit what router_kernel does.
template <int NB>
__device__ __forceinline__ void refine_dots(const bm_bf16 *__restrict__ xrow, const bm_bf16 *__restrict__ Wr,
                                            const float *__restrict__ bias, int D, const int (&ce)[4], float *l, int lane) {
    const bm_bf16 *wrow[NB];
    float acc[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) { wrow[j] = Wr + (size_t)ce[j] * D; acc[j] = 0.0f; }
#pragma unroll 4
    for (int k = lane * 8; k < D; k += 256) {
        const uint4 xv = __ldg(reinterpret_cast<const uint4 *>(xrow + k));
        uint4 wv[NB];
#pragma unroll
        for (int j = 0; j < NB; ++j) wv[j] = __ldg(reinterpret_cast<const uint4 *>(wrow[j] + k));
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            float p = acc[j];                    // ascending element order inside the chunk
            p = __fmaf_rn(bf16_lo(xv.x), bf16_lo(wv[j].x), p);
            p = __fmaf_rn(bf16_hi(xv.x), bf16_hi(wv[j].x), p);
            p = __fmaf_rn(bf16_lo(xv.y), bf16_lo(wv[j].y), p);
            p = __fmaf_rn(bf16_hi(xv.y), bf16_hi(wv[j].y), p);
            p = __fmaf_rn(bf16_lo(xv.z), bf16_lo(wv[j].z), p);
            p = __fmaf_rn(bf16_hi(xv.z), bf16_hi(wv[j].z), p);
            p = __fmaf_rn(bf16_lo(xv.w), bf16_lo(wv[j].w), p);
            p = __fmaf_rn(bf16_hi(xv.w), bf16_hi(wv[j].w), p);
            acc[j] = p;
        }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
        float p = acc[j];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) p = __fadd_rn(p, __shfl_xor_sync(kFullMask, p, o));
        if (lane == 0) {
            if (bias) p = __fadd_rn(p, bias[ce[j]]);
            l[ce[j]] = p;
        }
    }
}

// canonical dot products (A1) of the candidates only, then R2-R5; one warp per token, up to four candidates at a time
__global__ void __launch_bounds__(kWarps * 32)
router_refine_kernel(const bm_bf16 *__restrict__ x, int T, int D, const bm_bf16 *__restrict__ Wr,
                     const float *__restrict__ bias, int E, int K, GroupMap gm, const uint32_t *__restrict__ mask,
                     int mask_words, int32_t *__restrict__ expert_ids, int32_t *__restrict__ group_ids,
                     float *__restrict__ gate_w, int32_t *__restrict__ n_slots, int32_t *__restrict__ status) {
    extern __shared__ float s_rl[];       // [kWarps][E]
    // (never the first kernel of a call: its successor may be resident early -- it waits for this grid itself; see
    //  gemm_kernel's speculative start)
    grid_dep_launch();
    grid_dep_wait();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *l = s_rl + (size_t)warp * E;
    const int n_warps = gridDim.x * kWarps;
    for (int t = blockIdx.x * kWarps + warp; t < T; t += n_warps) {
        // experts outside the candidate set: a finite value below every real logit, never selected (the set holds >= K)
        for (int e = lane; e < E; e += 32) l[e] = -3.0e38f;
        __syncwarp();
        const bm_bf16 *xrow = x + (size_t)t * D;
        for (int w = 0; w < mask_words; ++w) {
            uint32_t bits = mask[(size_t)t * mask_words + w];
            if (w == mask_words - 1 && (E & 31)) bits &= (1u << (E & 31)) - 1u;
            while (bits) {
                const int nb = min(__popc(bits), 4);
                int ce[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    ce[j] = w * 32 + (bits ? __ffs(bits) - 1 : 0);
                    if (j < nb) bits &= bits - 1;
                }
                if (nb == 4) refine_dots<4>(xrow, Wr, bias, D, ce, l, lane);
                else if (nb == 3) refine_dots<3>(xrow, Wr, bias, D, ce, l, lane);
                else if (nb == 2) refine_dots<2>(xrow, Wr, bias, D, ce, l, lane);
                else refine_dots<1>(xrow, Wr, bias, D, ce, l, lane);
            }
        }
        __syncwarp();
        select_and_write(l, t, lane, E, K, gm, expert_ids, group_ids, gate_w, n_slots, status);
        __syncwarp();
    }
}

cudaError_t launch_filter_router(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                                 GroupMap gm, const bm_routing &r, int32_t *status, float *scratch, cudaStream_t stream) {
    const int sms = num_sms();
    float *norms = scratch;                                              // [T + E]
    const int mask_words = (E + 31) / 32;
    uint32_t *mask = reinterpret_cast<uint32_t *>(scratch + (((size_t)T + E + 3) & ~(size_t)3));     // [T][mask_words]
    cudaError_t e = launch_kernel(row_norm_kernel, dim3(std::min((T + E + 7) / 8, sms * 8)), dim3(256), 0, stream, x, T, Wr, E, D, norms);
    if (e != cudaSuccess) return e;
    const int N = std::max(16, (E + 15) & ~15);
    // token rows per CTA block: as many blocks as SMs when the batch allows it (the kernel streams x once: HBM / latency bound)
    const int BR = T >= 128 * sms ? 128 : (T >= 64 * sms ? 64 : 32);
    const size_t stage_bytes = 2 * ((((size_t)BR * 128 + 1023) & ~(size_t)1023) + (((size_t)N * 128 + 1023) & ~(size_t)1023));
    int n_stages = (int)((184 * 1024) / stage_bytes);
    n_stages = n_stages > 12 ? 12 : n_stages;
    const size_t smem = 1024 + (size_t)n_stages * stage_bytes + kFlXTile + 36 * 8 + 16 + 2 * kFlMaxE * sizeof(float);
    if ((e = ensure_dyn_smem(reinterpret_cast<const void *>(router_filter_kernel), smem)) != cudaSuccess) return e;
    CUtensorMap m_x, m_w;
    if (!make_map_2d_sw128(&m_x, x, (uint64_t)T, (uint64_t)D, (uint32_t)BR) || !make_map_2d_sw128(&m_w, Wr, (uint64_t)E, (uint64_t)D, (uint32_t)N))
        return cudaErrorInvalidValue;
    const int n_blocks = (T + BR - 1) / BR;
    const float kappa = 2.0f * (float)D * 1.1920929e-7f + 3.8146973e-6f;     // 2 D 2^-23 + 2^-18
    e = launch_kernel(router_filter_kernel, dim3(std::min(n_blocks, sms)), dim3(kFlThreads), smem, stream, m_x, m_w, T, D, E, K, N,
                      BR, n_blocks, n_stages, bias, (const float *)norms, kappa, mask_words, mask);
    if (e != cudaSuccess) return e;
    const size_t smem_r = (size_t)kWarps * E * sizeof(float);
    return launch_kernel(router_refine_kernel, dim3(std::min((T + kWarps - 1) / kWarps, sms * 8)), dim3(kWarps * 32), smem_r, stream,
                         x, T, D, Wr, bias, E, K, gm, (const uint32_t *)mask, mask_words, r.expert_ids, r.group_ids, r.gate_w,
                         r.n_slots, status);
}

template <int TOK, int ET>
cudaError_t launch_cfg(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                       GroupMap gm, int WT, int WE, const bm_routing &r, int32_t *status,
                       cudaStream_t stream) {
    const int TB = WT * TOK;
    const size_t smem = (size_t)TB * E * sizeof(float);
    auto kern = router_kernel<TOK, ET>;
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(kern), smem); ea != cudaSuccess) return ea;
    const int grid = (T + TB - 1) / TB;
    return launch_kernel(kern, dim3(grid), dim3(kWarps * 32), smem, stream, x, T, D, Wr, bias, E, K, gm, WT, WE,
                         r.expert_ids, r.group_ids, r.gate_w, r.n_slots, status);
}

}  // namespace

cudaError_t launch_router(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E,
                          int K, GroupMap gm, const bm_routing &r, int32_t *status, float *route_logits,
                          bool *fused_permute, cudaStream_t stream) {
    *fused_permute = false;
    if (T >= opt(OPT_ROUTER_TP_MIN_T)) {
        // throughput shapes: tensor-core filter + canonical refinement of the candidates when the shape allows it,
        // else all E canonical dots with the operands staged through shared memory
        // (worth it only when the candidates are few among many: E = 8, top-2 at T = 8192 measured 98 us against 54 us)
        const int fl = opt(OPT_ROUTER_FILTER);
        if (fl != 0 && E <= kFlMaxE && K <= kFlMaxK && K < E && (fl == 2 || E >= 4 * K + 8))
            return launch_filter_router(x, T, D, Wr, bias, E, K, gm, r, status, route_logits, stream);
        return launch_tp(x, T, D, Wr, bias, E, K, gm, r, status, stream);
    }
    // (measured: 2 us faster than router + permutation kernels at T = 1, even at T = 16, slower from T = 64 on:
    // more CTAs and two rounds of arrival counters)
    if (E > 8 && T <= opt(OPT_ROUTER_SPLIT_MAX_T)) {
        // latency shape, experts spread over CTAs; the last CTA also permutes when one CTA can
        constexpr int ET = 2;
        const int ES = (E + kSplitWarps * ET - 1) / (kSplitWarps * ET);
        const bool fuse = (long long)T * K <= kPermSmallItems;
        size_t smem = (size_t)E * sizeof(float);
        if (fuse) smem = std::max(smem, (size_t)(kSplitWarps * r.G + r.G + 512) * sizeof(int));
        if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(router_split_kernel<ET>), smem); ea != cudaSuccess) return ea;
        int per_warp = (int)(((long long)T * K + kSplitWarps - 1) / kSplitWarps);
        per_warp = (per_warp + 31) / 32 * 32;
        *fused_permute = fuse;
        return launch_kernel(router_split_kernel<ET>, dim3(ES, T), dim3(kSplitWarps * 32), smem, stream, x, T, D, Wr, bias, E, K,
                             gm, ES, route_logits, fuse ? 1 : 0, per_warp, r, status);
    }
    // latency shape: one token per warp pass, warps split the experts
    if (E <= 8) {
        int WE = 1;
        while (WE * 2 <= E && WE < kWarps) WE *= 2;
        return launch_cfg<1, 1>(x, T, D, Wr, bias, E, K, gm, kWarps / WE, WE, r, status, stream);
    }
    int tiles = (E + 7) / 8, WE = 1;
    while (WE * 2 <= tiles && WE < kWarps) WE *= 2;
    return launch_cfg<1, 8>(x, T, D, Wr, bias, E, K, gm, kWarps / WE, WE, r, status, stream);
}

}  // namespace bm
