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
#include "bm_common.cuh"

namespace bm {

namespace {

constexpr int kWarps = 8;

template <int TOK, int ET>
__global__ void __launch_bounds__(kWarps * 32)
router_kernel(const bm_bf16 *__restrict__ x, int T, int D, const bm_bf16 *__restrict__ Wr,
              const float *__restrict__ bias, int E, int K, const int32_t *__restrict__ gmap, int G,
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
        const float *l = s_logits + tl * E;
        unsigned taken = 0;                 // bit i: candidate e = lane + 32*i already selected (E <= 512)
        int sel_e[BM_MAX_K];
        float sel_l[BM_MAX_K];
        bool nonfinite = false;
#pragma unroll
        for (int i = 0; i < BM_MAX_K; ++i) {
            if (i < K) {
                // lane-local best: ascending e with a strict '>' keeps the lower index on ties
                float bv = -INFINITY;
                int bi = 0x7fffffff;
                for (int c = 0, e = lane; e < E; ++c, e += 32) {
                    if (taken & (1u << c)) continue;
                    float v = l[e];
                    if (!(fabsf(v) <= 3.402823466e38f)) nonfinite = true;
                    if (v != v) v = -INFINITY;            // NaN: unspecified result, keep indices valid
                    if (bi == 0x7fffffff || v > bv) { bv = v; bi = e; }
                }
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) {
                    const float ov = __shfl_xor_sync(kFullMask, bv, o);
                    const int oi = __shfl_xor_sync(kFullMask, bi, o);
                    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
                }
                if ((bi & 31) == lane) taken |= 1u << (bi >> 5);
                sel_e[i] = bi;
                sel_l[i] = l[bi];
            }
        }
        if (lane == 0) {
            // R3: softmax over the selected logits, sum in rank order
            float w[BM_MAX_K];
            const float m = sel_l[0];
            float sum = 0.0f;
#pragma unroll
            for (int i = 0; i < BM_MAX_K; ++i)
                if (i < K) {
                    w[i] = expf(__fsub_rn(sel_l[i], m));
                    sum = __fadd_rn(sum, w[i]);
                }
            // R4 + R5: remap and dedup in rank order; first occurrence keeps the slot
            int gid[BM_MAX_K];
            float gw[BM_MAX_K];
            int n = 0;
            bool bad_map = false;
#pragma unroll
            for (int i = 0; i < BM_MAX_K; ++i)
                if (i < K) {
                    const float wi = __fdiv_rn(w[i], sum);
                    int u = gmap[sel_e[i]];
                    if (u < 0 || u >= G) { bad_map = true; u = u < 0 ? 0 : G - 1; }
                    int s = n;                                     // index of the slot holding u, else n
#pragma unroll
                    for (int q = BM_MAX_K - 1; q >= 0; --q)
                        if (q < n && gid[q] == u) s = q;
                    if (s < n) {
#pragma unroll
                        for (int q = 0; q < BM_MAX_K; ++q)
                            if (q == s) gw[q] = __fadd_rn(gw[q], wi);
                    } else {
#pragma unroll
                        for (int q = 0; q < BM_MAX_K; ++q)
                            if (q == n) { gid[q] = u; gw[q] = wi; }
                        n++;
                    }
                }
            const size_t base = (size_t)t * K;
#pragma unroll
            for (int i = 0; i < BM_MAX_K; ++i)
                if (i < K) {
                    expert_ids[base + i] = sel_e[i];
                    group_ids[base + i] = i < n ? gid[i] : -1;
                    gate_w[base + i] = i < n ? gw[i] : 0.0f;
                }
            n_slots[t] = n;
            if (bad_map) atomicOr(status, BM_DEV_BAD_GROUP_MAP);
        }
        if (nonfinite) atomicOr(status, BM_DEV_NONFINITE_LOGIT);
    }
}

template <int TOK, int ET>
cudaError_t launch_cfg(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                       const int32_t *gmap, int G, int WT, int WE, const bm_routing &r, int32_t *status,
                       cudaStream_t stream) {
    const int TB = WT * TOK;
    const size_t smem = (size_t)TB * E * sizeof(float);
    auto kern = router_kernel<TOK, ET>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int grid = (T + TB - 1) / TB;
    return launch_kernel(kern, dim3(grid), dim3(kWarps * 32), smem, stream, x, T, D, Wr, bias, E, K, gmap, G, WT, WE,
                         r.expert_ids, r.group_ids, r.gate_w, r.n_slots, status);
}

}  // namespace

cudaError_t launch_router(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E,
                          int K, const int32_t *gmap, int G, const bm_routing &r, int32_t *status,
                          cudaStream_t stream) {
    if (T >= 2048) {
        // throughput shape: warps split tokens, 4 tokens x 8 experts per register tile
        return launch_cfg<4, 8>(x, T, D, Wr, bias, E, K, gmap, G, /*WT=*/kWarps, /*WE=*/1, r, status, stream);
    }
    // latency shape: one token per warp pass, warps split the experts
    if (E <= 8) {
        int WE = 1;
        while (WE * 2 <= E && WE < kWarps) WE *= 2;
        return launch_cfg<1, 1>(x, T, D, Wr, bias, E, K, gmap, G, kWarps / WE, WE, r, status, stream);
    }
    int tiles = (E + 7) / 8, WE = 1;
    while (WE * 2 <= tiles && WE < kWarps) WE *= 2;
    return launch_cfg<1, 8>(x, T, D, Wr, bias, E, K, gmap, G, kWarps / WE, WE, r, status, stream);
}

}  // namespace bm
