// bm_router.cuh -- R2-R5 for one token (top-K with lower-index tie-break, softmax over the selected logits, group
// remap, dedup with summed gate weights), shared by the router kernels (bm_router.cu) and the single-kernel layer for
// one or two tokens (bm_gemv.cu).  Cite: PAPER.md:42, PAPER.md:118-122 (Eq. 2); A2, A4, A5, A6.
#pragma once

#include "bm_common.cuh"

namespace bm {

// R2-R5 for one token, executed by one full warp: `l` = its E logits in shared memory.
// Rank i of the selection lives in lane i (K <= BM_MAX_K = 16 <= 32), so softmax, remap and dedup are
// lane-parallel; only the two rank-ordered fp32 sums (softmax denominator, merged gate weights) are
// sequential, as a chain of K shuffles.
__device__ __forceinline__ void select_and_write(const float *l, int t, int lane, int E, int K,
                                                 GroupMap gm,
                                                 int32_t *__restrict__ expert_ids, int32_t *__restrict__ group_ids,
                                                 float *__restrict__ gate_w, int32_t *__restrict__ n_slots,
                                                 int32_t *__restrict__ status) {
    // ---- R2: K rounds of warp arg-max; ties -> lower index --------------------------------------
    // A round is two warp reductions (redux.sync): the maximum of an order-preserving integer image of the
    // lane-local best values, then the minimum expert index among the lanes that hold that maximum.
    unsigned taken = 0;                 // bit c: candidate e = lane + 32*c already selected (E <= 512)
    int my_e = 0;                       // lane i < K: expert of rank i
    float my_l = 0.0f;                  //             and its logit
    bool nonfinite = false;
    for (int i = 0; i < K; ++i) {
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
        // monotone map float -> uint32 (a < b  <=>  key(a) < key(b)); -0 is first folded onto +0 so that the
        // two compare equal as they do under '=='; a lane without candidates gets key 0, below every float
        const uint32_t u = __float_as_uint(__fadd_rn(bv, 0.0f));
        uint32_t key = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
        if (bi == 0x7fffffff) key = 0u;
        const uint32_t kmax = __reduce_max_sync(kFullMask, key);
        const int win = __reduce_min_sync(kFullMask, (key == kmax) ? bi : 0x7fffffff);
        if ((win & 31) == lane) taken |= 1u << (win >> 5);
        if (lane == i) { my_e = win; my_l = l[win]; }
    }
    const bool active = lane < K;
    // ---- R3: softmax over the selected logits, denominator summed in rank order -------------------
    const float m = __shfl_sync(kFullMask, my_l, 0);
    const float w = active ? expf(__fsub_rn(my_l, m)) : 0.0f;
    float sum = 0.0f;
    for (int i = 0; i < K; ++i) sum = __fadd_rn(sum, __shfl_sync(kFullMask, w, i));
    const float wi = active ? __fdiv_rn(w, sum) : 0.0f;
    // ---- R4: remap ---------------------------------------------------------------------------------
    int u = -1 - lane;                  // inactive lanes: distinct negative keys, never matched
    bool bad_map = false;
    if (active) {
        u = gm.gmap[my_e];
        if (u < 0 || u >= gm.G) { bad_map = true; u = u < 0 ? 0 : gm.G - 1; }
        if (gm.cold && gm.cold[my_e] == 0) u = gm.G + my_e;        // partial brownout: a hot expert keeps its own set
    }
    // ---- R5: dedup in rank order; the first occurrence keeps the slot, weights added in rank order -----
    const unsigned peers = __match_any_sync(kFullMask, u);            // lanes (ranks) mapped to the same group
    const bool first = active && (__ffs(peers) - 1 == lane);
    const unsigned firsts = __ballot_sync(kFullMask, first);
    const int n = __popc(firsts);
    const int slot = __popc(firsts & ((1u << lane) - 1u));
    float gw = wi;
    for (int j = 1; j < K; ++j) {
        const float wj = __shfl_sync(kFullMask, wi, j);
        if (first && j > lane && ((peers >> j) & 1u)) gw = __fadd_rn(gw, wj);
    }
    const size_t base = (size_t)t * K;
    if (active) {
        expert_ids[base + lane] = my_e;
        if (lane >= n) { group_ids[base + lane] = -1; gate_w[base + lane] = 0.0f; }
    }
    if (first) { group_ids[base + slot] = u; gate_w[base + slot] = gw; }
    if (lane == 0) n_slots[t] = n;
    if (__any_sync(kFullMask, bad_map) && lane == 0) atomicOr(status, BM_DEV_BAD_GROUP_MAP);
    if (__any_sync(kFullMask, nonfinite) && lane == 0) atomicOr(status, BM_DEV_NONFINITE_LOGIT);
}

}  // namespace bm
