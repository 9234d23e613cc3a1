// bm_permute.cuh -- device-side building blocks of steps R6-R8 (histogram, exclusive scan, stable permutation),
// shared by the permutation kernels (bm_permute.cu) and the small-batch router, whose last CTA runs the whole
// permutation in place of a separate launch (bm_router.cu).  See bm_permute.cu for the algorithm.
// group_ids is read with ld.global.cg: in the fused router the ids were written by other CTAs of the same grid.
#pragma once

#include "bm_common.cuh"

namespace bm {

constexpr int kPermWarps = 8;
constexpr int kPermItemsPerWarp = kPermItemsPerBlock / kPermWarps;   // 64

// Count the items of this warp's slice into whist_w[0..G) (shared memory, zeroed by the caller).
__device__ __forceinline__ void warp_histogram(const int32_t *__restrict__ group_ids, long long items,
                                               long long first, int *whist_w, int lane, int per_warp = kPermItemsPerWarp) {
    for (int r = 0; r < per_warp && first + r < items; r += 32) {      // warp-uniform bound
        const long long i = first + r + lane;
        const int key = (i < items) ? __ldcg(group_ids + i) : -1;
        const unsigned peers = __match_any_sync(kFullMask, key);
        if (key >= 0 && lane == __ffs(peers) - 1) whist_w[key] += __popc(peers);
        __syncwarp();
    }
}

// Replay the walk with running bases wbase_w[0..G) (shared memory) and emit the permutation.
__device__ __forceinline__ void warp_permute(const int32_t *__restrict__ group_ids, long long items,
                                             long long first, int K, int *wbase_w, int lane, int A,
                                             int32_t *__restrict__ row_token, int32_t *__restrict__ row_slot,
                                             int32_t *__restrict__ slot_row, int per_warp = kPermItemsPerWarp) {
    for (int r = 0; r < per_warp && first + r < items; r += 32) {      // warp-uniform bound
        const long long i = first + r + lane;
        const int key = (i < items) ? __ldcg(group_ids + i) : -1;
        const unsigned peers = __match_any_sync(kFullMask, key);
        if (i < items) {
            if (key >= 0) {
                const int row = wbase_w[key] + __popc(peers & ((1u << lane) - 1u));
                row_token[row] = (int32_t)(i / K);
                row_slot[row] = (int32_t)(i % K);
                slot_row[i] = row;
            } else {
                slot_row[i] = -1;
            }
            if (i >= A) {                       // rows past A stay -1 (A <= items)
                row_token[i] = -1;
                row_slot[i] = -1;
            }
        }
        __syncwarp();
        if (key >= 0 && lane == __ffs(peers) - 1) wbase_w[key] += __popc(peers);
        __syncwarp();
    }
}

// Block-wide exclusive scan of v[0..n) (n <= 512) in shared memory; returns the total in *total.
// Exclusive scan of v[0..n) (n <= 512, shared memory) in place; *total = sum.  Warp 0 does it: lane l owns the 16
// consecutive slots 16l..16l+15 (serial prefix), the lane totals are scanned with shuffles.  Ends with a barrier.
__device__ __forceinline__ void block_exclusive_scan(int *v, int n, int *tmp, int *total) {
    (void)tmp;
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        int loc[16];
        int sum = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int idx = lane * 16 + i;
            const int x = idx < n ? v[idx] : 0;
            loc[i] = sum;
            sum += x;
        }
        int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(kFullMask, inc, o);
            if (lane >= o) inc += y;
        }
        const int base = inc - sum;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int idx = lane * 16 + i;
            if (idx < n) v[idx] = base + loc[i];
        }
        if (lane == 31) *total = inc;
    }
    __syncthreads();
}

// The whole permutation of T*K <= kPermSmallItems items by one CTA of kPermWarps warps (all of its threads call
// this): per-warp histograms -> exclusive scans -> replay.  s_mem: (nw*G + G + 512) ints of shared memory.
__device__ __forceinline__ void permute_block_small(const int32_t *__restrict__ group_ids, int T, int K, int G, int per_warp,
                                                    int32_t *__restrict__ counts, int32_t *__restrict__ offsets,
                                                    int32_t *__restrict__ row_token, int32_t *__restrict__ row_slot,
                                                    int32_t *__restrict__ slot_row, int32_t *__restrict__ status,
                                                    int *s_mem, int *s_total) {
    const int nw = blockDim.x >> 5;
    int *whist = s_mem;                  // [nw][G]
    int *gsum = whist + nw * G;          // [G] -> offsets
    int *tmp = gsum + G;                 // [512]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long items = (long long)T * K;
    for (int i = threadIdx.x; i < nw * G; i += blockDim.x) whist[i] = 0;
    __syncthreads();
    warp_histogram(group_ids, items, (long long)warp * per_warp, whist + warp * G, lane, per_warp);
    __syncthreads();
    for (int u = threadIdx.x; u < G; u += blockDim.x) {
        int run = 0;
        for (int w = 0; w < nw; ++w) {          // whist[w][u] := rows of group u in warps before w
            const int c = whist[w * G + u];
            whist[w * G + u] = run;
            run += c;
        }
        gsum[u] = run;
        counts[u] = run;
    }
    __syncthreads();
    block_exclusive_scan(gsum, G, tmp, s_total);
    for (int u = threadIdx.x; u < G; u += blockDim.x) {
        offsets[u] = gsum[u];
        for (int w = 0; w < nw; ++w) whist[w * G + u] += gsum[u];
    }
    if (threadIdx.x == 0) { offsets[G] = *s_total; status[1] = *s_total; }
    __syncthreads();
    warp_permute(group_ids, items, (long long)warp * per_warp, K, whist + warp * G, lane, *s_total,
                 row_token, row_slot, slot_row, per_warp);
}

}  // namespace bm
