// bm_permute.cu -- steps R6-R8: per-group histogram, exclusive scan and the stable permutation that
// builds the per-group token lists (BASELINE.json north_star (2): "a warp-level histogram plus
// prefix-scan permutation kernel"; reading A7: rows ordered by group, then token ascending).
//
// The (token, slot) pairs are "items" i = t*K + s.  After dedup a token holds a group at most once,
// so ordering the items of one group by i is ordering them by token: a STABLE counting sort of the
// items keyed by group is exactly the required permutation, and it is deterministic -- no atomics
// whose arrival order could matter.
//
//   block b owns items [b*512, (b+1)*512); warp w of the block owns a contiguous eighth of them and
//   walks it 32 items at a time.  __match_any_sync gives every lane the set of lanes holding its key:
//   rank inside the round = popc(set & lanes below), the round's count = popc(set).
//
//   P1  hist    : per-warp counts in shared memory -> per-block counts block_hist[b][u]
//   P2  scan    : counts[u] = sum_b, offsets = exclusive scan over u, block_hist[b][u] := rows of group u in
//                 the blocks before b (P3 adds offsets[u])
//   P3  permute : per-warp bases from P2's block bases, replay the walk, write row_token / row_slot /
//                 slot_row; pads get -1
//   T*K <= 2048 : one CTA does P1-P3 in a single launch (the decode case).
#include "bm_common.cuh"
#include "bm_permute.cuh"
#include "bm_ptx.cuh"

namespace bm {

namespace {

constexpr int kWarps = kPermWarps;
constexpr int kItemsPerWarp = kPermItemsPerWarp;

// ---- T*K <= 2048: everything in one CTA --------------------------------------------------------
// (One CTA of 32 warps for up to 32768 items was measured too: 31-46 us against 20-24 us for the three-kernel
// path -- the serial rounds of one CTA expose every global-load latency.)
__global__ void __launch_bounds__(1024)
permute_small_kernel(const int32_t *__restrict__ group_ids, int T, int K, int G, int per_warp,
                     int32_t *__restrict__ counts, int32_t *__restrict__ offsets,
                     int32_t *__restrict__ row_token, int32_t *__restrict__ row_slot,
                     int32_t *__restrict__ slot_row, int32_t *__restrict__ status) {
    extern __shared__ int s_mem[];
    __shared__ int s_total;
    // This one-CTA kernel lets its successor start BEFORE it waits for the router: the successor (a GEMM1 kernel) only
    // sets up barriers and TMEM and asks L2 for weights ahead of its own grid-dependency wait, and that wait still covers
    // this kernel and, through its wait below, the router.  The weight prefetch then overlaps router + permutation.
    grid_dep_launch();
    grid_dep_wait();
    permute_block_small(group_ids, T, K, G, per_warp, counts, offsets, row_token, row_slot, slot_row, status, s_mem,
                        &s_total);
}

// ---- general case: P1 / P2 / P3 ---------------------------------------------------------------
__global__ void __launch_bounds__(kWarps * 32)
permute_hist_kernel(const int32_t *__restrict__ group_ids, int T, int K, int G,
                    int32_t *__restrict__ block_hist) {
    extern __shared__ int s_mem[];
    grid_dep_launch();     // (not the first kernel of a call: the successor waits for this grid itself)
    grid_dep_wait();
    int *whist = s_mem;                  // [kWarps][G]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long items = (long long)T * K;
    for (int i = threadIdx.x; i < kWarps * G; i += blockDim.x) whist[i] = 0;
    __syncthreads();
    const long long first = (long long)blockIdx.x * kPermItemsPerBlock + (long long)warp * kItemsPerWarp;
    warp_histogram(group_ids, items, first, whist + warp * G, lane);
    __syncthreads();
    for (int u = threadIdx.x; u < G; u += blockDim.x) {
        int run = 0;
        for (int w = 0; w < kWarps; ++w) run += whist[w * G + u];
        block_hist[(size_t)blockIdx.x * G + u] = run;
    }
}

__global__ void __launch_bounds__(256)
permute_scan_kernel(int nb, int G, int32_t *__restrict__ block_hist, int32_t *__restrict__ counts,
                    int32_t *__restrict__ offsets, int32_t *__restrict__ status) {
    __shared__ int gsum[512];
    __shared__ int tmp[512];
    __shared__ int s_total;
    grid_dep_launch();     // (not the first kernel of a call: the successor waits for this grid itself)
    grid_dep_wait();
    // block_hist[b][u] := rows of group u in blocks before b (the scatter kernel adds offsets[u]).  Thread u
    // walks the blocks eight at a time: eight independent loads, then the running sums and eight stores --
    // one memory round trip per eight blocks instead of one per block (the first version took 8 us at 12
    // blocks and 44 us at 32).
    for (int u = threadIdx.x; u < G; u += blockDim.x) {
        int run = 0;
        for (int b0 = 0; b0 < nb; b0 += 8) {
            int c[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) c[j] = b0 + j < nb ? block_hist[(size_t)(b0 + j) * G + u] : 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (b0 + j < nb) block_hist[(size_t)(b0 + j) * G + u] = run;
                run += c[j];
            }
        }
        gsum[u] = run;
        counts[u] = run;
    }
    __syncthreads();
    block_exclusive_scan(gsum, G, tmp, &s_total);
    for (int u = threadIdx.x; u < G; u += blockDim.x) offsets[u] = gsum[u];
    if (threadIdx.x == 0) { offsets[G] = s_total; status[1] = s_total; }
}

__global__ void __launch_bounds__(kWarps * 32)
permute_scatter_kernel(const int32_t *__restrict__ group_ids, int T, int K, int G,
                       const int32_t *__restrict__ block_hist, const int32_t *__restrict__ offsets,
                       int32_t *__restrict__ row_token, int32_t *__restrict__ row_slot,
                       int32_t *__restrict__ slot_row) {
    extern __shared__ int s_mem[];
    grid_dep_launch();     // (not the first kernel of a call: the successor waits for this grid itself)
    grid_dep_wait();
    int *whist = s_mem;                  // [kWarps][G]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long items = (long long)T * K;
    for (int i = threadIdx.x; i < kWarps * G; i += blockDim.x) whist[i] = 0;
    __syncthreads();
    const long long first = (long long)blockIdx.x * kPermItemsPerBlock + (long long)warp * kItemsPerWarp;
    warp_histogram(group_ids, items, first, whist + warp * G, lane);
    __syncthreads();
    for (int u = threadIdx.x; u < G; u += blockDim.x) {
        int run = offsets[u] + block_hist[(size_t)blockIdx.x * G + u];
        for (int w = 0; w < kWarps; ++w) {
            const int c = whist[w * G + u];
            whist[w * G + u] = run;
            run += c;
        }
    }
    __syncthreads();
    warp_permute(group_ids, items, first, K, whist + warp * G, lane, offsets[G], row_token, row_slot,
                 slot_row);
}

// ---- 2048 < T*K <= 65536: one cluster of eight CTAs, one launch -----------------------------------------------
// The three-kernel path spends most of its 20-26 us (T = 4096 .. 16384, top-4) on two kernel boundaries and on a scan
// kernel whose single CTA walks the block histograms serially.  Here the eight CTAs of a thread-block cluster split the
// items 256 ways (32 warps each); a warp keeps its <= 8 rounds of keys in REGISTERS (all loads in flight at once, no
// second read for the replay), the CTAs publish their per-group counts in shared memory, and after one cluster barrier
// every CTA reads the other seven through distributed shared memory: counts, offsets and its own bases follow without a
// trip through global memory.  A second cluster barrier keeps every CTA's counts alive until all peers have read them.
constexpr int kClSize = 8, kClWarps = 16, kClMaxRounds = 16;
constexpr long long kPermClusterItems = (long long)kClSize * kClWarps * kClMaxRounds * 32;      // 65536

__device__ __forceinline__ int ld_shared_cluster(uint32_t addr) {
    int v;
    asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

__global__ void __launch_bounds__(kClWarps * 32, 1)
permute_cluster_kernel(const int32_t *__restrict__ group_ids, int T, int K, int G, int per_warp,
                       int32_t *__restrict__ counts, int32_t *__restrict__ offsets,
                       int32_t *__restrict__ row_token, int32_t *__restrict__ row_slot,
                       int32_t *__restrict__ slot_row, int32_t *__restrict__ status) {
    extern __shared__ int s_mem[];
    __shared__ int s_total;
    int *whist = s_mem;                      // [kClWarps][G]: counts, then bases of this CTA's warps
    int *ctot = whist + kClWarps * G;        // [G] this CTA's counts, read by its peers
    int *gsum = ctot + G;                    // [G] group totals -> offsets
    grid_dep_launch();     // (not the first kernel of a call: the successor waits for this grid itself)
    grid_dep_wait();
    const int rank = (int)ptx::cluster_ctarank();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long items = (long long)T * K;
    const long long first = ((long long)rank * kClWarps + warp) * per_warp;
    int keys[kClMaxRounds];
#pragma unroll
    for (int r = 0; r < kClMaxRounds; ++r) {
        const long long i = first + r * 32 + lane;
        keys[r] = (r * 32 < per_warp && i < items) ? __ldcg(group_ids + i) : -1;
    }
    for (int i = threadIdx.x; i < kClWarps * G; i += blockDim.x) whist[i] = 0;
    __syncthreads();
    int *whist_w = whist + warp * G;
#pragma unroll
    for (int r = 0; r < kClMaxRounds; ++r) {
        if (r * 32 < per_warp) {                                       // warp-uniform
            const unsigned peers = __match_any_sync(kFullMask, keys[r]);
            if (keys[r] >= 0 && lane == __ffs(peers) - 1) whist_w[keys[r]] += __popc(peers);
            __syncwarp();
        }
    }
    __syncthreads();
    const int u = threadIdx.x;               // G <= 512 < blockDim.x: one thread per group
    if (u < G) {
        int run = 0;
        for (int w = 0; w < kClWarps; ++w) {                           // whist[w][u] := rows of group u in this CTA's warps before w
            const int c = whist[w * G + u];
            whist[w * G + u] = run;
            run += c;
        }
        ctot[u] = run;
    }
    ptx::cluster_sync_all();
    int before = 0;
    if (u < G) {
        int tot = 0;
#pragma unroll
        for (int c = 0; c < kClSize; ++c) {
            const int v = ld_shared_cluster(ptx::mapa_u32(&ctot[u], (uint32_t)c));
            if (c < rank) before += v;
            tot += v;
        }
        gsum[u] = tot;
        if (rank == 0) counts[u] = tot;
    }
    block_exclusive_scan(gsum, G, nullptr, &s_total);
    if (u < G) {
        const int base = gsum[u] + before;
        for (int w = 0; w < kClWarps; ++w) whist[w * G + u] += base;
        if (rank == 0) offsets[u] = gsum[u];
    }
    if (rank == 0 && threadIdx.x == 0) { offsets[G] = s_total; status[1] = s_total; }
    ptx::cluster_sync_all();                 // peers have read ctot; this CTA's bases are complete
    const int A = s_total;
#pragma unroll
    for (int r = 0; r < kClMaxRounds; ++r) {
        if (r * 32 < per_warp) {
            const long long i = first + r * 32 + lane;
            const int key = keys[r];
            const unsigned peers = __match_any_sync(kFullMask, key);
            if (i < items) {
                if (key >= 0) {
                    const int row = whist_w[key] + __popc(peers & ((1u << lane) - 1u));
                    row_token[row] = (int32_t)(i / K);
                    row_slot[row] = (int32_t)(i % K);
                    slot_row[i] = row;
                } else {
                    slot_row[i] = -1;
                }
                if (i >= A) {                   // rows past A stay -1 (A <= items)
                    row_token[i] = -1;
                    row_slot[i] = -1;
                }
            }
            __syncwarp();
            if (key >= 0 && lane == __ffs(peers) - 1) whist_w[key] += __popc(peers);
            __syncwarp();
        }
    }
}

}  // namespace

cudaError_t launch_permute(int T, int K, int G, const bm_routing &r, int32_t *block_hist, int32_t *status,
                           cudaStream_t stream) {
    const long long items = (long long)T * K;
    const int nb = (int)((items + kPermItemsPerBlock - 1) / kPermItemsPerBlock);
    const size_t smem_w = (size_t)kWarps * G * sizeof(int);
    if (items <= kPermSmallItems) {
        // few items: 8 warps; otherwise 16 warps with a few rounds of 32 items each, so the serial chain of
        // rounds (load -> match -> shared-memory update, twice) stays short
        int nw = opt(OPT_PERM_SMALL_WARPS);
        if (nw <= 0) nw = items <= 256 ? 8 : 16;      // measured at 1024 items: 8 warps 10.2, 16 warps 8.7, 32 warps 9.9 us
        int per_warp = (int)((items + nw - 1) / nw);
        per_warp = (per_warp + 31) / 32 * 32;
        const size_t smem = (size_t)nw * G * sizeof(int) + (size_t)(G + 512) * sizeof(int);
        if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(permute_small_kernel), smem); ea != cudaSuccess) return ea;
        return launch_kernel(permute_small_kernel, dim3(1), dim3(nw * 32), smem, stream, (const int32_t *)r.group_ids,
                             T, K, G, per_warp, r.counts, r.offsets, r.row_token, r.row_slot, r.slot_row, status);
    }
    if (items <= kPermClusterItems && G <= 512 && opt(OPT_PERM_CLUSTER) != 0) {
        int per_warp = (int)((items + kClSize * kClWarps - 1) / (kClSize * kClWarps));
        per_warp = (per_warp + 31) / 32 * 32;
        const size_t smem = (size_t)(kClWarps + 2) * G * sizeof(int);
        if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(permute_cluster_kernel), smem); ea != cudaSuccess) return ea;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(kClSize); cfg.blockDim = dim3(kClWarps * 32); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = kClSize; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = pdl_enabled() ? 2 : 1;
        count_launch();
        return cudaLaunchKernelEx(&cfg, permute_cluster_kernel, (const int32_t *)r.group_ids, T, K, G, per_warp, r.counts, r.offsets,
                                  r.row_token, r.row_slot, r.slot_row, status);
    }
    cudaError_t e = launch_kernel(permute_hist_kernel, dim3(nb), dim3(kWarps * 32), smem_w, stream,
                                  (const int32_t *)r.group_ids, T, K, G, block_hist);
    if (e != cudaSuccess) return e;
    e = launch_kernel(permute_scan_kernel, dim3(1), dim3(256), 0, stream, nb, G, block_hist, r.counts, r.offsets, status);
    if (e != cudaSuccess) return e;
    return launch_kernel(permute_scatter_kernel, dim3(nb), dim3(kWarps * 32), smem_w, stream,
                         (const int32_t *)r.group_ids, T, K, G, (const int32_t *)block_hist, (const int32_t *)r.offsets,
                         r.row_token, r.row_slot, r.slot_row);
}

}  // namespace bm
