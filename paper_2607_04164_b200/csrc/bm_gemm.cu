// bm_gemm.cu -- steps 9-13 on the tensor cores: gather, grouped W1/W3 GEMM + SwiGLU, grouped W2 GEMM +
// gate-weighted scatter-combine, for both regimes.
//
// Cite: PAPER.md:42 (h_t = sum g_i FFN_i(x_t)), PAPER.md:46 (united experts: fewer expert weight sets
// loaded), BASELINE.json north_star (3), (4) and the decode/prefill split; A3, A11, A12.
//
// One persistent warp-specialised kernel template, four modes:
//   PF_GEMM1  prefill  H[r, f]   = SiLU(xs_r . W1[u]_f) * (xs_r . W3[u]_f)        tokens on the MMA M side
//   PF_GEMM2  prefill  acc[t, d] += gate_w * (H_r . W2[u]_d)                       128 x 256 tiles
//   DC_GEMM1  decode   same math, WEIGHT rows on the MMA M side (swap-AB): a tile streams R weight
//   DC_GEMM2  decode   rows x 64 columns per stage, the <= 128 token rows of the group are the N side
// Roles (192 threads): warp 0 lane 0 = TMA producer, warp 1 lane 0 = tcgen05.mma issuer (warp 1 also
// owns the TMEM allocation), warps 2-5 = epilogue (TMEM lane quarter = warp & 3).
// Pipelines: a 4-stage shared-memory ring (full/empty mbarriers, 48 KB per stage, 128B-swizzled K-major
// tiles written by TMA) and two TMEM accumulator stages of 256 columns (tmem_full/tmem_empty), so the
// epilogue of item i overlaps the main loop of item i+1.  Work items are enumerated identically by all
// roles from a small schedule (non-empty segments and their 128-row chunks) that warp 0 of every CTA builds in
// shared memory from counts/offsets (build_schedule) -- the host never sees the data-dependent counts.
//
// Combine.  A token's <= K group rows live in different tiles.  Fused form (FC; prefill tiles with F >= 4096, decode up
// to 64 tokens): the GEMM2 epilogue adds gate_w * y into the fp32 accumulator out_acc with red.global.add (vectorised and
// row-coalesced on the prefill tiles), takes a ticket, and the arrival that completes an output piece rounds it to bf16
// and clears accumulator and ticket -- no y rows, no combine / finalize kernel, no zeroing pass.  Two-pass form where the
// fused epilogue was measured slower: prefill tiles store y rows (bf16, coalesced 128-byte pieces) and combine_kernel sums
// a token's rows in slot order (deterministic); the decode kernel's reductions are rounded and cleared by finalize_kernel.
#include <algorithm>
#include <mutex>

#include "bm_common.cuh"
#include "bm_ptx.cuh"

namespace bm {

namespace {

constexpr int kBlockK = 64;                 // bf16 elements per stage row = 128 bytes = one swizzle row
constexpr int kMaxStages = 12;
constexpr int kTileBytes16K = 128 * 128;    // 128 rows x 128 bytes
constexpr int kAccStages = 2;
constexpr int kAccCols = 256;
constexpr int kTmemCols = kAccStages * kAccCols;
constexpr int kThreads = 192;
constexpr int kGatherCopyThreads = 128; // GA: warps 6..9 gather the token rows of GEMM1's A tile
constexpr int kGatherRelays = 6;        // + warps 10..15, which relay "copies landed" to the stages' full barriers (ring stage s -> relay s % 6)
constexpr int kGatherThreads = kGatherCopyThreads + 32 * kGatherRelays;
constexpr int kChunkRows = 128;
constexpr int kMaxSeg = BM_MAX_G + kMaxShared;
constexpr size_t kSmemMax = 232448;         // 227 KB, the per-CTA opt-in limit of sm_100
constexpr size_t kSmemBars = 512;           // (3*kMaxStages + 2*kAccStages) mbarriers + the TMEM base address
constexpr int kSchedBarSlot = 3 * kMaxStages + 2 * kAccStages + 1 + 3;   // behind the schedule header (3 ints): "schedule built"
static_assert((kSchedBarSlot + 1) * 8 <= kSmemBars, "barrier block too small");
constexpr size_t kEpiStageBytes = 32 * 32 * 4;   // PF_GEMM2: per-epilogue-warp transpose buffer (32 rows x 32 fp32)
constexpr size_t kSmemEpi = 4 * kEpiStageBytes;
constexpr size_t kSmemRing = kSmemMax - 1024 /*align slack*/ - kSmemBars;   // minus kSmemEpi for PF_GEMM2
static_assert((3 * kMaxStages + 2 * kAccStages + 1) * 8 <= kSmemBars, "barrier block too small");

enum Mode { PF_GEMM1 = 0, PF_GEMM2 = 1, DC_GEMM1 = 2, DC_GEMM2 = 3 };

// schedule: the non-empty segments (groups, then shared experts), five int arrays of seg_cap entries in each CTA's
// shared memory (build_schedule):  u = weight set; chunk0 = first 128-row chunk (entry n_seg = total); rows;
// off = first permuted row (offsets[u]; 0 for a shared expert); pair0 = first chunk PAIR (CTA-pair tiles).
struct SchedView {
    int n_seg, total_chunks, total_pairs;
    const int32_t *u, *chunk0, *rows, *off, *pair0;
};
struct GemmParams {
    int T, D, F, K, G, S, TK;
    int stages;         // depth of the shared-memory ring (<= kMaxStages)
    int stage_bytes;    // bytes of one ring stage (multiple of 1024)
    int off_b;          // decode: offset of the token rows (MMA B operand) inside a stage
    int wslot;          // decode: bytes between the W1 and W3 tiles of a stage (R*128 rounded up to 1024)
    int tail_pad;       // decode: bytes kept free after the ring (an M=128 MMA reads 16 KB from a tile base, R < 128 rows of it real)
    int kblocks;        // k-blocks of one item (per split)
    int kpack;          // decode: k-blocks per ring stage (1 or 2; kblocks % kpack == 0).  The single-thread issue loop costs
                        // ~0.25 us per barrier turn whatever the tile holds, so a stage carries two k-blocks when it can
    int mini_bytes;     // decode: bytes of one k-block inside a stage (stage_bytes = kpack * mini_bytes)
    int ksplit;         // K splits (DC_GEMM2), else 1
    int R;              // weight rows per tile (prefill: 128 for GEMM1 per matrix, 256 for GEMM2)
    int n_wtiles;       // tiles along the weight-row dimension
    int band_c;         // prefill item order: chunk units (chunks, or chunk pairs) per L2 band ...
    int band_w;         // ... and weight tiles per band (see get_item); <= 0: one band
    const bm_bf16 *w1, *w3;   // DC_GEMM1: weight arrays, for the L2 prefetch before the grid-dependency wait
    unsigned long long pf_set_bytes, pf_bytes;   // bytes of one weight set (F * D * 2) and how many leading bytes of each to prefetch
    int dense;          // decode, T <= 64: every active set takes ALL T tokens as its rows (no gather, no permutation needed):
                        // H row = segment * T + token; GEMM2 weighs token t of set u with its gate weight, 0 if not routed there
    int32_t *status;    // device status word (BM_DEV_BAD_ROUTING)
    const int32_t *group_ids;
    int hints;          // L2 eviction hints of the TMA loads, 10 * activations + weights: 0 = evict_first, 1 = normal, 2 = evict_last
    int seg_cap;        // G + S + 1: entries per schedule array cached in shared memory
    const int32_t *counts, *offsets, *row_token, *row_slot;
    const bm_bf16 *x;   // GA: token rows gathered straight from x [T, D]
    const float *gate_w;
    const int32_t *n_slots;
    bm_bf16 *h;
    float *out_acc;     // zero region: fp32 accumulator of the fused combine [T, D]
    int32_t *tickets;   // zero region: arrivals per (token, output piece)
    bm_bf16 *y;         // two-pass combine: per-row expert outputs
    int y_tm;           // calibration: y is token-major [T, S, D] (row of shared set j, token t = t * S + j)
    int dense_u;        // dense decode with G <= T*K: H rows are indexed by the weight set itself (row u * T + t)
    int spec_sets;      // DC_GEMM1, dense_u: routed sets 0 .. spec_sets-1 are multiplied BEFORE the routing is known
    int spec_shared;    // PF_GEMM1: the S shared experts' items (all T tokens, no routing needed) run BEFORE the routing is known
    bm_bf16 *out;       // fused combine: the layer output [T, D] bf16 ...
    float *out_f32;     // ... or, when non-null, the fp32 sums (tensor-parallel partial)
};

struct Item {
    int u;          // weight set (group, or G+j for shared expert j)
    int n;          // valid rows in this chunk (1..128)
    int act_row0;   // first row in the activation source (xs / x for GEMM1, H for GEMM2)
    int h_row0;     // first row in H space
    int perm_row0;  // first permuted row (routed) -- index into row_token/row_slot
    int tok0;       // first token (shared experts)
    int wt;         // weight tile index
    int ks;         // K split index
    bool shared;
};

// K2 (CTA-pair prefill tiles): an item is a PAIR of consecutive 128-row chunks of one segment on one weight
// tile; `rank` (0 or 1) picks this CTA's chunk.  A segment with an odd chunk count leaves rank 1 of its last
// pair without rows (it.n = 0: it loads a valid tile, multiplies it and stores nothing).
template <int MODE, bool K2 = false>
__device__ __forceinline__ bool get_item(const GemmParams &p, const SchedView &sv, int item, Item &it, int rank = 0) {
    const int per_chunk = p.n_wtiles * p.ksplit;
    const int32_t *first = K2 ? sv.pair0 : sv.chunk0;
    const long long n_items = (long long)(K2 ? sv.total_pairs : sv.total_chunks) * per_chunk;
    if (item >= n_items) return false;
    int lo = 0, hi = sv.n_seg - 1;            // last segment s with first[s] * per_chunk <= item
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((long long)first[mid] * per_chunk <= item) lo = mid; else hi = mid - 1;
    }
    const int s = lo;
    const int u = sv.u[s];
    const int c0 = first[s];
    const int units_s = first[s + 1] - c0;
    const int local = item - c0 * per_chunk;
    int unit, rest;
    if (MODE == PF_GEMM1 || MODE == PF_GEMM2) {
        // L2-aware item order.  The CTAs work on ~148 consecutive items at a time, all streaming through K in step, so
        // what reaches DRAM is the set of DISTINCT operand tiles of those items plus whatever L2 cannot keep until the
        // next visit.  A segment's (chunk unit x weight tile) grid is therefore walked in bands:
        //   [weight-tile band of band_w][chunk band of band_c][weight tile in band][chunk unit in band]   (unit fastest)
        // GEMM1 uses one weight band (band_w = all): a chunk band's token rows (band_c x 128/256 rows x D) stay in L2
        // while all weight tiles stream past once.  GEMM2's operands are K = F long: a band of band_w W2 tiles is kept
        // while the H rows of the chunk bands stream past.  The plain chunk-fastest order of round 1 re-read the token
        // rows of a large group (60 MB at BJ:configs[2]) for every weight tile: 3.4x / 4.7x the algorithmic DRAM bytes.
        const int Bw = (p.band_w > 0 && p.band_w < p.n_wtiles) ? p.band_w : p.n_wtiles;
        const int Bc = (p.band_c > 0 && p.band_c < units_s) ? p.band_c : units_s;
        const int per_wb = units_s * Bw;
        const int wb = local / per_wb, r1 = local - wb * per_wb;
        const int bw = min(Bw, p.n_wtiles - wb * Bw);
        const int cb = r1 / (Bc * bw), r2 = r1 - cb * (Bc * bw);
        const int bc = min(Bc, units_s - cb * Bc);
        const int wt_in = r2 / bc;
        unit = cb * Bc + (r2 - wt_in * bc);
        rest = wb * Bw + wt_in;
    } else {
        unit = local % units_s;
        rest = local / units_s;
    }
    int chunk = K2 ? 2 * unit + rank : unit;
    it.u = u;
    it.ks = rest % p.ksplit;
    it.wt = rest / p.ksplit;
    it.shared = u >= p.G;
    const int rows = sv.rows[s];
    it.n = min(kChunkRows, rows - chunk * kChunkRows);
    if (K2 && it.n <= 0) { it.n = 0; chunk = 0; }        // absent half of the last pair: point at real rows
    if (p.dense) {
        it.tok0 = chunk * kChunkRows;
        it.perm_row0 = 0;
        it.h_row0 = (p.dense_u ? u : s) * p.T + it.tok0;
        it.act_row0 = (MODE == PF_GEMM1 || MODE == DC_GEMM1) ? it.tok0 : it.h_row0;
    } else if (it.shared) {
        it.tok0 = chunk * kChunkRows;
        it.perm_row0 = 0;
        it.h_row0 = p.TK + (u - p.G) * p.T + it.tok0;
        it.act_row0 = (MODE == PF_GEMM1 || MODE == DC_GEMM1) ? it.tok0 : it.h_row0;
    } else {
        it.tok0 = 0;
        it.perm_row0 = sv.off[s] + chunk * kChunkRows;
        it.h_row0 = it.perm_row0;
        it.act_row0 = it.perm_row0;
    }
    return true;
}

// The schedule, built by warp 0 of every CTA in its own shared memory straight from counts / offsets (one coalesced
// global read, then ballot + shuffle scans 32 sets at a time): the non-empty segments (groups, then the S shared
// experts with T rows each), their first chunk / chunk pair, rows and first permuted row.  Round 1 had a prep kernel
// write this to global memory and every CTA copy it -- the same latency on the critical path plus a launch.
// hdr[0..2] = segments, chunks, chunk pairs.  dense: an active group takes all T tokens as rows.
__device__ __forceinline__ void build_schedule(const GemmParams &p, int32_t *s_sched, int cap, int *hdr) {
    const int lane = threadIdx.x & 31;
    const int n = p.G + p.S;
    int seg_base = 0, chunk_base = 0, pair_base = 0;
    bool bad = false;
    for (int u0 = 0; u0 < n; u0 += 32) {
        const int u = u0 + lane;
        int rows = 0, off = 0;
        if (u < n) {
            if (u < p.G) {
                rows = p.counts[u];
                off = p.offsets[u];
                if (rows < 0 || off < 0 || off + rows > p.TK) { bad = true; rows = 0; }
                if (p.dense && rows > 0) rows = p.T;
                if (u < p.spec_sets) rows = 0;          // done ahead of the routing (DC_GEMM1 only)
            } else {
                rows = p.spec_shared ? 0 : p.T;         // (PF_GEMM1 only: done ahead of the routing)
            }
        }
        const bool ne = rows > 0;
        const int ch = ne ? (rows + kChunkRows - 1) / kChunkRows : 0;
        const unsigned m = __ballot_sync(kFullMask, ne);
        const int seg = seg_base + __popc(m & ((1u << lane) - 1u));
        const int pr = (ch + 1) >> 1;
        int inc = ch, incp = pr;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(kFullMask, inc, o);
            const int vp = __shfl_up_sync(kFullMask, incp, o);
            if (lane >= o) { inc += v; incp += vp; }
        }
        if (ne && seg < cap - 1) {
            s_sched[seg] = u;
            s_sched[cap + seg] = chunk_base + inc - ch;
            s_sched[2 * cap + seg] = rows;
            s_sched[3 * cap + seg] = off;
            s_sched[4 * cap + seg] = pair_base + incp - pr;
        }
        seg_base += __popc(m);
        chunk_base += __shfl_sync(kFullMask, inc, 31);
        pair_base += __shfl_sync(kFullMask, incp, 31);
    }
    bad = __any_sync(kFullMask, bad);
    if (lane == 0) {
        if (seg_base > cap - 1) seg_base = cap - 1;
        s_sched[cap + seg_base] = chunk_base;
        s_sched[4 * cap + seg_base] = pair_base;
        hdr[0] = seg_base; hdr[1] = chunk_base; hdr[2] = pair_base;
        if (bad && blockIdx.x == 0 && p.status) atomicOr(p.status, BM_DEV_BAD_ROUTING);
    }
    __syncwarp();
}

__device__ __forceinline__ float silu_mul(float a, float b) {
    return __fdividef(a, 1.0f + __expf(-a)) * b;
}

// Fused combine (FC, GEMM2 only; north_star kernel (4)): the epilogue multiplies its rows by their gate weights and adds
// them into the fp32 accumulator out_acc [T, D] with vector reductions at L2 (red.global.add.v4.f32), then takes a
// ticket per (token, output piece).  The arrival that completes a piece -- all n_slots[t] + S source rows of the
// token (times the K splits on the decode path) have been added -- reads the sums back, rounds them to bf16 into
// `out` (or stores them as fp32 into out_f32) and puts accumulator and ticket back to zero, so neither a zeroing
// pass, nor y rows, nor a combine / finalize kernel exist.  fp32 addition is commutative, so with at most two
// sources per token (K + S <= 2, e.g. Mixtral's top-2) the result is bit-deterministic; with more sources the
// association follows the arrival order (last-bit differences before the bf16 rounding).  Writers fence between
// their reductions and the ticket, the finisher fences between the ticket and its reads (threadFenceReduction).
template <int MODE, bool K2 = false, bool GA = false, bool FC = false>
__global__ void __launch_bounds__(kThreads + (GA ? kGatherThreads : 0), 1)
gemm_kernel(const __grid_constant__ CUtensorMap tm_act0,   // GEMM1: xs [TK, D]; GEMM2: H [TK+S*T, F]
            const __grid_constant__ CUtensorMap tm_act1,   // GEMM1: x [T, D] (shared experts); GEMM2: unused
            const __grid_constant__ CUtensorMap tm_w0,     // GEMM1: W1 [G+S, F, D]; GEMM2: W2 [G+S, D, F]
            const __grid_constant__ CUtensorMap tm_w1,     // GEMM1: W3; GEMM2: unused
            const GemmParams p) {
    constexpr bool kDecode = (MODE == DC_GEMM1 || MODE == DC_GEMM2);
    constexpr bool kGemm1 = (MODE == PF_GEMM1 || MODE == DC_GEMM1);
    static_assert(!K2 || !kDecode, "CTA pairs are a prefill-tile feature");
    static_assert(!GA || MODE == PF_GEMM1, "the in-kernel gather feeds GEMM1's activation tile");
    static_assert(!FC || MODE == PF_GEMM2 || MODE == DC_GEMM2, "the fused combine is GEMM2's epilogue");
    // K2: the two CTAs of a cluster form a CTA pair; rank 0 (the leader) issues the M = 256 MMAs for both
    const uint32_t rank = K2 ? ptx::cluster_ctarank() : 0u;
    const bool leader = rank == 0;
    const int item0 = K2 ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
    const int item_stride = K2 ? (int)(gridDim.x >> 1) : (int)gridDim.x;

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int n_stages = p.stages;
    const uint32_t stage_bytes = (uint32_t)p.stage_bytes;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + (size_t)n_stages * stage_bytes);
    uint64_t *full = bars;                       // [kMaxStages]
    uint64_t *empty = bars + kMaxStages;         // [kMaxStages]
    uint64_t *tfull = bars + 2 * kMaxStages;     // [kAccStages]
    uint64_t *tempty = tfull + kAccStages;       // [kAccStages]
    uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(tempty + kAccStages);
    uint64_t *gfull = tempty + kAccStages + 1;   // [kMaxStages] GA: the gather threads' copies of a stage have landed
    uint8_t *epi_stage = reinterpret_cast<uint8_t *>(bars) + kSmemBars;   // [4][kEpiStageBytes], 256-byte aligned
    int32_t *s_sched = reinterpret_cast<int32_t *>(epi_stage + (MODE == PF_GEMM2 ? kSmemEpi : 0));   // [5][seg_cap]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // ---- prologue: nothing here depends on a predecessor kernel, so under PDL it overlaps its tail ----
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tm_act0);
        ptx::prefetch_tmap(&tm_w0);
        if (kGemm1) { ptx::prefetch_tmap(&tm_act1); ptx::prefetch_tmap(&tm_w1); }
        // GA: a stage is full when the TMA bytes (weights) have landed AND the relay warp (both CTAs' under K2) has signalled that the gathered rows are in place
        for (int i = 0; i < n_stages; ++i) { ptx::mbar_init(&full[i], GA ? 1 + (K2 ? 2 : 1) : 1); ptx::mbar_init(&empty[i], 1); }
        if (GA) for (int i = 0; i < n_stages; ++i) ptx::mbar_init(&gfull[i], kGatherCopyThreads);
        if (kGemm1) ptx::mbar_init(bars + kSchedBarSlot, 1);     // "schedule built" (speculative start, below)
        // K2: the leader's tempty collects the 4 epilogue warps of BOTH CTAs
        for (int i = 0; i < kAccStages; ++i) { ptx::mbar_init(&tfull[i], 1); ptx::mbar_init(&tempty[i], K2 ? 8 : 4); }
        ptx::fence_barrier_init();
    }
    if (warp == 1) {
        if (K2) ptx::tmem_alloc_pair(tmem_ptr, kTmemCols); else ptx::tmem_alloc(tmem_ptr, kTmemCols);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (K2) ptx::cluster_sync_all();      // both CTAs' barriers exist before either signals the other
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    const int kp = kDecode ? p.kpack : 1;                 // k-blocks per ring stage
    const int nkb = p.kblocks / kp;                       // ring stages of one item
    const uint32_t mini = kDecode ? (uint32_t)p.mini_bytes : stage_bytes;
    // bytes one stage receives: constant per launch (decode always loads the full padded token box)
    // bytes one stage receives.  Decode: the weight box(es) of R rows plus the item's token rows in 32-row
    // boxes (tok_tx(n)): only the rows the group really has travel from L2.
    // K2: a CTA stages A (16 KB) + its half of B (16 KB); the leader's barrier counts both CTAs' bytes
    const uint32_t w_tx = GA ? 2u * kTileBytes16K : K2 ? 4u * kTileBytes16K : !kDecode ? 3u * kTileBytes16K : (uint32_t)((kGemm1 ? 2 : 1) * p.R * 128);
    auto stage_tx_of = [&](int n) -> uint32_t { return kDecode ? (uint32_t)kp * (w_tx + (uint32_t)((n + 31) >> 5) * 4096u) : w_tx; };

    // Schedule (build_schedule): from counts / offsets, which bm_route's kernels wrote.  GEMM1 is their direct
    // successor and builds it after the grid-dependency wait.  GEMM2 builds it BEFORE the wait: its predecessor GEMM1
    // let this grid start only after its own wait had returned, i.e. after the routing kernels had completed.
    // DC_GEMM2: W2 does not depend on GEMM1 either, so warp 0 also fills the ring with the weight tiles of its first
    // item before the wait: the HBM stream starts while GEMM1's last CTAs drain.
    int *s_hdr = reinterpret_cast<int *>(gfull + kMaxStages);
    const int cap = p.seg_cap;
    SchedView sv;
    sv.u = s_sched; sv.chunk0 = s_sched + cap; sv.rows = s_sched + 2 * cap; sv.off = s_sched + 3 * cap;
    sv.pair0 = s_sched + 4 * cap;
    Item it0;
    bool have0 = false;
    int pre = 0;
    if (!kGemm1 && warp == 0) build_schedule(p, s_sched, cap, s_hdr);
    if (MODE == DC_GEMM2 && warp == 0) {
        sv.n_seg = s_hdr[0]; sv.total_chunks = s_hdr[1]; sv.total_pairs = s_hdr[2];
        have0 = get_item<MODE, false>(p, sv, blockIdx.x, it0);
        pre = have0 ? min(n_stages, nkb) : 0;
        if (ptx::elect_one())
            for (int kb = 0; kb < pre; ++kb) {
                ptx::mbar_arrive_expect_tx(&full[kb], stage_tx_of(it0.n));
                for (int kk = 0; kk < kp; ++kk)
                    ptx::tma_load_3d(smem + (size_t)kb * stage_bytes + kk * mini, &tm_w0, &full[kb],
                                     ((it0.ks * nkb + kb) * kp + kk) * kBlockK, it0.wt * p.R, it0.u, ptx::kEvictFirst);
            }
        __syncwarp();
    }
    if (MODE == DC_GEMM1 && warp == 2 && p.pf_bytes) {
        // The weights do not depend on the routing, and while the router runs HBM is idle: every CTA asks L2 for its
        // share of the leading pf_bytes of each W1 / W3 set (16 KB pieces, round-robin over the grid) before it waits
        // for the routing.  Sets that turn out inactive cost idle bandwidth only.
        const unsigned long long pieces_per_set = p.pf_bytes >> 14;
        const unsigned long long total = pieces_per_set * 2ull * (unsigned long long)(p.G + p.S);
        for (unsigned long long i = (unsigned long long)blockIdx.x * 32 + lane; i < total; i += (unsigned long long)gridDim.x * 32) {
            const unsigned long long set2 = i / pieces_per_set, piece = i - set2 * pieces_per_set;
            const bm_bf16 *base = (set2 & 1) ? p.w3 : p.w1;
            const char *addr = reinterpret_cast<const char *>(base) + (set2 >> 1) * p.pf_set_bytes + (piece << 14);
            ptx::prefetch_l2_bulk(addr, 16384u);
        }
    }
    // Speculative start (DC_GEMM1, dense decode inside bm_moe_layer): with T*K >= 2 G tokens x slots nearly every set is
    // active, and a dense item needs nothing from the routing -- all T tokens times one weight tile.  So the CTAs run the
    // items of the first spec_sets sets (n_spec items, the same static round-robin) while the router and the permutation
    // are still at work, and only then wait for them and build the schedule of the remaining active sets.  The router's
    // latency (~10 us of an idle HBM) disappears behind the weight stream; a set that turns out inactive cost only
    // bandwidth that nobody else wanted.  Item numbers below n_spec are synthesised by fetch(); the first request beyond
    // makes the producer warp wait for the routing, build the schedule and release the other warps through an mbarrier.
    // The dependent grid (GEMM2) is let go only then, so "GEMM1 let GEMM2 start => the routing is complete" still holds.
    // PF_GEMM1 has the same start for the S shared experts (spec_shared): their items take all T tokens straight from x and
    // write H rows that no routed item touches, so they run while the router, the permutation and the gather pass are
    // still at work -- at BJ:configs[3] (two shared experts: 30% of the rows) that hides most of the routing chain.  The
    // kernels of that chain let their successor start before their own wait, so that this grid is resident early.
    const bool spec = (MODE == DC_GEMM1 && p.spec_sets > 0) || (MODE == PF_GEMM1 && p.spec_shared != 0);
    const int pf_units = K2 ? ((p.T + kChunkRows - 1) / kChunkRows + 1) >> 1 : (p.T + kChunkRows - 1) / kChunkRows;
    const int n_spec = !spec ? 0 : MODE == DC_GEMM1 ? p.spec_sets * p.n_wtiles : p.S * pf_units * p.n_wtiles;
    uint64_t *sched_bar = bars + kSchedBarSlot;
    if (!spec) {
        grid_dep_wait();
        if (kGemm1 && warp == 0) build_schedule(p, s_sched, cap, s_hdr);
        __syncthreads();
        sv.n_seg = s_hdr[0]; sv.total_chunks = s_hdr[1]; sv.total_pairs = s_hdr[2];
        if (threadIdx.x == 0) grid_dep_launch();
    }
    bool sched_seen = !spec;
    auto fetch = [&](int item, Item &it) -> bool {         // warp-uniform
        if ((MODE == DC_GEMM1 || MODE == PF_GEMM1) && spec) {
            if (item < n_spec) {
                if (MODE == DC_GEMM1) {
                    it.u = item / p.n_wtiles; it.wt = item - it.u * p.n_wtiles; it.ks = 0;
                    it.n = p.T; it.act_row0 = 0; it.tok0 = 0; it.perm_row0 = 0; it.h_row0 = it.u * p.T; it.shared = false;
                } else {
                    // shared expert j, (chunk unit, weight tile) in get_item's order: unit fastest
                    const int per_set = pf_units * p.n_wtiles;
                    const int j = item / per_set, local = item - j * per_set;
                    it.wt = local / pf_units;
                    int chunk = local - it.wt * pf_units;
                    if (K2) chunk = 2 * chunk + (int)rank;
                    it.n = min(kChunkRows, p.T - chunk * kChunkRows);
                    if (it.n <= 0) { it.n = 0; chunk = 0; }          // absent half of the last pair: point at real rows
                    it.u = p.G + j; it.ks = 0; it.shared = true; it.perm_row0 = 0;
                    it.tok0 = chunk * kChunkRows;
                    it.h_row0 = p.TK + j * p.T + it.tok0;
                    it.act_row0 = it.tok0;
                }
                return true;
            }
            if (!sched_seen) {
                if (warp == 0) {
                    grid_dep_wait();
                    build_schedule(p, s_sched, cap, s_hdr);
                    if (lane == 0) { grid_dep_launch(); ptx::mbar_arrive(sched_bar); }
                    __syncwarp();
                } else {
                    ptx::mbar_wait(sched_bar, 0);
                }
                sv.n_seg = s_hdr[0]; sv.total_chunks = s_hdr[1]; sv.total_pairs = s_hdr[2];
                sched_seen = true;
            }
            item -= n_spec;
        }
        return get_item<MODE, K2>(p, sv, item, it, rank);
    };

    // The producer and the MMA issuer run their loops with the WHOLE warp (warp-uniform control flow keeps
    // addresses and descriptors in uniform registers) and elect one lane for the issuing instructions: the
    // single-thread instruction stream per k-block is what paces a decode tile, so it is kept short.
    if (warp == 0) {
        // =========================== TMA producer ===========================
        int stage = 0;
        uint32_t phase = 0;
        Item it;
        int item = item0;
        int kb_first = 0;
        bool have;
        if (MODE == DC_GEMM2) {
            it = it0;
            have = have0;
            if (ptx::elect_one())
                for (int kb = 0; kb < pre; ++kb)
                    for (int kk = 0; kk < kp; ++kk)
                        for (int j = 0; j * 32 < it.n; ++j)
                            ptx::tma_load_2d(smem + (size_t)kb * stage_bytes + kk * mini + p.off_b + j * 4096, &tm_act0, &full[kb],
                                             ((it.ks * nkb + kb) * kp + kk) * kBlockK, it.act_row0 + j * 32, ptx::kEvictLast);
            __syncwarp();
            kb_first = pre;
            stage = pre;
            if (stage == n_stages) { stage = 0; phase = 1; }
        } else {
            have = fetch(item, it);
        }
        auto policy = [](int h) { return h == 0 ? ptx::kEvictFirst : (h == 1 ? ptx::kEvictNormal : ptx::kEvictLast); };
        const uint64_t pol_a = policy(p.hints / 10), pol_w = policy(p.hints % 10);
        for (; have; item += item_stride, have = fetch(item, it), kb_first = 0) {
            const CUtensorMap *tm_act = (kGemm1 && (it.shared || p.dense)) ? &tm_act1 : &tm_act0;
            const int wrow0 = it.wt * p.R;
            int kc = (it.ks * nkb + kb_first) * kp * kBlockK;
            const uint32_t stage_tx = stage_tx_of(it.n);
            for (int kb = kb_first; kb < nkb; ++kb, kc += kp * kBlockK) {
                ptx::mbar_wait(&empty[stage], phase ^ 1);
                if (K2) {
                    if (ptx::elect_one()) {
                        uint8_t *st = smem + (size_t)stage * stage_bytes;
                        if (leader) ptx::mbar_arrive_expect_tx(&full[stage], stage_tx);
                        if (!GA) ptx::tma_load_2d_pair(st, tm_act, &full[stage], kc, it.act_row0, pol_a);
                        if (MODE == PF_GEMM1)       // B rows 0-127 = the W1 tile (leader), 128-255 = the W3 tile (peer)
                            ptx::tma_load_3d_pair(st + kTileBytes16K, leader ? &tm_w0 : &tm_w1, &full[stage], kc, wrow0, it.u,
                                                  pol_w);
                        else                        // each CTA half of the 256 W2 rows
                            ptx::tma_load_3d_pair(st + kTileBytes16K, &tm_w0, &full[stage], kc, wrow0 + (int)rank * 128, it.u,
                                                  pol_w);
                    }
                } else if (ptx::elect_one()) {
                    uint8_t *st = smem + (size_t)stage * stage_bytes;
                    ptx::mbar_arrive_expect_tx(&full[stage], stage_tx);
                    if (!kDecode) {
                        // A = 128 activation rows, B = 256 weight rows (W1|W3 tiles, or one W2 tile of 256)
                        if (!GA) ptx::tma_load_2d(st, tm_act, &full[stage], kc, it.act_row0, pol_a);
                        ptx::tma_load_3d(st + kTileBytes16K, &tm_w0, &full[stage], kc, wrow0, it.u, pol_w);
                        if (MODE == PF_GEMM1)
                            ptx::tma_load_3d(st + 2 * kTileBytes16K, &tm_w1, &full[stage], kc, wrow0, it.u, pol_w);
                    } else {
                        // M side = R weight rows (streamed once from HBM), N side = the group's token rows
                        // (32-row boxes; rows past the group's within the last box are loaded and never stored)
                        for (int kk = 0; kk < kp; ++kk, st += mini) {
                            const int kcc = kc + kk * kBlockK;
                            ptx::tma_load_3d(st, &tm_w0, &full[stage], kcc, wrow0, it.u, pol_w);
                            if (MODE == DC_GEMM1)
                                ptx::tma_load_3d(st + p.wslot, &tm_w1, &full[stage], kcc, wrow0, it.u, pol_w);
                            for (int j = 0; j * 32 < it.n; ++j)
                                ptx::tma_load_2d(st + p.off_b + j * 4096, tm_act, &full[stage], kcc, it.act_row0 + j * 32,
                                                 pol_a);
                        }
                    }
                }
                __syncwarp();
                if (++stage == n_stages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        // descriptor low words: (smem address >> 4) | LBO; the high word (SBO, version, swizzle) is constant
        const uint32_t a_lo0 = ptx::smem_desc_lo(ptx::smem_u32(smem));
        const uint32_t b_off = (uint32_t)(kDecode ? p.off_b : kTileBytes16K) >> 4;
        const uint32_t stage_step = stage_bytes >> 4;
        const uint32_t w3_off = (uint32_t)p.wslot >> 4;
        uint32_t a_lo = a_lo0;
        int stage = 0;
        uint32_t phase = 0;
        int acc = 0;
        uint32_t acc_phase = 0;
        Item it;
        // K2: only the leader issues MMAs (for both CTAs); the peer's warp 1 just keeps the TMEM allocation
        for (int item = item0; (!K2 || leader) && fetch(item, it); item += item_stride) {
            const uint32_t idesc = kDecode ? ptx::make_idesc_bf16(128, (it.n + 31) & ~31)
                                           : ptx::make_idesc_bf16(K2 ? 256 : 128, 256);
            ptx::mbar_wait(&tempty[acc], acc_phase ^ 1);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * kAccCols;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(&full[stage], phase);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
                    for (int kk = 0; kk < kp; ++kk) {
                        const uint32_t a_kk = a_lo + (uint32_t)kk * (mini >> 4);
#pragma unroll
                        for (int k = 0; k < kBlockK / 16; ++k) {
                            const uint32_t accum = (kb | kk | k) ? 1u : 0u;
                            const uint32_t ko = 2 * k;             // 16 bf16 = 32 bytes = 2 descriptor units
                            if (K2)
                                ptx::mma_bf16_ss_pair(d_tmem, ptx::smem_desc(a_kk + ko), ptx::smem_desc(a_kk + b_off + ko), idesc, accum);
                            else
                                ptx::mma_bf16_ss(d_tmem, ptx::smem_desc(a_kk + ko), ptx::smem_desc(a_kk + b_off + ko), idesc, accum);
                            if (MODE == DC_GEMM1)
                                ptx::mma_bf16_ss(d_tmem + 128, ptx::smem_desc(a_kk + w3_off + ko),
                                                 ptx::smem_desc(a_kk + b_off + ko), idesc, accum);
                        }
                    }
                    if (K2) {       // the same barriers in both CTAs
                        ptx::mma_commit_pair(&empty[stage]);
                        if (kb == nkb - 1) ptx::mma_commit_pair(&tfull[acc]);
                    } else {
                        ptx::mma_commit(&empty[stage]);                  // frees the smem stage when the MMAs retire
                        if (kb == nkb - 1) ptx::mma_commit(&tfull[acc]);   // accumulator complete
                    }
                }
                __syncwarp();
                a_lo += stage_step;
                if (++stage == n_stages) { stage = 0; phase ^= 1; a_lo = a_lo0; }
            }
            if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
        }
    } else if (GA && warp >= 6 && warp < 10) {
        // =========================== gather (warps 6..9, GA) ===========================
        // Step 9 inside GEMM1: the gather threads copy the 128 rows of the item's A tile straight from x -- 128 bytes per
        // row and k-block as eight 16-byte cp.async, written in the 128B-swizzle layout TMA would have produced (16-byte
        // chunk j of row r at chunk j ^ (r & 7)); columns past D are zero-filled like TMA's out-of-bounds fill.
        // Thread g = (row group rg = g / 8, chunk j = g % 8) copies chunk j of rows rg, rg + 16, ..., rg + 112: eight
        // neighbouring lanes cover one row's 128 contiguous bytes, so a warp instruction touches 4 rows x 4 sectors
        // (one row per lane scattered every 16-byte piece into its own sector request: 2-4x slower GEMM1).
        // Completion is signalled by the hardware: cp.async.mbarrier.arrive.noinc makes the thread's arrival on the
        // stage's gfull barrier happen when its copies have landed, so the thread never waits for its own copies and
        // the whole ring depth stays in flight (a cp.async.wait_group + arrive version kept only 2-3 k-blocks in
        // flight: 3x slower with CTA pairs).  This replaces the separate gather pass (gather_kernel): A*D*4 bytes of HBM
        // traffic and a launch-wide pass less.
        const int g = (int)threadIdx.x - kThreads;
        const int j = g & 7, rg = g >> 3;
        uint32_t dst_off[8];             // row * 128 + swizzled chunk offset
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int r = rg + 16 * i;
            dst_off[i] = (uint32_t)r * 128u + ((uint32_t)(j ^ (r & 7)) << 4);
        }
        int stage = 0;
        uint32_t phase = 0;
        Item it;
        for (int item = item0; fetch(item, it); item += item_stride) {
            const bm_bf16 *src[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int r = rg + 16 * i;
                const int rr = it.n > 0 ? min(r, it.n - 1) : 0;      // rows past the chunk's: a valid row, never stored
                int tok = it.shared ? it.tok0 + rr : p.row_token[it.perm_row0 + rr];
                tok = tok < 0 ? 0 : (tok >= p.T ? p.T - 1 : tok);
                src[i] = p.x + (size_t)tok * p.D + j * 8;
            }
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(&empty[stage], phase ^ 1);
                const uint32_t dst = ptx::smem_u32(smem + (size_t)stage * stage_bytes);
                const int kc = kb * kBlockK;
                const bool in = kc + j * 8 < p.D;                    // columns past D: zero fill, like TMA
#pragma unroll
                for (int i = 0; i < 8; ++i) ptx::cp_async_16(dst + dst_off[i], src[i] + (in ? kc : 0), in ? 16u : 0u);
                ptx::cp_async_mbar_arrive_noinc(&gfull[stage]);
                if (++stage == n_stages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (GA && warp >= 10) {
        // =========================== gather relays (warps 10..15, GA) ===========================
        // Relay w owns the ring stages s = w, w + 6, ... (one relay per stage keeps the waits on a stage's barrier in
        // phase order): for each k-block of such a stage it waits until all 128 gather threads' copies
        // have landed, fences them towards the async proxy (tcgen05.mma reads shared memory through it) and
        // arrives on the stage's full barrier -- the leader's under K2.  Fence + cluster-scope arrive cost one relay
        // about a k-block's time (ncu: the single relay of the first version was the kernel's bottleneck with CTA
        // pairs, GEMM1 3x slower), so up to six work side by side.
        const uint32_t full_base = K2 ? ptx::mapa_u32(&full[0], 0) : ptx::smem_u32(&full[0]);
        const int rw = warp - 10;
        int n = 0;                       // running k-block number of this CTA
        Item it;
        for (int item = item0; fetch(item, it); item += item_stride) {
            for (int kb = 0; kb < nkb; ++kb, ++n) {
                const int stage = n % n_stages;
                if (stage % kGatherRelays != rw) continue;
                ptx::mbar_wait(&gfull[stage], (uint32_t)(n / n_stages) & 1u);
                if (lane == 0) {
                    ptx::fence_proxy_async_smem();
                    if (K2) ptx::mbar_arrive_cluster(full_base + (uint32_t)stage * 8u);
                    else ptx::mbar_arrive(&full[stage]);
                }
                __syncwarp();
            }
        }
    } else if (!GA || warp < 6) {
        // =========================== epilogue (warps 2..5) ===========================
        const int q = warp & 3;                      // TMEM lane quarter this warp may read
        const int row = q * 32 + lane;               // accumulator row (M index) owned by this thread
        int acc = 0;
        uint32_t acc_phase = 0;
        Item it;
        for (int item = item0; fetch(item, it); item += item_stride) {
            // FC: token, gate weight and source count of this thread's rows are fetched BEFORE the wait for the
            // accumulator (two dependent global loads hidden behind the item's main loop).
            // PF_GEMM2: row `row` of the chunk (index 0); DC_GEMM2: chunk rows lane, lane + 32, ... (the columns).
            int tokr[4] = {-1, -1, -1, -1};
            float gwr[4] = {0.f, 0.f, 0.f, 0.f};
            int nsrcr[4] = {0, 0, 0, 0};
            if (FC || MODE == DC_GEMM2) {
#pragma unroll
                for (int j = 0; j < (MODE == DC_GEMM2 ? 4 : 1); ++j) {
                    const int r = MODE == DC_GEMM2 ? j * 32 + lane : row;
                    if (r < it.n && p.dense && !it.shared) {
                        // dense decode: column r is token tok0 + r; it counts only if the token was routed to this set
                        const int tok = it.tok0 + r;
                        if (tok < p.T) {
                            const int ns = min(max(p.n_slots[tok], 0), p.K);
                            for (int sl = 0; sl < ns; ++sl)
                                if (p.group_ids[(size_t)tok * p.K + sl] == it.u) {
                                    tokr[j] = tok;
                                    gwr[j] = p.gate_w[(size_t)tok * p.K + sl];
                                }
                        }
                    } else if (r < it.n) {
                        int tok, slot = 0;
                        if (it.shared) {
                            tok = it.tok0 + r;
                        } else {
                            tok = p.row_token[it.perm_row0 + r];
                            slot = p.row_slot[it.perm_row0 + r];
                        }
                        if (tok >= 0 && tok < p.T && slot >= 0 && slot < p.K) {
                            tokr[j] = tok;
                            gwr[j] = it.shared ? 1.0f : p.gate_w[(size_t)tok * p.K + slot];
                            if (MODE == PF_GEMM2) nsrcr[j] = min(max(p.n_slots[tok], 0), p.K) + p.S;
                        }
                    }
                }
            }
            ptx::mbar_wait(&tfull[acc], acc_phase);
            ptx::tc_fence_after();
            const uint32_t t_addr = tmem_base + acc * kAccCols + ((uint32_t)(q * 32) << 16);
            bool released = false;
            auto release_acc = [&]() {              // hand the accumulator stage back to the MMA issuer
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (K2) ptx::mbar_arrive_cluster(ptx::mapa_u32(&tempty[acc], 0));      // the leader's barrier
                    else ptx::mbar_arrive(&tempty[acc]);
                }
                released = true;
            };

            if (MODE == PF_GEMM1) {
                // row = token row of the chunk; columns [0,128) = W1 products, [128,256) = W3 products
                const bool row_ok = row < it.n;
                const int f0 = it.wt * 128;
                bm_bf16 *hrow = p.h + (size_t)(it.h_row0 + row) * p.F + f0;
#pragma unroll 1
                for (int c = 0; c < 128; c += 16) {
                    uint32_t a[16], b[16];
                    ptx::tmem_ld_x16(t_addr + c, a);
                    ptx::tmem_ld_x16(t_addr + 128 + c, b);
                    ptx::tmem_ld_wait();
                    uint32_t o[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        o[i] = pack_bf16x2(silu_mul(__uint_as_float(a[2 * i]), __uint_as_float(b[2 * i])),
                                           silu_mul(__uint_as_float(a[2 * i + 1]), __uint_as_float(b[2 * i + 1])));
                    if (row_ok) {
                        if (f0 + c + 8 <= p.F) *reinterpret_cast<uint4 *>(hrow + c) = make_uint4(o[0], o[1], o[2], o[3]);
                        if (f0 + c + 16 <= p.F) *reinterpret_cast<uint4 *>(hrow + c + 8) = make_uint4(o[4], o[5], o[6], o[7]);
                    }
                }
            } else if (MODE == PF_GEMM2 && FC) {
                // row = token row of the chunk; columns = 256 output features d0..d0+255 of y_r = H_r . W2[u]^T.
                // gw * y_r is added into out_acc[tok, d0..]: 32 columns at a time the accumulator leaves TMEM with one
                // row per lane, is scaled, transposed through the warp's shared-memory stage (32 rows x 32 fp32,
                // 16-byte units xor-swizzled by the row) and goes out as red.global.add.v4.f32, every instruction
                // 4 rows x 128 contiguous bytes (whole sectors) -- the "coalesced 128-bit" scatter of north_star (4).
                const int d0 = it.wt * 256;
                const int n_dt = (p.D + 255) >> 8;
                float4 *stg = reinterpret_cast<float4 *>(epi_stage + (size_t)q * kEpiStageBytes);
                const int rl = lane >> 3, ul = lane & 7;        // read phase: row (mod 4) and 16-byte unit of this lane
                float *rptr[8];                                 // accumulator row of chunk row 4j + rl (nullptr: no row)
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int tk = __shfl_sync(kFullMask, tokr[0], 4 * j + rl);
                    rptr[j] = tk >= 0 ? p.out_acc + (size_t)tk * p.D + d0 + 4 * ul : nullptr;
                }
                const float gw = gwr[0];
#pragma unroll 1
                for (int c = 0; c < 256; c += 32) {
                    if (d0 + c >= p.D) break;                   // ragged last tile: whole 32-column steps past D
                    uint32_t v[32];
                    ptx::tmem_ld_x32(t_addr + c, v);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        stg[lane * 8 + (u ^ (lane & 7))] =
                            make_float4(gw * __uint_as_float(v[4 * u]), gw * __uint_as_float(v[4 * u + 1]),
                                        gw * __uint_as_float(v[4 * u + 2]), gw * __uint_as_float(v[4 * u + 3]));
                    __syncwarp();
                    if (d0 + c + 4 * ul + 4 <= p.D) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int r = 4 * j + rl;
                            if (rptr[j]) {
                                const float4 x = stg[r * 8 + (ul ^ (r & 7))];
                                ptx::red_add_v4_f32(rptr[j] + c, x.x, x.y, x.z, x.w);
                            }
                        }
                    }
                    __syncwarp();
                }
                release_acc();                                  // the MMA of the item after next may start
                // tickets: one arrival per (token, 256-column piece) and source row
                __threadfence();
                __syncwarp();
                bool done = false;
                if (tokr[0] >= 0)
                    done = atomicAdd(p.tickets + (size_t)tokr[0] * n_dt + it.wt, 1) == nsrcr[0] - 1;
                unsigned dm = __ballot_sync(kFullMask, done);
                if (dm) __threadfence();
                // completed pieces (this row was the token's last source): lane l owns columns d0 + 8l .. + 7 of every
                // one; four pieces per round so that their eight loads per lane are in flight together
                const int d = d0 + lane * 8;
                const bool d_in = d + 8 <= p.D;
                while (dm) {
                    int tk[4];
                    float4 a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int r = dm ? __ffs(dm) - 1 : -1;
                        if (dm) dm &= dm - 1;
                        tk[i] = r >= 0 ? __shfl_sync(kFullMask, tokr[0], r) : -1;       // (r is warp-uniform)
                        if (tk[i] >= 0 && d_in) {
                            const float4 *src = reinterpret_cast<const float4 *>(p.out_acc + (size_t)tk[i] * p.D + d);
                            a[i] = __ldcg(src);
                            b[i] = __ldcg(src + 1);
                        }
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        if (tk[i] < 0) continue;
                        if (d_in) {
                            float4 *src = reinterpret_cast<float4 *>(p.out_acc + (size_t)tk[i] * p.D + d);
                            if (p.out_f32) {
                                float4 *o = reinterpret_cast<float4 *>(p.out_f32 + (size_t)tk[i] * p.D + d);
                                o[0] = a[i]; o[1] = b[i];
                            } else {
                                *reinterpret_cast<uint4 *>(p.out + (size_t)tk[i] * p.D + d) =
                                    make_uint4(pack_bf16x2(a[i].x, a[i].y), pack_bf16x2(a[i].z, a[i].w),
                                               pack_bf16x2(b[i].x, b[i].y), pack_bf16x2(b[i].z, b[i].w));
                            }
                            src[0] = make_float4(0.f, 0.f, 0.f, 0.f);
                            src[1] = make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                        if (lane == 0) p.tickets[(size_t)tk[i] * n_dt + it.wt] = 0;
                    }
                }
            } else if (MODE == PF_GEMM2) {
                // row = token row of the chunk; columns = 256 output features d0..d0+255 of y_r = H_r . W2[u]^T.
                // y is stored as bf16 rows (same row numbering as H); combine_kernel applies the gate weights and
                // sums a token's rows in slot order.  The accumulator leaves TMEM with one row per lane; a
                // per-warp shared-memory transpose (32 rows x 64 bf16 columns, 16-byte units xor-swizzled by
                // the row) turns that into row-contiguous pieces, so every 128-bit store instruction of a warp
                // writes 4 rows x 128 contiguous bytes (whole L2 lines) instead of 32 scattered pieces.
                const int d0 = it.wt * 256;
                const int n_q = it.n - q * 32;                     // valid rows of this warp's quarter
                uint4 *stg = reinterpret_cast<uint4 *>(epi_stage + (size_t)q * kEpiStageBytes);
                const int rl = lane >> 3, ul = lane & 7;        // read phase: row (mod 4) and 16-byte unit of this lane
                const size_t yrow0 = p.y_tm ? (size_t)(it.tok0 + q * 32) * p.S + (size_t)(it.u - p.G) : (size_t)(it.h_row0 + q * 32);
                const size_t yrs = p.y_tm ? (size_t)p.S * p.D : (size_t)p.D;        // elements between consecutive chunk rows
                bm_bf16 *ybase = p.y + yrow0 * p.D + d0 + 8 * ul;
#pragma unroll 1
                for (int c = 0; c < 256; c += 64) {
                    uint32_t v[32], w[32];
                    ptx::tmem_ld_x32(t_addr + c, v);
                    ptx::tmem_ld_x32(t_addr + c + 32, w);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        stg[lane * 8 + (u ^ (lane & 7))] =
                            make_uint4(pack_bf16x2(__uint_as_float(v[8 * u]), __uint_as_float(v[8 * u + 1])),
                                       pack_bf16x2(__uint_as_float(v[8 * u + 2]), __uint_as_float(v[8 * u + 3])),
                                       pack_bf16x2(__uint_as_float(v[8 * u + 4]), __uint_as_float(v[8 * u + 5])),
                                       pack_bf16x2(__uint_as_float(v[8 * u + 6]), __uint_as_float(v[8 * u + 7])));
                        stg[lane * 8 + ((u + 4) ^ (lane & 7))] =
                            make_uint4(pack_bf16x2(__uint_as_float(w[8 * u]), __uint_as_float(w[8 * u + 1])),
                                       pack_bf16x2(__uint_as_float(w[8 * u + 2]), __uint_as_float(w[8 * u + 3])),
                                       pack_bf16x2(__uint_as_float(w[8 * u + 4]), __uint_as_float(w[8 * u + 5])),
                                       pack_bf16x2(__uint_as_float(w[8 * u + 6]), __uint_as_float(w[8 * u + 7])));
                    }
                    __syncwarp();
                    if (d0 + c + 8 * ul + 8 <= p.D) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int r = 4 * j + rl;
                            if (r < n_q)
                                *reinterpret_cast<uint4 *>(ybase + (size_t)r * yrs + c) = stg[r * 8 + (ul ^ (r & 7))];
                        }
                    }
                    __syncwarp();
                }
            } else if (MODE == DC_GEMM1) {
                // row = weight row f (R rows per tile); columns [0,npad) = W1 products per token,
                // [128, 128+npad) = W3 products
                const int f = it.wt * p.R + row;
                const bool f_ok = row < p.R && f < p.F;
                const int npad = (it.n + 31) & ~31;
                bm_bf16 *hcol = p.h + (size_t)it.h_row0 * p.F + f;
#pragma unroll 1
                for (int c = 0; c < npad; c += 16) {
                    uint32_t a[16], b[16];
                    ptx::tmem_ld_x16(t_addr + c, a);
                    ptx::tmem_ld_x16(t_addr + 128 + c, b);
                    ptx::tmem_ld_wait();
                    if (f_ok) {
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (c + i < it.n)
                                hcol[(size_t)(c + i) * p.F] =
                                    (bm_bf16)f32_to_bf16_bits(silu_mul(__uint_as_float(a[i]), __uint_as_float(b[i])));
                    }
                }
            } else {
                // DC_GEMM2: row = output feature d; columns = token rows of the chunk; partial over this K split.
                // Token and gate weight of chunk rows lane, lane + 32, ... were fetched above (one dependent-load
                // chain per item instead of one per token); the loop broadcasts them with shuffles.
                const int d = it.wt * p.R + row;
                const bool d_ok = row < p.R && d < p.D;
                float *ocol = p.out_acc + d;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (j * 32 < it.n) {                 // warp-uniform
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            const int c = j * 32 + hh * 16;
                            if (c < it.n) {              // warp-uniform
                                uint32_t v[16];
                                ptx::tmem_ld_x16(t_addr + c, v);
                                ptx::tmem_ld_wait();
#pragma unroll
                                for (int i = 0; i < 16; ++i) {
                                    const int tok = __shfl_sync(0xffffffffu, tokr[j], hh * 16 + i);
                                    const float gw = __shfl_sync(0xffffffffu, gwr[j], hh * 16 + i);
                                    if (tok >= 0 && d_ok)
                                        ptx::red_add_f32(ocol + (size_t)tok * p.D, gw * __uint_as_float(v[i]));
                                }
                            }
                        }
                    }
                }
                release_acc();
                // FC: tickets, piece = (weight tile, 32-row quarter q) over ALL tokens (a decode batch is small); every item
                // (chunk of any segment, K split) on this weight tile arrives once, total_chunks * ksplit in all.  The warp
                // that completes a piece finishes it for every token.  Quarters without a valid output row take no tickets.
                // (Taking all tickets once at the end of the kernel instead -- one fence per warp -- was measured slower:
                // every piece then completes in the kernel's tail.)  Without FC a finalize kernel rounds and clears.
                if (FC && q * 32 < p.R && it.wt * p.R + q * 32 < p.D) {      // warp-uniform
                    __threadfence();
                    __syncwarp();
                    int last = 0;
                    if (lane == 0) last = atomicAdd(p.tickets + it.wt * 4 + q, 1) == sv.total_chunks * p.ksplit - 1;
                    last = __shfl_sync(kFullMask, last, 0);
                    if (last) {
                        // lane = (token sub-row lane / 8, four output features 4 * (lane % 8) .. + 3): R is a multiple of 4
                        // on this kernel, so a 32-feature quarter is made of whole 16-byte pieces; 64 tokens per round
                        __threadfence();
                        const int dq = it.wt * p.R + q * 32 + 4 * (lane & 7);
                        const bool q_ok = q * 32 + 4 * (lane & 7) < p.R && dq < p.D;
                        for (int t0 = lane >> 3; t0 < p.T; t0 += 64) {
                            float4 v[16];
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                const int t = t0 + 4 * i;
                                v[i] = (q_ok && t < p.T) ? __ldcg(reinterpret_cast<const float4 *>(p.out_acc + (size_t)t * p.D + dq))
                                                         : make_float4(0.f, 0.f, 0.f, 0.f);
                            }
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                const int t = t0 + 4 * i;
                                if (q_ok && t < p.T) {
                                    const size_t o = (size_t)t * p.D + dq;
                                    if (p.out_f32) *reinterpret_cast<float4 *>(p.out_f32 + o) = v[i];
                                    else *reinterpret_cast<uint2 *>(p.out + o) = make_uint2(pack_bf16x2(v[i].x, v[i].y), pack_bf16x2(v[i].z, v[i].w));
                                    *reinterpret_cast<float4 *>(p.out_acc + o) = make_float4(0.f, 0.f, 0.f, 0.f);
                                }
                            }
                        }
                        if (lane == 0) p.tickets[it.wt * 4 + q] = 0;
                    }
                }
            }
            if (!released) release_acc();
            if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (K2) ptx::cluster_sync_all();      // the peer's shared memory, barriers and TMEM stay alive until both are done
    if (warp == 1) {
        ptx::tc_fence_after();
        if (K2) ptx::tmem_dealloc_pair(tmem_base, kTmemCols); else ptx::tmem_dealloc(tmem_base, kTmemCols);
    }
}

// -------------------------------------------------------------------------------------------------
// gather (step 9, only for the kernels that take their token rows by TMA from xs: CTA-pair prefill tiles and the
// decode kernel beyond 64 tokens): one warp per permuted row.  (A tile::gather4 producer in GEMM1 was measured
// instead of this pass: ~12 cycles per 128-byte row made GEMM1 3x slower.)
// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
gather_kernel(const bm_bf16 *__restrict__ x, int T, int D, int K, int G, const int32_t *__restrict__ offsets,
              const int32_t *__restrict__ row_token, bm_bf16 *__restrict__ xs) {
    grid_dep_launch();     // GEMM1 may be resident (and at work on the shared experts) before this pass has run; it waits for it
    grid_dep_wait();
    const int A = min(max(offsets[G], 0), T * K);
    const int warps = (gridDim.x * blockDim.x) >> 5;
    const int lane = threadIdx.x & 31;
    const int vec = D / 8;
    for (int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; r < A; r += warps) {
        int t = row_token[r];
        t = t < 0 ? 0 : (t >= T ? T - 1 : t);
        const uint4 *src = reinterpret_cast<const uint4 *>(x + (size_t)t * D);
        uint4 *dst = reinterpret_cast<uint4 *>(xs + (size_t)r * D);
        for (int i = lane; i < vec; i += 32) dst[i] = __ldg(src + i);
    }
}

// out = bf16(acc) (or a copy into out_f32).  clear != 0: acc is the zero region's accumulator and is put back to zero
// (decode beyond 64 tokens, where the in-kernel finish costs more than this pass).
__global__ void __launch_bounds__(256)
finalize_kernel(float *__restrict__ acc, bm_bf16 *__restrict__ out, float *__restrict__ out_f32, size_t n8, int clear) {
    grid_dep_wait();
    grid_dep_launch();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
        float4 *src = reinterpret_cast<float4 *>(acc) + 2 * i;
        const float4 a = src[0], b = src[1];
        if (out_f32) {
            reinterpret_cast<float4 *>(out_f32)[2 * i] = a;
            reinterpret_cast<float4 *>(out_f32)[2 * i + 1] = b;
        } else {
            reinterpret_cast<uint4 *>(out)[i] = make_uint4(pack_bf16x2(a.x, a.y), pack_bf16x2(a.z, a.w),
                                                           pack_bf16x2(b.x, b.y), pack_bf16x2(b.z, b.w));
        }
        if (clear) { src[0] = make_float4(0.f, 0.f, 0.f, 0.f); src[1] = make_float4(0.f, 0.f, 0.f, 0.f); }
    }
}

// Prefill combine (F2): out[t] = sum_{s < n_slots[t]} gate_w[t,s] * y[slot_row[t,s]]  (slot order)
//                               + sum_{j < S} y[TK + j*T + t]                          (shared experts)
// fp32 accumulation in a fixed order -> deterministic.  A warp item = (token, column slice); lane s parks the
// row pointer and weight of source s (K + S <= 32) in shared memory once per item, then the warp walks its
// columns 16 bytes per lane (512 contiguous bytes per row and step), four source rows in flight; the eight
// products of a 16-byte chunk are four FFMA2 (the weight is the broadcast operand).  (The first version re-read
// row and weight with three shuffles per source and chunk: 67 instructions per 512-byte row load, issue-bound
// at 4 TB/s.)
constexpr int kCombineBatch = 4;     // source rows in flight per lane (8 measured slower: 79 -> 117 us at BJ:configs[2])

__device__ __forceinline__ void fma2_bcast(float &d0, float &d1, float x, float w0, float w1) {
    uint64_t a, b, c;
    asm("mov.b64 %0, {%1, %1};" : "=l"(a) : "f"(x));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(w0), "f"(w1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(d0), "f"(d1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(c));
}

__global__ void __launch_bounds__(256)
combine_kernel(const bm_bf16 *__restrict__ y, int T, int D, int K, int S, const int32_t *__restrict__ n_slots,
               const int32_t *__restrict__ slot_row, const float *__restrict__ gate_w, bm_bf16 *__restrict__ out,
               float *__restrict__ out_f32, int split) {
    __shared__ const uint4 *s_src[8][32];     // per warp: row pointers of the item's sources (nullptr: skip)
    __shared__ float s_gw[8][32];
    grid_dep_wait();
    grid_dep_launch();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int vec = D / 8;
    const size_t TK = (size_t)T * K;
    const int warps = (gridDim.x * blockDim.x) >> 5;
    // a warp item = (token, column slice); split > 1 spreads a token's columns over several warps (small T)
    const long long items = (long long)T * split;
    for (long long item = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; item < items; item += warps) {
        const int t = (int)(item / split), sl = (int)(item - (long long)t * split);
        const int n = min(max(n_slots[t], 0), K);
        const int n_src = n + S;
        const uint4 *my_src = nullptr;                           // nullptr: skip (invalid slot_row)
        float my_gw = 1.0f;
        if (lane < n) {
            const int r = slot_row[(size_t)t * K + lane];
            if (r >= 0 && (size_t)r < TK) my_src = reinterpret_cast<const uint4 *>(y + (size_t)r * D);
            my_gw = gate_w[(size_t)t * K + lane];
        } else if (lane < n_src) {
            my_src = reinterpret_cast<const uint4 *>(y + (TK + (size_t)(lane - n) * T + t) * D);
        }
        __syncwarp();                                            // the previous item's readers are done
        s_src[w][lane] = my_src;
        s_gw[w][lane] = my_src ? my_gw : 0.0f;
        __syncwarp();
        for (int c0 = sl * 32; c0 < vec; c0 += 32 * split) {
            const int c = c0 + lane;
            const bool col_ok = c < vec;
            float acc[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[e] = 0.0f;
            for (int s0 = 0; s0 < n_src; s0 += kCombineBatch) {
                uint4 v[kCombineBatch];
                float gw[kCombineBatch];
#pragma unroll
                for (int q = 0; q < kCombineBatch; ++q) {
                    const int src = min(s0 + q, 31);
                    const uint4 *ptr = s_src[w][src];            // broadcast reads
                    gw[q] = s_gw[w][src];
                    const bool ok = s0 + q < n_src && ptr != nullptr && col_ok;
                    v[q] = ok ? ptr[c] : make_uint4(0, 0, 0, 0);
                }
#pragma unroll
                for (int q = 0; q < kCombineBatch; ++q) {
                    if (s0 + q < n_src) {                        // warp-uniform; skipped sources add nothing (weight 0, value 0)
                        fma2_bcast(acc[0], acc[1], gw[q], bf16_lo(v[q].x), bf16_hi(v[q].x));
                        fma2_bcast(acc[2], acc[3], gw[q], bf16_lo(v[q].y), bf16_hi(v[q].y));
                        fma2_bcast(acc[4], acc[5], gw[q], bf16_lo(v[q].z), bf16_hi(v[q].z));
                        fma2_bcast(acc[6], acc[7], gw[q], bf16_lo(v[q].w), bf16_hi(v[q].w));
                    }
                }
            }
            if (!col_ok) continue;
            if (out_f32) {      // tensor-parallel partial: the fp32 sums, rounded after the cross-rank reduction
                float4 *o = reinterpret_cast<float4 *>(out_f32 + (size_t)t * D + (size_t)c * 8);
                o[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
                o[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
            } else {
                *reinterpret_cast<uint4 *>(out + (size_t)t * D + (size_t)c * 8) =
                    make_uint4(pack_bf16x2(acc[0], acc[1]), pack_bf16x2(acc[2], acc[3]), pack_bf16x2(acc[4], acc[5]),
                               pack_bf16x2(acc[6], acc[7]));
            }
        }
    }
}

// -------------------------------------------------------------------------------------------------
// host: tensor maps
// -------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
    return fn;
}

// Tensor maps depend only on (base pointer, shape, box, swizzle), and a serving loop calls the layer with the same
// buffers over and over, so encoded maps are kept in a small direct-mapped cache instead of being re-encoded on the
// host in every call (eight cuTensorMapEncodeTiled calls were ~5 us of host time per layer call).  An entry is never
// stale: its content is a pure function of its key.
struct MapKey {
    const void *base;
    uint64_t d0, d1, d2;        // cols, rows, sets (d2 = 0: 2-D)
    uint32_t box_cols, box_rows, swizzle;
    bool operator==(const MapKey &o) const {
        return base == o.base && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && box_cols == o.box_cols &&
               box_rows == o.box_rows && swizzle == o.swizzle;
    }
};
struct MapEntry { MapKey key; CUtensorMap map; bool valid; };
constexpr int kMapCacheSize = 256;
MapEntry g_map_cache[kMapCacheSize];
std::mutex g_map_mutex;

bool encode_map(CUtensorMap *m, const MapKey &k) {
    uint64_t h = reinterpret_cast<uintptr_t>(k.base) * 0x9E3779B97F4A7C15ull;
    h ^= (k.d0 * 31 + k.d1) * 0xC2B2AE3D27D4EB4Full + k.d2 * 0x165667B19E3779F9ull + k.box_cols * 131 + k.box_rows * 7 + k.swizzle;
    MapEntry &e = g_map_cache[(h >> 24) % kMapCacheSize];
    std::lock_guard<std::mutex> lock(g_map_mutex);
    if (e.valid && e.key == k) { *m = e.map; return true; }
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    const int rank = k.d2 ? 3 : 2;
    cuuint64_t dims[3] = {k.d0, k.d1, k.d2};
    cuuint64_t strides[2] = {k.d0 * sizeof(bm_bf16), k.d1 * k.d0 * sizeof(bm_bf16)};
    cuuint32_t box[3] = {k.box_cols, k.box_rows, 1};
    cuuint32_t es[3] = {1, 1, 1};
    if (enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, const_cast<void *>(k.base), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, k.swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    e.key = k; e.map = *m; e.valid = true;
    return true;
}

// [rows, cols] bf16 row-major, box = box_rows x 64 columns, 128B swizzle
bool make_map_2d(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    return encode_map(m, MapKey{base, cols, rows, 0, kBlockK, box_rows, 1});
}

// [n, rows, cols] bf16, box = 1 x box_rows x 64
bool make_map_3d(CUtensorMap *m, const void *base, uint64_t n, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    return encode_map(m, MapKey{base, cols, rows, n, kBlockK, box_rows, 1});
}

// Decode tiling: rows-per-tile R in [32,128] and the K-split count, chosen with a small time model of the
// static round-robin schedule (all figures measured on B200):
//   * a k-block iteration costs at least t0 whatever R is -- the swap-AB MMA reads a full M=128 A tile
//     from shared memory per instruction, so 4 (GEMM2) or 8 (GEMM1) MMAs per k-block take ~0.30-0.37 us;
//   * a wave of `act` concurrent items moves act * item_bytes at the chip's HBM rate, and one SM cannot
//     pull more than ~0.1 MB/us on its own;
//   * items / SMs full waves plus one partial wave.
// Small R (many equal items, perfect wave count) used to win the old "wave occupancy" score and lost up to
// 40% in practice to the per-k-block floor; large R wins whenever the HBM time of a wave covers it.
double decode_time_model(int wrows, int kblocks, int n_seg, int R, int ks, int mats, int sms) {
    const double kChipBytesPerUs = 6.5e6, kSmBytesPerUs = 0.1e6;
    const double t0 = mats == 2 ? 0.37 : 0.30;
    const int tiles = (wrows + R - 1) / R;
    const long long items = (long long)tiles * n_seg * ks;
    const int kbi = kblocks / ks;
    const double b_item = (double)R * 128.0 * mats * kbi;
    const double t_issue = kbi * t0;
    auto wave = [&](double act) {
        double t = t_issue;
        if (b_item * act / kChipBytesPerUs > t) t = b_item * act / kChipBytesPerUs;
        if (b_item / kSmBytesPerUs > t) t = b_item / kSmBytesPerUs;
        return t;
    };
    const long long full = items / sms, rem = items % sms;
    double t = (double)full * wave((double)sms) + (rem ? wave((double)rem) : 0.0);
    // split-K: every split adds its own fp32 reductions in the epilogue and a k-loop ramp per (shorter) item -- measured at
    // D = 2048, F = 1408, T = 16, one split / two: G = 60 112.6 / 116.4 us, G = 30 74.4 / 79.1, G = 15 48.8 / 52.8
    return t * (1.0 + 0.05 * (ks - 1));
}

void choose_decode_tiling(int wrows, int kblocks, int n_seg, bool allow_split, int mats, int sms, int *R_out,
                          int *ks_out) {
    double best = 1e30;
    int bestR = 128, bestKs = 1;
    const int max_ks = allow_split ? 16 : 1;
    int rmax = opt(OPT_DC_RMAX);
    rmax = rmax < 32 ? 32 : (rmax > 128 ? 128 : rmax);
    const int ks_force = allow_split ? opt(OPT_DC_KS_FORCE) : 0;
    for (int ks = 1; ks <= max_ks; ++ks) {
        if (ks > 1 && (kblocks % ks != 0 || kblocks / ks < 4)) continue;
        if (ks_force > 0 && ks != ks_force && kblocks % ks_force == 0 && kblocks / ks_force >= 4) continue;
        for (int R = rmax; R >= 32; --R) {
            if (mats == 1 && (R & 3)) continue;      // GEMM2: whole 16-byte pieces per 32-row quarter (the fused finish)
            const double t = decode_time_model(wrows, kblocks, n_seg, R, ks, mats, sms);
            if (t < best * 0.99) { best = t; bestR = R; bestKs = ks; }   // within 1%: keep the larger tile
        }
    }
    // Long K (Mixtral's F = 14336: 224 k-blocks): the model is blind to the ramp and tail of few long items --
    // measured at BJ:configs[1], GEMM2 83.3 us with one split, 80.1 us with four (81.3 with two, 80.7 with eight).
    if (allow_split && ks_force <= 0 && bestKs == 1 && kblocks >= 128 && kblocks % 4 == 0) bestKs = 4;
    *R_out = bestR;
    *ks_out = bestKs;
}

size_t sched_smem_bytes(int seg_cap) { return ((size_t)5 * seg_cap * sizeof(int32_t) + 255) & ~(size_t)255; }

void ring_geometry(bool decode, bool gemm1, int T, GemmParams *p, bool pair = false) {
    p->tail_pad = 0;
    if (!decode) {
        p->stage_bytes = (pair ? 2 : 3) * kTileBytes16K;      // a CTA of a pair stages half of the B rows
        p->off_b = kTileBytes16K;
        p->wslot = kTileBytes16K;
    } else {
        // a stage = the weight tile(s), R rows x 128 B each (slot rounded up to the 1024-byte swizzle atom), and
        // room for the largest token chunk (rows padded to 32).  An M=128 MMA reads 16 KB from a tile base
        // whatever R is (rows >= R give accumulator rows that are never stored), so the last tile of the last
        // stage needs that much addressable shared memory behind it: tail_pad.
        const int rows = T < kChunkRows ? T : kChunkRows;
        const int tok_bytes = ((rows + 31) & ~31) * 128;
        p->wslot = (p->R * 128 + 1023) & ~1023;
        p->off_b = (gemm1 ? 2 : 1) * p->wslot;
        p->mini_bytes = p->off_b + tok_bytes;
        const int kp_opt = opt(OPT_DC_KPACK);
        p->kpack = (kp_opt >= 1 && kp_opt <= 2 ? kp_opt : 2);
        if (p->kblocks % p->kpack != 0) p->kpack = 1;
        p->stage_bytes = p->kpack * p->mini_bytes;
        const int behind = p->wslot + tok_bytes;
        p->tail_pad = behind >= kTileBytes16K ? 0 : kTileBytes16K - behind;
    }
    const size_t fixed = (decode ? 0 : kSmemEpi) + sched_smem_bytes(p->seg_cap) + (size_t)p->tail_pad;
    if (decode && p->kpack == 2 && (kSmemRing - fixed) / (size_t)p->stage_bytes < 3) {     // keep at least a 3-deep ring
        p->kpack = 1;
        p->stage_bytes = p->mini_bytes;
    }
    int st = (int)((kSmemRing - fixed) / (size_t)p->stage_bytes);
    const int cap = opt(decode ? OPT_DC_STAGES : OPT_PF_STAGES);
    if (st > cap) st = cap;
    if (st > kMaxStages) st = kMaxStages;
    if (st < 2) st = 2;
    p->stages = st;
}

template <int MODE, bool K2 = false, bool GA = false, bool FC = false>
cudaError_t launch_gemm(const CUtensorMap &a0, const CUtensorMap &a1, const CUtensorMap &w0, const CUtensorMap &w1,
                        const GemmParams &p, cudaStream_t stream) {
    auto kern = gemm_kernel<MODE, K2, GA, FC>;
    constexpr int kBlock = kThreads + (GA ? kGatherThreads : 0);
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(kern), kSmemMax); ea != cudaSuccess) return ea;
    constexpr int kid = (MODE == PF_GEMM1 || MODE == DC_GEMM1) ? BM_KERNEL_GEMM1 : BM_KERNEL_GEMM2;
    const size_t smem = 1024 + (size_t)p.stages * p.stage_bytes + kSmemBars + (MODE == PF_GEMM2 ? kSmemEpi : 0) +
                        sched_smem_bytes(p.seg_cap) + (size_t)p.tail_pad;
    profile_begin(kid, stream);
    cudaError_t e;
    if (!K2) {
        e = launch_kernel(kern, dim3(num_sms()), dim3(kBlock), smem, stream, a0, a1, w0, w1, p);
    } else {
        // CTA pairs: clusters of two CTAs (one TPC each), one pair per two SMs
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(num_sms() & ~1); cfg.blockDim = dim3(kBlock); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = pdl_enabled() ? 2 : 1;
        count_launch();
        e = cudaLaunchKernelEx(&cfg, kern, a0, a1, w0, w1, p);
    }
    profile_end(kid, stream);
    return e;
}

}  // namespace

// [rows, cols] bf16 row-major, box = box_rows x box_cols, no swizzle (rows of a box are contiguous in shared
// memory); out-of-bounds elements are zero-filled.  Used by the router's slab ring.
bool make_map_3d_sw128(CUtensorMap *m, const void *base, uint64_t n, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    return make_map_3d(m, base, n, rows, cols, box_rows);
}

bool make_map_2d_sw128(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    return make_map_2d(m, base, rows, cols, box_rows);
}

bool make_map_2d_plain(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows,
                       uint32_t box_cols) {
    return encode_map(m, MapKey{base, cols, rows, 0, box_cols, box_rows, 0});
}

static cudaError_t launch_combine_raw(const ForwardArgs &a, cudaStream_t stream) {
    // one warp per token; with few tokens a token's 32-chunk column slices go to different warps
    const int n_slices = (a.D / 8 + 31) / 32;
    int split = 1;
    while (split < n_slices && (long long)a.T * split < (long long)num_sms() * opt(OPT_COMBINE_WARPS)) split *= 2;   // fill the SMs' warp slots
    if (split > n_slices) split = n_slices;
    const long long items = (long long)a.T * split;
    return launch_kernel(combine_kernel, dim3((unsigned)std::min<long long>((items + 7) / 8, (long long)num_sms() * 8)),
                         dim3(256), 0, stream, (const bm_bf16 *)a.y, a.T, a.D, a.K, a.S,
                         (const int32_t *)a.r.n_slots, (const int32_t *)a.r.slot_row, (const float *)a.r.gate_w, a.out,
                         a.out_f32, split);
}

// F2 over bf16 y rows (prefill and GEMV paths), bracketed as BM_KERNEL_FINALIZE for the profile hooks
cudaError_t launch_combine(const ForwardArgs &a, cudaStream_t stream) {
    profile_begin(BM_KERNEL_FINALIZE, stream);
    cudaError_t e = launch_combine_raw(a, stream);
    profile_end(BM_KERNEL_FINALIZE, stream);
    return e;
}

// the decode path's tiling (host guess of the non-empty segments; the data-dependent truth lives on the device)
static void decode_tiling(int T, int D, int F, int K, int G, int S, int *R1, int *R2, int *ks2) {
    const int kb1 = (D + kBlockK - 1) / kBlockK, kb2 = (F + kBlockK - 1) / kBlockK;
    const long long TK = (long long)T * K;
    int n_seg = (int)(G < TK ? G : TK);
    n_seg += S;
    if (n_seg < 1) n_seg = 1;
    int ks1;
    choose_decode_tiling(F, kb1, n_seg, false, 2, num_sms(), R1, &ks1);
    choose_decode_tiling(D, kb2, n_seg, true, 1, num_sms(), R2, ks2);
    if (opt(OPT_DC_R2) > 0) { *R2 = std::max(32, std::min(128, opt(OPT_DC_R2)) & ~3); *ks2 = std::max(1, opt(OPT_DC_KS2)); }
    if (opt(OPT_DC_R1) > 0) *R1 = opt(OPT_DC_R1);
}

int decode_ksplit(int T, int D, int F, int K, int G, int S) {
    int R1, R2, ks2;
    decode_tiling(T, D, F, K, G, S, &R1, &R2, &ks2);
    return ks2;
}

cudaError_t launch_forward_tc(const ForwardArgs &a, bool decode, cudaStream_t stream) {
    const int TK = a.T * a.K;
    const int sms = num_sms();

    // Combine: fused into the GEMM2 epilogue (fp32 reductions into the zero region + last-arriver rounding) unless
    // option FUSED_COMBINE = 0 asks for the two-pass form on the prefill tiles (bf16 y rows + combine_kernel, slot
    // order: bit-deterministic for any K + S).  The decode kernel always finishes its output itself.
    // Decode kernel: its reductions are rounded and cleared by finalize_kernel.  Finishing inside the kernel (FC: fence +
    // ticket per item, the last arriver of a piece rounds it) saves that launch but was slower wherever it was measured --
    // G = 15, T = 16: 58.8 vs 54.9 us; G = 60, T = 16: 98.4 vs 92.7; G = 60, T = 256: 218 vs 190; BJ:configs[1]: equal --
    // because the items are short and the fence waits for the item's reductions; option FUSED_COMBINE = 1 selects it.
    // Prefill tiles: the fused epilogue (scale, transpose, vector reductions, fence, ticket, finish) takes ~10 us per
    // 128 x 256 tile and hides behind the tile's main loop only when the W2 reduction is long: fused from F = 4096 on
    // (Mixtral: 56 us per tile; also where the outputs are large enough for the fp32 sum to matter against the
    // tolerance), the two-pass form below (Qwen-like F = 1408: 6 us per tile; measured 5-10% faster there).
    const int fc_opt = opt(OPT_FUSED_COMBINE);
    const bool fused = decode ? fc_opt == 1 : (fc_opt < 0 ? a.F >= 4096 : fc_opt != 0);

    // CTA pairs (cta_group::2, M = 256 per pair): a pair shares the weight tile, so a CTA stages 32 KB per
    // k-block instead of 48 KB (measured: GEMM1 232 -> 201 us at BJ:configs[3]).  A segment with an odd chunk
    // count wastes half a pair, so pairs are used when a group expects >= 3 chunks.  Measured layer times, pairs /
    // single CTAs (which gather their rows themselves), D = 2048, F = 1408, E = 60, top-4: 410 rows per group
    // 253 / 274 us (G = 30, T = 3072) and 511 / 525 us (G = 60, T = 6144); 273 rows per group 198 / 206 us (G = 30)
    // but 402 / 392 us (G = 60); 137-205 rows per group 293 / 267 and 348 / 338 us.  BM_PF_PAIR=0/1 overrides.
    const int pair_env = opt(OPT_PF_PAIR);
    const bool many_rows = (long long)a.T * a.K >= 3LL * kChunkRows * a.G;
    const bool pair = !decode && (sms & 1) == 0 && (pair_env < 0 ? many_rows : pair_env != 0);
    // GA: GEMM1's own warps gather the token rows (single-CTA prefill tiles).  Measured (T = 4096, G = 60): step
    // 410 -> 398 us (GEMM1 +14 us, gather pass -20 us, A*D*4 bytes of HBM traffic less).  Not with CTA pairs: the peer's
    // "rows landed" must reach the leader's barrier through a fence and a cluster-scope arrive per k-block, which
    // lengthens the ring's turn-around -- GEMM1 30-36% slower than the TMA-fed pair kernel even with one relay warp
    // per ring stage (option PF_GATHER = 2 forces it).
    const int ga_env = opt(OPT_PF_GATHER);
    const bool gather_in_gemm = !decode && (ga_env == 2 || (ga_env == 1 && !pair));
    // Dense decode (T <= DC_DENSE_MAX_T = 64): every active weight set multiplies ALL T tokens (the MMA N side is the
    // token block of x itself, <= 64 columns: free under the weight stream) and GEMM2's epilogue weighs token t of
    // set u with its gate weight, zero where t was not routed to u.  No gathered copy of x, no dependence on the
    // permutation: the step is router (+ permutation for the API) -> GEMM1 -> GEMM2.
    const bool dense = decode && a.T <= std::min(opt(OPT_DC_DENSE_MAX_T), kDenseMaxT);

    // step 9 for the kernels that read token rows from xs
    if (!gather_in_gemm && !dense && TK > 0) {
        profile_begin(BM_KERNEL_PREP, stream);
        cudaError_t e = launch_kernel(gather_kernel, dim3(sms * 4), dim3(256), 0, stream, a.x, a.T, a.D, a.K, a.G,
                                      (const int32_t *)a.r.offsets, (const int32_t *)a.r.row_token, a.xs);
        if (e != cudaSuccess) return e;
        profile_end(BM_KERNEL_PREP, stream);
    }

    GemmParams p{};
    p.hints = 20;            // activations evict_last, weights evict_first (decode: the weights stream once)
    p.dense = dense ? 1 : 0;
    // G <= T*K: the dense H rows fit when indexed by the weight set itself (h_rows_needed), which lets GEMM1 write them
    // before it knows which sets are active
    p.dense_u = dense && (long long)a.G <= (long long)TK ? 1 : 0;
    p.status = a.status;
    p.seg_cap = a.G + a.S + 1;
    p.T = a.T; p.D = a.D; p.F = a.F; p.K = a.K; p.G = a.G; p.S = a.S; p.TK = TK;
    p.counts = a.r.counts; p.offsets = a.r.offsets; p.row_token = a.r.row_token; p.row_slot = a.r.row_slot;
    p.gate_w = a.r.gate_w; p.n_slots = a.r.n_slots; p.group_ids = a.r.group_ids; p.h = a.h; p.out_acc = a.out_acc; p.tickets = a.tickets;
    p.y = a.y; p.x = a.x; p.out = a.out; p.out_f32 = a.out_f32;

    const uint64_t h_rows = h_rows_needed(a.T, a.K, a.G, a.S);
    const int kb1 = (a.D + kBlockK - 1) / kBlockK, kb2 = (a.F + kBlockK - 1) / kBlockK;
    CUtensorMap m_xs, m_x, m_w1, m_w3, m_w2, m_h;
    cudaError_t err;

    if (!decode) {
        if (!make_map_2d(&m_xs, a.xs, TK > 0 ? TK : 1, a.D, 128) || !make_map_2d(&m_x, a.x, a.T, a.D, 128) ||
            !make_map_3d(&m_w1, a.W1, a.G + a.S, a.F, a.D, 128) || !make_map_3d(&m_w3, a.W3, a.G + a.S, a.F, a.D, 128) ||
            !make_map_3d(&m_w2, a.W2, a.G + a.S, a.D, a.F, 256) || !make_map_2d(&m_h, a.h, h_rows, a.F, 128))
            return cudaErrorInvalidValue;
        p.ksplit = 1;
        CUtensorMap m_w2h;
        if (pair && !make_map_3d(&m_w2h, a.W2, a.G + a.S, a.D, a.F, 128)) return cudaErrorInvalidValue;
        ring_geometry(false, true, a.T, &p, pair);
        p.kblocks = kb1; p.R = 128; p.n_wtiles = (a.F + 127) / 128;
        // L2 behaviour of the prefill tiles (ncu at BJ:configs[2], DRAM bytes read by GEMM1 / GEMM2; algorithmic 1.06 / 0.90 GB):
        //   weights evict_first (round 1)             4.64 / 5.81 GB   -- a weight tile is shared by every chunk of its group, but
        //   weights evict_normal or evict_last        1.95 / 3.65 GB      an evict_first line is gone before the other CTAs ask for it
        //   + chunk bands of 8 / 16 pairs (GEMM1)     4.1 / 2.2 GB     -- fewer CTAs share a weight tile at a time: worse
        //   + square bands 9 chunks x 8 tiles (GEMM2) 4.3 GB           -- worse as well
        // so the hints changed (cold-cache kernel time -7% / -8.5%) and the band order stays available but off (options
        // PF_G1_BC, PF_G2_BC, PF_G2_BW; get_item).
        p.band_c = opt(OPT_PF_G1_BC) > 0 ? opt(OPT_PF_G1_BC) : 0;
        p.band_w = 0;
        // (with single-CTA tiles a group has at most ~2 chunks: its weights stream once -> evict_first, as on the decode path;
        //  G = 8, T = 256: 69 -> 64 us)
        p.hints = opt(OPT_PF_G1_HINTS) >= 0 ? opt(OPT_PF_G1_HINTS) : (pair ? 21 : 20);
        // shared experts ahead of the routing (gemm_kernel, "speculative start"): inside bm_moe_layer only -- there the
        // routing kernels are known to be this launch's predecessors and to let it start early
        p.spec_shared = a.after_router && a.S > 0 && opt(OPT_PF_SPEC) != 0 ? 1 : 0;
        if (gather_in_gemm)
            err = pair ? launch_gemm<PF_GEMM1, true, true>(m_xs, m_x, m_w1, m_w3, p, stream)
                       : launch_gemm<PF_GEMM1, false, true>(m_xs, m_x, m_w1, m_w3, p, stream);
        else
            err = pair ? launch_gemm<PF_GEMM1, true>(m_xs, m_x, m_w1, m_w3, p, stream)
                       : launch_gemm<PF_GEMM1>(m_xs, m_x, m_w1, m_w3, p, stream);
        if (err != cudaSuccess) return err;
        p.kblocks = kb2; p.R = 256; p.n_wtiles = (a.D + 255) / 256;
        p.spec_shared = 0;
        p.band_w = opt(OPT_PF_G2_BW) > 0 ? opt(OPT_PF_G2_BW) : 0;
        p.band_c = opt(OPT_PF_G2_BC) > 0 ? opt(OPT_PF_G2_BC) : 0;
        p.hints = opt(OPT_PF_G2_HINTS) >= 0 ? opt(OPT_PF_G2_HINTS) : (pair ? 21 : 20);
        if (fused)
            err = pair ? launch_gemm<PF_GEMM2, true, false, true>(m_h, m_h, m_w2h, m_w2h, p, stream)
                       : launch_gemm<PF_GEMM2, false, false, true>(m_h, m_h, m_w2, m_w2, p, stream);
        else
            err = pair ? launch_gemm<PF_GEMM2, true>(m_h, m_h, m_w2h, m_w2h, p, stream)
                       : launch_gemm<PF_GEMM2>(m_h, m_h, m_w2, m_w2, p, stream);
        if (err != cudaSuccess) return err;
    } else {
        int R1, R2, ks2;
        decode_tiling(a.T, a.D, a.F, a.K, a.G, a.S, &R1, &R2, &ks2);
        const int nbox = 32;                         // token rows travel in 32-row boxes, as many as the chunk has
        if (!make_map_2d(&m_xs, a.xs, TK > 0 ? TK : 1, a.D, nbox) || !make_map_2d(&m_x, a.x, a.T, a.D, nbox) ||
            !make_map_3d(&m_w1, a.W1, a.G + a.S, a.F, a.D, R1) || !make_map_3d(&m_w3, a.W3, a.G + a.S, a.F, a.D, R1) ||
            !make_map_3d(&m_w2, a.W2, a.G + a.S, a.D, a.F, R2) || !make_map_2d(&m_h, a.h, h_rows, a.F, nbox))
            return cudaErrorInvalidValue;
        p.ksplit = 1; p.kblocks = kb1; p.R = R1; p.n_wtiles = (a.F + R1 - 1) / R1;
        ring_geometry(true, true, a.T, &p);
        {
            // L2 prefetch budget (option DC_PREFETCH_MB, default 48 MB): spread evenly over the W1 / W3 sets, whole 16 KB pieces
            const unsigned long long set_bytes = (unsigned long long)a.F * a.D * 2ull;
            unsigned long long per = ((unsigned long long)std::max(opt(OPT_DC_PREFETCH_MB), 0) << 20) / (2ull * (a.G + a.S));
            if (per > set_bytes) per = set_bytes;
            p.w1 = a.W1; p.w3 = a.W3; p.pf_set_bytes = set_bytes; p.pf_bytes = per & ~16383ull;
            // Speculative start (gemm_kernel): inside bm_moe_layer, as many leading sets as the HBM streams in DC_SPEC_US
            // microseconds -- about the time the routing kernels take -- at least one.  A speculated set that turns out
            // inactive costs bandwidth that was idle anyway, as long as the speculated part does not outlast the routing:
            // D = 2048, F = 1408, E = 60, top-4, T = 16 (us, off / 12 us / 24 us): G = 15 55.3 / 49.3 / 48.9, G = 30 85.8 /
            // 76.9 / 76.9 and with zipf-2 routing (13 of 30 sets active) 56.6 / 49.9 / 53.0; G = 60, 15 of 60 active: 64.9 /
            // 60.4.  DC_SPEC_MIN_ROWS (1) asks for that many expected rows per set, T*K >= rows * G, before speculating.
            // BJ:configs[1] (117 MB per weight matrix) gains nothing: its L2 prefetch already hides the routing kernels.
            const int spec_us = opt(OPT_DC_SPEC_US);
            if (p.dense_u && a.after_router && spec_us > 0 && a.G > 0 &&
                (long long)TK >= (long long)std::max(opt(OPT_DC_SPEC_MIN_ROWS), 1) * a.G) {
                const unsigned long long budget = (unsigned long long)spec_us * 6400000ull;      // bytes at 6.4 TB/s
                unsigned long long n = (budget + 2 * set_bytes - 1) / (2 * set_bytes);
                p.spec_sets = (int)std::min<unsigned long long>(std::max<unsigned long long>(n, 1), (unsigned long long)a.G);
                // what would be left fills less than one wave of CTAs: take it along instead of waiting for the routing with
                // most SMs idle (G = 8, T = 16: 39.3 -> 34.5 us)
                if ((long long)(a.G - p.spec_sets) * p.n_wtiles < sms) p.spec_sets = a.G;
            }
        }
        if ((err = launch_gemm<DC_GEMM1>(m_xs, m_x, m_w1, m_w3, p, stream)) != cudaSuccess) return err;
        p.ksplit = ks2; p.kblocks = kb2 / ks2; p.R = R2; p.n_wtiles = (a.D + R2 - 1) / R2;
        p.spec_sets = 0;
        ring_geometry(true, false, a.T, &p);
        err = fused ? launch_gemm<DC_GEMM2, false, false, true>(m_h, m_h, m_w2, m_w2, p, stream)
                    : launch_gemm<DC_GEMM2>(m_h, m_h, m_w2, m_w2, p, stream);
        if (err != cudaSuccess) return err;
        if (!fused) {
            const size_t n8 = (size_t)a.T * a.D / 8;
            int grid = (int)std::min<size_t>((n8 + 255) / 256, (size_t)sms * 8);
            profile_begin(BM_KERNEL_FINALIZE, stream);
            err = launch_kernel(finalize_kernel, dim3(grid < 1 ? 1 : grid), dim3(256), 0, stream, a.out_acc, a.out, a.out_f32, n8, 1);
            profile_end(BM_KERNEL_FINALIZE, stream);
        }
        return err;
    }

    if (fused) return cudaSuccess;
    profile_begin(BM_KERNEL_FINALIZE, stream);
    err = launch_combine_raw(a, stream);
    profile_end(BM_KERNEL_FINALIZE, stream);
    return err;
}

// f_e(x_t) for every expert and token (calibration forward): the prefill GEMM kernels over a
// all-shared schedule (G = 0 routed groups, S = E always-on weight sets); y: token-major [T, E, D] bf16.
cudaError_t launch_expert_outputs(const bm_bf16 *x, int T, int D, const bm_bf16 *W1, const bm_bf16 *W3,
                                  const bm_bf16 *W2, int E, int F, bm_bf16 *y, bm_bf16 *h, cudaStream_t stream) {
    cudaError_t err;
    GemmParams p{};
    p.hints = 20;
    p.seg_cap = E + 1;
    p.T = T; p.D = D; p.F = F; p.K = 1; p.G = 0; p.S = E; p.TK = 0;
    p.h = h; p.y = y; p.x = x; p.y_tm = 1;
    p.ksplit = 1;
    const bool pair = (num_sms() & 1) == 0 && T >= 3 * kChunkRows && opt(OPT_PF_PAIR) != 0;   // as launch_forward_tc
    CUtensorMap m_x, m_w1, m_w3, m_w2, m_h;
    if (!make_map_2d(&m_x, x, T, D, 128) || !make_map_3d(&m_w1, W1, E, F, D, 128) || !make_map_3d(&m_w3, W3, E, F, D, 128) ||
        !make_map_3d(&m_w2, W2, E, D, F, pair ? 128 : 256) || !make_map_2d(&m_h, h, (uint64_t)E * T, F, 128))
        return cudaErrorInvalidValue;
    ring_geometry(false, true, T, &p, pair);
    p.hints = pair ? 21 : 20;          // every chunk of a segment shares its weight tiles (see launch_forward_tc)
    p.kblocks = (D + kBlockK - 1) / kBlockK; p.R = 128; p.n_wtiles = (F + 127) / 128;
    err = pair ? launch_gemm<PF_GEMM1, true>(m_x, m_x, m_w1, m_w3, p, stream) : launch_gemm<PF_GEMM1>(m_x, m_x, m_w1, m_w3, p, stream);
    if (err != cudaSuccess) return err;
    p.kblocks = (F + kBlockK - 1) / kBlockK; p.R = 256; p.n_wtiles = (D + 255) / 256;
    return pair ? launch_gemm<PF_GEMM2, true>(m_h, m_h, m_w2, m_w2, p, stream) : launch_gemm<PF_GEMM2>(m_h, m_h, m_w2, m_w2, p, stream);
}

cudaError_t launch_round_bf16(const float *in, size_t n, bm_bf16 *out, cudaStream_t stream) {
    const size_t n8 = n / 8;
    long long grid = (long long)((n8 + 255) / 256);
    if (grid > num_sms() * 8) grid = num_sms() * 8;
    if (grid < 1) grid = 1;
    return launch_kernel(finalize_kernel, dim3((unsigned)grid), dim3(256), 0, stream, const_cast<float *>(in), out,
                         (float *)nullptr, n8, 0);
}

}  // namespace bm
