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
// roles from a small device-side schedule (non-empty segments and their 128-row chunks) that the prep
// kernel builds from counts/offsets -- the host never sees the data-dependent counts.
//
// The combine accumulates in fp32 (`out_acc`, red.global.add) because a token's <= K group rows live in
// different tiles (and, in decode, in different K-splits); a last pass rounds to bf16.
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
constexpr int kChunkRows = 128;
constexpr int kMaxSeg = BM_MAX_G + kMaxShared;
constexpr size_t kSmemMax = 232448;         // 227 KB, the per-CTA opt-in limit of sm_100
constexpr size_t kSmemBars = 256;           // (2*kMaxStages + 2*kAccStages) mbarriers + the TMEM base address
constexpr size_t kEpiStageBytes = 32 * 32 * 4;   // PF_GEMM2: per-epilogue-warp transpose buffer (32 rows x 32 fp32)
constexpr size_t kSmemEpi = 4 * kEpiStageBytes;
constexpr size_t kSmemRing = kSmemMax - 1024 /*align slack*/ - kSmemBars;   // minus kSmemEpi for PF_GEMM2
static_assert((2 * kMaxStages + 2 * kAccStages) * 8 + 4 <= kSmemBars, "barrier block too small");

enum Mode { PF_GEMM1 = 0, PF_GEMM2 = 1, DC_GEMM1 = 2, DC_GEMM2 = 3 };

// schedule (int32) written by the prep kernel
//   [0] n_seg   [1] total_chunks   [4 .. 4+kMaxSeg) seg_u   [4+kMaxSeg .. 4+2*kMaxSeg+1) seg_chunk0
constexpr int kSchedSegU = 4;
constexpr int kSchedChunk0 = 4 + kMaxSeg;
static_assert(kSchedChunk0 + kMaxSeg + 1 <= kSchedInts, "sched too small");

struct GemmParams {
    int T, D, F, K, G, S, TK;
    int stages;         // depth of the shared-memory ring (<= kMaxStages)
    int stage_bytes;    // bytes of one ring stage (multiple of 1024)
    int off_b;          // decode: offset of the token rows (MMA B operand) inside a stage
    int npad_box;       // decode: rows of the token box every stage loads (host: T rounded up to 32, <= 128)
    int kblocks;        // k-blocks of one item (per split)
    int ksplit;         // K splits (DC_GEMM2), else 1
    int R;              // weight rows per tile (prefill: 128 for GEMM1 per matrix, 256 for GEMM2)
    int n_wtiles;       // tiles along the weight-row dimension
    const int32_t *counts, *offsets, *row_token, *row_slot;
    const float *gate_w;
    const int32_t *sched;
    bm_bf16 *h;
    float *out_acc;
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

template <int MODE>
__device__ __forceinline__ bool get_item(const GemmParams &p, int item, Item &it) {
    const int32_t *sched = p.sched;
    const int n_seg = sched[0];
    const int per_chunk = p.n_wtiles * p.ksplit;
    const long long n_items = (long long)sched[1] * per_chunk;
    if (item >= n_items) return false;
    const int32_t *chunk0 = sched + kSchedChunk0;
    int lo = 0, hi = n_seg - 1;               // last segment s with chunk0[s] * per_chunk <= item
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((long long)chunk0[mid] * per_chunk <= item) lo = mid; else hi = mid - 1;
    }
    const int s = lo;
    const int u = sched[kSchedSegU + s];
    const int chunks_s = chunk0[s + 1] - chunk0[s];
    const int local = item - chunk0[s] * per_chunk;
    const int chunk = local % chunks_s;
    const int rest = local / chunks_s;
    it.u = u;
    it.ks = rest % p.ksplit;
    it.wt = rest / p.ksplit;
    it.shared = u >= p.G;
    const int rows = it.shared ? p.T : p.counts[u];
    it.n = min(kChunkRows, rows - chunk * kChunkRows);
    if (it.shared) {
        it.tok0 = chunk * kChunkRows;
        it.perm_row0 = 0;
        it.h_row0 = p.TK + (u - p.G) * p.T + it.tok0;
        it.act_row0 = (MODE == PF_GEMM1 || MODE == DC_GEMM1) ? it.tok0 : it.h_row0;
    } else {
        it.tok0 = 0;
        it.perm_row0 = p.offsets[u] + chunk * kChunkRows;
        it.h_row0 = it.perm_row0;
        it.act_row0 = it.perm_row0;
    }
    return true;
}

__device__ __forceinline__ float silu_mul(float a, float b) {
    return __fdividef(a, 1.0f + __expf(-a)) * b;
}

template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
gemm_kernel(const __grid_constant__ CUtensorMap tm_act0,   // GEMM1: xs [TK, D]; GEMM2: H [TK+S*T, F]
            const __grid_constant__ CUtensorMap tm_act1,   // GEMM1: x [T, D] (shared experts); GEMM2: unused
            const __grid_constant__ CUtensorMap tm_w0,     // GEMM1: W1 [G+S, F, D]; GEMM2: W2 [G+S, D, F]
            const __grid_constant__ CUtensorMap tm_w1,     // GEMM1: W3; GEMM2: unused
            const GemmParams p) {
    constexpr bool kDecode = (MODE == DC_GEMM1 || MODE == DC_GEMM2);
    constexpr bool kGemm1 = (MODE == PF_GEMM1 || MODE == DC_GEMM1);

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
    uint8_t *epi_stage = reinterpret_cast<uint8_t *>(bars) + kSmemBars;   // [4][kEpiStageBytes], 256-byte aligned

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // ---- prologue: nothing here depends on a predecessor kernel, so under PDL it overlaps its tail ----
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tm_act0);
        ptx::prefetch_tmap(&tm_w0);
        if (kGemm1) { ptx::prefetch_tmap(&tm_act1); ptx::prefetch_tmap(&tm_w1); }
        for (int i = 0; i < n_stages; ++i) { ptx::mbar_init(&full[i], 1); ptx::mbar_init(&empty[i], 1); }
        for (int i = 0; i < kAccStages; ++i) { ptx::mbar_init(&tfull[i], 1); ptx::mbar_init(&tempty[i], 4); }
        ptx::fence_barrier_init();
    }
    if (warp == 1) ptx::tmem_alloc(tmem_ptr, kTmemCols);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;

    const int nkb = p.kblocks;
    // bytes one stage receives: constant per launch (decode always loads the full padded token box)
    const uint32_t stage_tx = !kDecode ? 3u * kTileBytes16K
                                       : (uint32_t)((kGemm1 ? 2 : 1) * p.R * 128 + p.npad_box * 128);

    // The producer and the MMA issuer run their loops with the WHOLE warp (warp-uniform control flow keeps
    // addresses and descriptors in uniform registers) and elect one lane for the issuing instructions: the
    // single-thread instruction stream per k-block is what paces a decode tile, so it is kept short.
    if (warp == 0) {
        // =========================== TMA producer ===========================
        int stage = 0;
        uint32_t phase = 0;
        Item it;
        int item = blockIdx.x;
        int kb_first = 0;
        bool have;
        if (MODE == DC_GEMM2) {
            // W2 does not depend on the predecessor (GEMM1): fill the ring with weight tiles BEFORE the
            // grid-dependency wait, so the HBM stream starts while GEMM1's last CTAs drain.  The schedule
            // read by get_item was written by the prep kernel, which completed before GEMM1 (which
            // triggers this launch only after its own wait) let this grid start.
            have = get_item<MODE>(p, item, it);
            const int pre = have ? min(n_stages, nkb) : 0;
            if (ptx::elect_one())
                for (int kb = 0; kb < pre; ++kb) {
                    ptx::mbar_arrive_expect_tx(&full[kb], stage_tx);
                    ptx::tma_load_3d(smem + (size_t)kb * stage_bytes, &tm_w0, &full[kb], (it.ks * nkb + kb) * kBlockK,
                                     it.wt * p.R, it.u, ptx::kEvictFirst);
                }
            __syncwarp();
            grid_dep_wait();
            if (ptx::elect_one())
                for (int kb = 0; kb < pre; ++kb)
                    ptx::tma_load_2d(smem + (size_t)kb * stage_bytes + p.off_b, &tm_act0, &full[kb],
                                     (it.ks * nkb + kb) * kBlockK, it.act_row0, ptx::kEvictLast);
            __syncwarp();
            kb_first = pre;
            stage = pre;
            if (stage == n_stages) { stage = 0; phase = 1; }
        } else {
            grid_dep_wait();
            have = get_item<MODE>(p, item, it);
        }
        if (lane == 0) grid_dep_launch();
        for (; have; item += gridDim.x, have = get_item<MODE>(p, item, it), kb_first = 0) {
            const CUtensorMap *tm_act = (kGemm1 && it.shared) ? &tm_act1 : &tm_act0;
            const int wrow0 = it.wt * p.R;
            int kc = (it.ks * nkb + kb_first) * kBlockK;
            for (int kb = kb_first; kb < nkb; ++kb, kc += kBlockK) {
                ptx::mbar_wait(&empty[stage], phase ^ 1);
                if (ptx::elect_one()) {
                    uint8_t *st = smem + (size_t)stage * stage_bytes;
                    ptx::mbar_arrive_expect_tx(&full[stage], stage_tx);
                    if (!kDecode) {
                        // A = 128 activation rows, B = 256 weight rows (W1|W3 tiles, or one W2 tile of 256)
                        ptx::tma_load_2d(st, tm_act, &full[stage], kc, it.act_row0, ptx::kEvictLast);
                        ptx::tma_load_3d(st + kTileBytes16K, &tm_w0, &full[stage], kc, wrow0, it.u, ptx::kEvictFirst);
                        if (MODE == PF_GEMM1)
                            ptx::tma_load_3d(st + 2 * kTileBytes16K, &tm_w1, &full[stage], kc, wrow0, it.u, ptx::kEvictFirst);
                    } else {
                        // M side = R weight rows (streamed once from HBM), N side = the group's token rows
                        // (one box of npad_box rows; rows past the group's are loaded and never multiplied)
                        ptx::tma_load_3d(st, &tm_w0, &full[stage], kc, wrow0, it.u, ptx::kEvictFirst);
                        if (MODE == DC_GEMM1)
                            ptx::tma_load_3d(st + kTileBytes16K, &tm_w1, &full[stage], kc, wrow0, it.u, ptx::kEvictFirst);
                        ptx::tma_load_2d(st + p.off_b, tm_act, &full[stage], kc, it.act_row0, ptx::kEvictLast);
                    }
                }
                __syncwarp();
                if (++stage == n_stages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        grid_dep_wait();
        // descriptor low words: (smem address >> 4) | LBO; the high word (SBO, version, swizzle) is constant
        const uint32_t a_lo0 = ptx::smem_desc_lo(ptx::smem_u32(smem));
        const uint32_t b_off = (uint32_t)(kDecode ? p.off_b : kTileBytes16K) >> 4;
        const uint32_t stage_step = stage_bytes >> 4;
        uint32_t a_lo = a_lo0;
        int stage = 0;
        uint32_t phase = 0;
        int acc = 0;
        uint32_t acc_phase = 0;
        Item it;
        for (int item = blockIdx.x; get_item<MODE>(p, item, it); item += gridDim.x) {
            const uint32_t idesc = kDecode ? ptx::make_idesc_bf16(128, (it.n + 31) & ~31) : ptx::make_idesc_bf16(128, 256);
            ptx::mbar_wait(&tempty[acc], acc_phase ^ 1);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * kAccCols;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(&full[stage], phase);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
#pragma unroll
                    for (int k = 0; k < kBlockK / 16; ++k) {
                        const uint32_t accum = (kb | k) ? 1u : 0u;
                        const uint32_t ko = 2 * k;             // 16 bf16 = 32 bytes = 2 descriptor units
                        ptx::mma_bf16_ss(d_tmem, ptx::smem_desc(a_lo + ko), ptx::smem_desc(a_lo + b_off + ko), idesc, accum);
                        if (MODE == DC_GEMM1)
                            ptx::mma_bf16_ss(d_tmem + 128, ptx::smem_desc(a_lo + (kTileBytes16K >> 4) + ko),
                                             ptx::smem_desc(a_lo + b_off + ko), idesc, accum);
                    }
                    ptx::mma_commit(&empty[stage]);                  // frees the smem stage when the MMAs retire
                    if (kb == nkb - 1) ptx::mma_commit(&tfull[acc]);   // accumulator complete
                }
                __syncwarp();
                a_lo += stage_step;
                if (++stage == n_stages) { stage = 0; phase ^= 1; a_lo = a_lo0; }
            }
            if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
        }
    } else {
        // =========================== epilogue (warps 2..5) ===========================
        grid_dep_wait();
        const int q = warp & 3;                      // TMEM lane quarter this warp may read
        const int row = q * 32 + lane;               // accumulator row (M index) owned by this thread
        int acc = 0;
        uint32_t acc_phase = 0;
        Item it;
        for (int item = blockIdx.x; get_item<MODE>(p, item, it); item += gridDim.x) {
            ptx::mbar_wait(&tfull[acc], acc_phase);
            ptx::tc_fence_after();
            const uint32_t t_addr = tmem_base + acc * kAccCols + ((uint32_t)(q * 32) << 16);

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
            } else if (MODE == PF_GEMM2) {
                // row = token row; columns = 256 output features d0..d0+255; scatter-combine with the gate weight.
                // The accumulator leaves TMEM with one row per lane; a per-warp shared-memory transpose (32 rows
                // x 32 columns fp32, 16-byte units xor-swizzled by the row) turns that into row-contiguous
                // pieces, so every red.global.add.v4.f32 of a warp covers 4 rows x 128 contiguous bytes
                // (whole L2 lines) instead of 32 scattered 16-byte pieces.
                int tok = -1;
                float gw = 1.0f;
                if (row < it.n) {
                    if (it.shared) {
                        tok = it.tok0 + row;
                    } else {
                        tok = p.row_token[it.perm_row0 + row];
                        gw = p.gate_w[(size_t)tok * p.K + p.row_slot[it.perm_row0 + row]];
                    }
                }
                const int d0 = it.wt * 256;
                float4 *stg = reinterpret_cast<float4 *>(epi_stage + (size_t)q * kEpiStageBytes);
                const int rl = lane >> 3, ul = lane & 7;        // read phase: row (mod 4) and 16-byte unit of this lane
#pragma unroll 1
                for (int c = 0; c < 256; c += 32) {
                    uint32_t v[32];
                    ptx::tmem_ld_x32(t_addr + c, v);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        stg[lane * 8 + (u ^ (lane & 7))] =
                            make_float4(gw * __uint_as_float(v[4 * u]), gw * __uint_as_float(v[4 * u + 1]),
                                        gw * __uint_as_float(v[4 * u + 2]), gw * __uint_as_float(v[4 * u + 3]));
                    __syncwarp();
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int r = 4 * j + rl;
                        const float4 o = stg[r * 8 + (ul ^ (r & 7))];
                        const int tk = __shfl_sync(0xffffffffu, tok, r);
                        const int d = d0 + c + 4 * ul;
                        if (tk >= 0 && d + 4 <= p.D)
                            ptx::red_add_v4_f32(p.out_acc + (size_t)tk * p.D + d, o.x, o.y, o.z, o.w);
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
                // Lane l first fetches token and gate weight of chunk rows l, l+32, ... (one dependent-load chain
                // per item instead of one per token); the loop broadcasts them with shuffles.
                const int d = it.wt * p.R + row;
                const bool d_ok = row < p.R && d < p.D;
                int tokr[4];
                float gwr[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int r = j * 32 + lane;
                    tokr[j] = -1;
                    gwr[j] = 1.0f;
                    if (r < it.n) {
                        if (it.shared) {
                            tokr[j] = it.tok0 + r;
                        } else {
                            tokr[j] = p.row_token[it.perm_row0 + r];
                            gwr[j] = p.gate_w[(size_t)tokr[j] * p.K + p.row_slot[it.perm_row0 + r]];
                        }
                    }
                }
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
            }
            // release the accumulator stage
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&tempty[acc]);
            if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, kTmemCols);
    }
}

// -------------------------------------------------------------------------------------------------
// prep: build the schedule, zero the fp32 accumulator, gather token rows into permuted order (step 9)
// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
prep_kernel(const bm_bf16 *__restrict__ x, int T, int D, int K, int G, int S,
            const int32_t *__restrict__ counts, const int32_t *__restrict__ offsets,
            const int32_t *__restrict__ row_token, int32_t *__restrict__ sched, bm_bf16 *__restrict__ xs,
            float *__restrict__ out_acc, int32_t *__restrict__ status) {
    grid_dep_wait();
    grid_dep_launch();
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        int n_seg = 0, chunks = 0;
        bool bad = false;
        for (int u = 0; u < G + S; ++u) {
            const int rows = u < G ? counts[u] : T;
            if (u < G && (rows < 0 || offsets[u] < 0 || offsets[u] + rows > T * K)) { bad = true; continue; }
            if (rows <= 0) continue;
            sched[kSchedSegU + n_seg] = u;
            sched[kSchedChunk0 + n_seg] = chunks;
            chunks += (rows + kChunkRows - 1) / kChunkRows;
            ++n_seg;
        }
        sched[kSchedChunk0 + n_seg] = chunks;
        sched[0] = n_seg;
        sched[1] = chunks;
        if (bad) atomicOr(status, BM_DEV_BAD_ROUTING);
    }
    // zero out_acc
    const size_t n4 = (size_t)T * D / 4;
    float4 *o4 = reinterpret_cast<float4 *>(out_acc);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x)
        o4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    // gather: one warp per permuted row
    const int A = min(offsets[G], T * K);
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

__global__ void __launch_bounds__(256)
finalize_kernel(const float *__restrict__ out_acc, bm_bf16 *__restrict__ out, size_t n8) {
    grid_dep_wait();
    grid_dep_launch();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
        const float4 a = reinterpret_cast<const float4 *>(out_acc)[2 * i];
        const float4 b = reinterpret_cast<const float4 *>(out_acc)[2 * i + 1];
        reinterpret_cast<uint4 *>(out)[i] = make_uint4(pack_bf16x2(a.x, a.y), pack_bf16x2(a.z, a.w),
                                                       pack_bf16x2(b.x, b.y), pack_bf16x2(b.z, b.w));
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

// [rows, cols] bf16 row-major, box = box_rows x 64 columns, 128B swizzle
bool make_map_2d(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * sizeof(bm_bf16)};
    cuuint32_t box[2] = {kBlockK, box_rows};
    cuuint32_t es[2] = {1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// [n, rows, cols] bf16, box = 1 x box_rows x 64
bool make_map_3d(CUtensorMap *m, const void *base, uint64_t n, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[3] = {cols, rows, n};
    cuuint64_t strides[2] = {cols * sizeof(bm_bf16), rows * cols * sizeof(bm_bf16)};
    cuuint32_t box[3] = {kBlockK, box_rows, 1};
    cuuint32_t es[3] = {1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(base), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Decode tiling: rows-per-tile R in [32,128] and K-split count so that the number of equal-cost items
// is as close as possible to a multiple of the SM count (static round-robin schedule).
void choose_decode_tiling(int wrows, int kblocks, int n_seg, bool allow_split, int sms, int *R_out, int *ks_out) {
    double best = -1.0;
    int bestR = 128, bestKs = 1;
    const int max_ks = allow_split ? 16 : 1;
    int rmax = tune_int("BM_DC_RMAX", 128);
    rmax = rmax < 32 ? 32 : (rmax > 128 ? 128 : rmax);
    for (int ks = 1; ks <= max_ks; ++ks) {
        if (kblocks % ks != 0 || kblocks / ks < 4) { if (ks > 1) continue; }
        for (int R = rmax; R >= 32; --R) {
            const int tiles = (wrows + R - 1) / R;
            const long long items = (long long)tiles * n_seg * ks;
            const long long waves = (items + sms - 1) / sms;
            // useful rows / rows paid for, times wave occupancy; mild penalty for tiny tiles
            double eff = (double)wrows / ((double)tiles * R) * (double)items / (double)(waves * sms);
            eff -= 0.0005 * (rmax - R) / 96.0 + 0.002 * (ks - 1);
            if (eff > best + 1e-9) { best = eff; bestR = R; bestKs = ks; }
        }
    }
    *R_out = bestR;
    *ks_out = bestKs;
}

// Ring geometry.  Prefill: 4 stages x (16 KB tokens + 32 KB weights).  Decode: a stage holds the weight
// tile(s) (16 KB each, R <= 128 rows used) and the token rows padded to 32 (npad_max x 128 B); as many
// stages as fit in 227 KB, because the bytes in flight per SM are what the HBM stream lives on.
void ring_geometry(bool decode, bool gemm1, int T, GemmParams *p) {
    if (!decode) {
        p->stage_bytes = 3 * kTileBytes16K;
        p->off_b = kTileBytes16K;
    } else {
        const int rows = T < kChunkRows ? T : kChunkRows;
        const int npad_max = (rows + 31) & ~31;
        p->off_b = (gemm1 ? 2 : 1) * kTileBytes16K;
        p->stage_bytes = p->off_b + npad_max * 128;
        p->npad_box = npad_max;
    }
    int st = (int)((kSmemRing - (decode ? 0 : kSmemEpi)) / (size_t)p->stage_bytes);
    const int cap = tune_int(decode ? "BM_DC_STAGES" : "BM_PF_STAGES", kMaxStages);
    if (st > cap) st = cap;
    if (st > kMaxStages) st = kMaxStages;
    if (st < 2) st = 2;
    p->stages = st;
}

template <int MODE>
cudaError_t launch_gemm(const CUtensorMap &a0, const CUtensorMap &a1, const CUtensorMap &w0, const CUtensorMap &w1,
                        const GemmParams &p, cudaStream_t stream) {
    auto kern = gemm_kernel<MODE>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    constexpr int kid = (MODE == PF_GEMM1 || MODE == DC_GEMM1) ? BM_KERNEL_GEMM1 : BM_KERNEL_GEMM2;
    const size_t smem = 1024 + (size_t)p.stages * p.stage_bytes + kSmemBars + (MODE == PF_GEMM2 ? kSmemEpi : 0);
    profile_begin(kid, stream);
    cudaError_t e = launch_kernel(kern, dim3(num_sms()), dim3(kThreads), smem, stream, a0, a1, w0, w1, p);
    profile_end(kid, stream);
    return e;
}

}  // namespace

cudaError_t launch_forward_tc(const ForwardArgs &a, bool decode, cudaStream_t stream) {
    const int TK = a.T * a.K;
    const int sms = num_sms();

    // step 9 (+ schedule, + zero)
    {
        const int grid = sms * 4;
        profile_begin(BM_KERNEL_PREP, stream);
        cudaError_t e = launch_kernel(prep_kernel, dim3(grid), dim3(256), 0, stream, a.x, a.T, a.D, a.K, a.G, a.S,
                                      a.r.counts, a.r.offsets, a.r.row_token, a.sched, a.xs, a.out_acc, a.status);
        if (e != cudaSuccess) return e;
        profile_end(BM_KERNEL_PREP, stream);
    }

    GemmParams p{};
    p.T = a.T; p.D = a.D; p.F = a.F; p.K = a.K; p.G = a.G; p.S = a.S; p.TK = TK;
    p.counts = a.r.counts; p.offsets = a.r.offsets; p.row_token = a.r.row_token; p.row_slot = a.r.row_slot;
    p.gate_w = a.r.gate_w; p.sched = a.sched; p.h = a.h; p.out_acc = a.out_acc;


    const uint64_t h_rows = (uint64_t)TK + (uint64_t)a.S * a.T;
    const int kb1 = (a.D + kBlockK - 1) / kBlockK, kb2 = (a.F + kBlockK - 1) / kBlockK;
    CUtensorMap m_xs, m_x, m_w1, m_w3, m_w2, m_h;
    cudaError_t err;

    if (!decode) {
        if (!make_map_2d(&m_xs, a.xs, TK > 0 ? TK : 1, a.D, 128) || !make_map_2d(&m_x, a.x, a.T, a.D, 128) ||
            !make_map_3d(&m_w1, a.W1, a.G + a.S, a.F, a.D, 128) || !make_map_3d(&m_w3, a.W3, a.G + a.S, a.F, a.D, 128) ||
            !make_map_3d(&m_w2, a.W2, a.G + a.S, a.D, a.F, 256) || !make_map_2d(&m_h, a.h, h_rows, a.F, 128))
            return cudaErrorInvalidValue;
        p.ksplit = 1;
        ring_geometry(false, true, a.T, &p);
        p.kblocks = kb1; p.R = 128; p.n_wtiles = (a.F + 127) / 128;
        if ((err = launch_gemm<PF_GEMM1>(m_xs, m_x, m_w1, m_w3, p, stream)) != cudaSuccess) return err;
        p.kblocks = kb2; p.R = 256; p.n_wtiles = (a.D + 255) / 256;
        if ((err = launch_gemm<PF_GEMM2>(m_h, m_h, m_w2, m_w2, p, stream)) != cudaSuccess) return err;
    } else {
        // segments expected to be non-empty (host guess; the data-dependent truth lives on the device)
        int n_seg = a.G < TK ? a.G : TK;
        n_seg += a.S;
        if (n_seg < 1) n_seg = 1;
        int R1, R2, ks1, ks2;
        choose_decode_tiling(a.F, kb1, n_seg, false, sms, &R1, &ks1);
        choose_decode_tiling(a.D, kb2, n_seg, true, sms, &R2, &ks2);
        if (tune_int("BM_DC_R2", 0) > 0) { R2 = tune_int("BM_DC_R2", 0); ks2 = tune_int("BM_DC_KS2", 1); }
        if (tune_int("BM_DC_R1", 0) > 0) R1 = tune_int("BM_DC_R1", 0);
        const int rows_max = a.T < kChunkRows ? a.T : kChunkRows;
        const int nbox = (rows_max + 31) & ~31;      // token rows every stage loads (ring_geometry: npad_box)
        if (!make_map_2d(&m_xs, a.xs, TK > 0 ? TK : 1, a.D, nbox) || !make_map_2d(&m_x, a.x, a.T, a.D, nbox) ||
            !make_map_3d(&m_w1, a.W1, a.G + a.S, a.F, a.D, R1) || !make_map_3d(&m_w3, a.W3, a.G + a.S, a.F, a.D, R1) ||
            !make_map_3d(&m_w2, a.W2, a.G + a.S, a.D, a.F, R2) || !make_map_2d(&m_h, a.h, h_rows, a.F, nbox))
            return cudaErrorInvalidValue;
        ring_geometry(true, true, a.T, &p);
        p.ksplit = 1; p.kblocks = kb1; p.R = R1; p.n_wtiles = (a.F + R1 - 1) / R1;
        if ((err = launch_gemm<DC_GEMM1>(m_xs, m_x, m_w1, m_w3, p, stream)) != cudaSuccess) return err;
        ring_geometry(true, false, a.T, &p);
        p.ksplit = ks2; p.kblocks = kb2 / ks2; p.R = R2; p.n_wtiles = (a.D + R2 - 1) / R2;
        if ((err = launch_gemm<DC_GEMM2>(m_h, m_h, m_w2, m_w2, p, stream)) != cudaSuccess) return err;
    }

    {
        const size_t n8 = (size_t)a.T * a.D / 8;
        int grid = (int)((n8 + 255) / 256);
        if (grid > sms * 8) grid = sms * 8;
        if (grid < 1) grid = 1;
        profile_begin(BM_KERNEL_FINALIZE, stream);
        cudaError_t e = launch_kernel(finalize_kernel, dim3(grid), dim3(256), 0, stream, (const float *)a.out_acc, a.out, n8);
        profile_end(BM_KERNEL_FINALIZE, stream);
        return e;
    }
}

}  // namespace bm
