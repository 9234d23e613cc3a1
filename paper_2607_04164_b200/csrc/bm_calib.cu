// bm_calib.cu -- calibration forward kernels: the forward half of the reward evaluation
// of the grouping search (PAPER.md 4.2-4.3), which the paper reports as > 95% of the search time.
//
//   expert_hist_kernel   w_e = how often expert e is selected on the calibration tokens
//   gram_kernel          gram[e,e'] = <Y_e, Y_e'> over all calibration outputs, on tcgen05 (A19)
//   gram_finish_kernel   fixed-order sum of the per-CTA partial Gram tiles, cos = gram / (|Y_e| |Y_e'|)
//   mse_partial_kernel   Eq. 5 target t_k(x) = sum alpha_e f_e(x) and the squared error of a united expert
//   mse_finish_kernel    MSE_r, beta_r and MSE_total = sum beta_r MSE_r (Eq. 6); reading A20
// (the expert outputs f_e(x) themselves come from the grouped GEMM kernels: launch_expert_outputs, bm_gemm.cu)
#include "bm_common.cuh"
#include "bm_ptx.cuh"

namespace bm {

namespace {

// ---------------------------------------------------------------------------------------------------
// routing frequency
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
expert_hist_kernel(const int32_t *__restrict__ expert_ids, long long items, int E, int32_t *__restrict__ w) {
    __shared__ int s_h[BM_MAX_E];
    for (int e = threadIdx.x; e < E; e += blockDim.x) s_h[e] = 0;
    __syncthreads();
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < items; i += (long long)gridDim.x * blockDim.x) {
        const int e = expert_ids[i];
        if (e >= 0 && e < E) atomicAdd(&s_h[e], 1);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += blockDim.x)
        if (s_h[e]) atomicAdd(&w[e], s_h[e]);
}

// ---------------------------------------------------------------------------------------------------
// Gram matrix of the expert outputs.  Y is TOKEN-MAJOR, [T, E, D] bf16: the E rows of one token are D*2 bytes apart, so
// ONE TMA tile (3-D map {D, E, T}: 128 rows x 64 columns of one token; rows >= E are out of bounds and arrive as zeros)
// gathers from a few neighbouring DRAM pages and feeds the A and the B descriptor of tcgen05.mma.  CTA c owns the
// a contiguous run of k-blocks (k-block = (token, 64-column piece)) and keeps its 128 x N fp32 partial in TMEM until the
// end; partial tiles go to the workspace and are summed in CTA order.
// Round 1 took Y as [E, T*D]: the rows of a tile were 16 MB apart and the kernel ran at 3.5-3.7 TB/s (0.55 of the HBM copy
// rate) whatever E was -- a stand-alone TMA probe streams 7.0 TB/s at an 8 KB row stride and 4.5 TB/s at 8 MB.  Hence the
// token-major output of bm_expert_outputs.
// ---------------------------------------------------------------------------------------------------
constexpr int kGramThreads = 192;
constexpr int kGramStages = 12;
constexpr int kGramTile = 128 * 128;     // bytes: 128 rows x 64 bf16

__global__ void __launch_bounds__(kGramThreads, 1)
gram_kernel(const __grid_constant__ CUtensorMap tm_y, int E, int n_kblocks, int kb_per_token, float *__restrict__ partial) {
    extern __shared__ uint8_t g_smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(g_smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)kGramStages * kGramTile);
    uint64_t *empty = full + kGramStages;
    uint64_t *done = empty + kGramStages;
    uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(done + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N = (E + 15) & ~15;                       // MMA N: experts rounded up to 16

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tm_y);
        for (int i = 0; i < kGramStages; ++i) { ptx::mbar_init(&full[i], 1); ptx::mbar_init(&empty[i], 1); }
        ptx::mbar_init(done, 1);
        ptx::fence_barrier_init();
    }
    if (warp == 1) ptx::tmem_alloc(tmem_ptr, 128);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    // CTA c owns a CONTIGUOUS run of k-blocks: consecutive loads walk along the experts' rows of one token (whole DRAM pages)
    const int per_cta = (n_kblocks + gridDim.x - 1) / gridDim.x;
    const int kb0 = blockIdx.x * per_cta;
    const int my_kb = max(0, min(per_cta, n_kblocks - kb0));

    if (warp == 0) {
        int stage = 0;
        uint32_t phase = 0;
        for (int i = 0; i < my_kb; ++i) {
            ptx::mbar_wait(&empty[stage], phase ^ 1);
            if (ptx::elect_one()) {
                ptx::mbar_arrive_expect_tx(&full[stage], kGramTile);
                const int kbi = kb0 + i;                                // k-block = (token, 64-column piece of its D outputs)
                const int tok = kbi / kb_per_token;
                ptx::tma_load_3d(smem + (size_t)stage * kGramTile, &tm_y, &full[stage], (kbi - tok * kb_per_token) * 64, 0, tok,
                                 ptx::kEvictFirst);
            }
            __syncwarp();
            if (++stage == kGramStages) { stage = 0; phase ^= 1; }
        }
    } else if (warp == 1) {
        const uint32_t idesc = ptx::make_idesc_bf16(128, N);
        const uint32_t a_lo0 = ptx::smem_desc_lo(ptx::smem_u32(smem));
        int stage = 0;
        uint32_t phase = 0;
        for (int i = 0; i < my_kb; ++i) {
            ptx::mbar_wait(&full[stage], phase);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                const uint32_t a_lo = a_lo0 + stage * (kGramTile >> 4);
#pragma unroll
                for (int k = 0; k < 4; ++k)             // the same tile is the A and the B operand
                    ptx::mma_bf16_ss(tmem_base, ptx::smem_desc(a_lo + 2 * k), ptx::smem_desc(a_lo + 2 * k), idesc,
                                     (i | k) ? 1u : 0u);
                ptx::mma_commit(&empty[stage]);
                if (i == my_kb - 1) ptx::mma_commit(done);
            }
            __syncwarp();
            if (++stage == kGramStages) { stage = 0; phase ^= 1; }
        }
    } else {
        // epilogue: row e of the partial tile lives in TMEM lane e
        const int q = warp & 3;
        const int e = q * 32 + lane;
        float *prow = partial + ((size_t)blockIdx.x * E + e) * E;
        if (my_kb > 0) {
            ptx::mbar_wait(done, 0);
            ptx::tc_fence_after();
            for (int c = 0; c < N; c += 16) {
                uint32_t v[16];
                ptx::tmem_ld_x16(tmem_base + ((uint32_t)(q * 32) << 16) + c, v);
                ptx::tmem_ld_wait();
                if (e < E)
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        if (c + i < E) prow[c + i] = __uint_as_float(v[i]);
            }
        } else if (e < E) {
            for (int c = 0; c < E; ++c) prow[c] = 0.0f;
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, 128);
    }
}

// gram[e,e'] = sum of the per-CTA partial tiles in CTA order (deterministic); cos = gram / sqrt(gram[e,e] gram[e',e']).
// Block e owns row e; thread j sums element (e, j) and the diagonal element (j, j) it needs for the cosine.
__global__ void __launch_bounds__(128)
gram_finish_kernel(const float *__restrict__ partial, int n_cta, int E, float *__restrict__ gram,
                   float *__restrict__ cosine) {
    __shared__ float s_diag_e;
    const int e = blockIdx.x, j = threadIdx.x;
    float acc = 0.0f, dj = 0.0f;
    if (j < E) {
        const size_t ee = (size_t)E * E;
        const float *pr = partial + (size_t)e * E + j, *pd = partial + (size_t)j * E + j;
        int c = 0;
        for (; c + 4 <= n_cta; c += 4) {                 // four loads in flight, added in CTA order
            const float r0 = pr[c * ee], r1 = pr[(c + 1) * ee], r2 = pr[(c + 2) * ee], r3 = pr[(c + 3) * ee];
            const float d0 = pd[c * ee], d1 = pd[(c + 1) * ee], d2 = pd[(c + 2) * ee], d3 = pd[(c + 3) * ee];
            acc = (((acc + r0) + r1) + r2) + r3;
            dj = (((dj + d0) + d1) + d2) + d3;
        }
        for (; c < n_cta; ++c) { acc += pr[c * ee]; dj += pd[c * ee]; }
        gram[(size_t)e * E + j] = acc;
        if (j == e) s_diag_e = dj;
    }
    __syncthreads();
    if (cosine && j < E) {
        const float d = s_diag_e * dj;
        cosine[(size_t)e * E + j] = d > 0.0f ? acc * rsqrtf(d) : 0.0f;
    }
}

// ---------------------------------------------------------------------------------------------------
// Eq. 5 / Eq. 6.  Block (bx, r): the members of group r and their alpha_e = w_e / sum_{G_r} w (uniform if the
// group was never selected, A20) go to shared memory; a thread owns 8 consecutive elements of the [T*D]
// output plane: target = sum alpha_e Y[e], err = (U[r] - target)^2, block sum -> part[r][bx] (fp32; the finish
// kernel adds the blocks in index order in fp64).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
mse_partial_kernel(const bm_bf16 *__restrict__ Y, const bm_bf16 *__restrict__ U, size_t n8, size_t d8,
                   const int32_t *__restrict__ w, const int32_t *__restrict__ gmap, int E, int G,
                   float *__restrict__ part) {
    __shared__ int32_t s_member[BM_MAX_E];
    __shared__ float s_alpha[BM_MAX_E];
    __shared__ int s_cnt;
    __shared__ float s_red[8];
    const int r = blockIdx.y;
    if (threadIdx.x == 0) {
        int c = 0;
        long long wsum = 0;
        for (int e = 0; e < E; ++e)
            if (gmap[e] == r) { s_member[c++] = e; wsum += w[e]; }
        for (int m = 0; m < c; ++m)
            s_alpha[m] = wsum > 0 ? (float)((double)w[s_member[m]] / (double)wsum) : 1.0f / (float)c;
        s_cnt = c;
    }
    __syncthreads();
    const int cnt = s_cnt;
    float err = 0.0f;
    if (cnt > 0) {
        // token-major layouts: Y [T, E, D], U [T, G, D]; i walks the (token, 8-column piece) pairs
        const uint4 *Y4 = reinterpret_cast<const uint4 *>(Y);
        const uint4 *U4 = reinterpret_cast<const uint4 *>(U);
        const size_t n_tok = n8 / d8;
        for (size_t tok = blockIdx.x; tok < n_tok; tok += gridDim.x)
        for (size_t c = threadIdx.x; c < d8; c += blockDim.x) {
            float t[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) t[k] = 0.0f;
            for (int m = 0; m < cnt; ++m) {
                const uint4 v = __ldg(Y4 + (tok * E + s_member[m]) * d8 + c);
                const float a = s_alpha[m];
                t[0] = fmaf(a, bf16_lo(v.x), t[0]); t[1] = fmaf(a, bf16_hi(v.x), t[1]);
                t[2] = fmaf(a, bf16_lo(v.y), t[2]); t[3] = fmaf(a, bf16_hi(v.y), t[3]);
                t[4] = fmaf(a, bf16_lo(v.z), t[4]); t[5] = fmaf(a, bf16_hi(v.z), t[5]);
                t[6] = fmaf(a, bf16_lo(v.w), t[6]); t[7] = fmaf(a, bf16_hi(v.w), t[7]);
            }
            const uint4 u = __ldg(U4 + (tok * G + r) * d8 + c);
            const float d0 = bf16_lo(u.x) - t[0], d1 = bf16_hi(u.x) - t[1], d2 = bf16_lo(u.y) - t[2], d3 = bf16_hi(u.y) - t[3];
            const float d4 = bf16_lo(u.z) - t[4], d5 = bf16_hi(u.z) - t[5], d6 = bf16_lo(u.w) - t[6], d7 = bf16_hi(u.w) - t[7];
            err += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3 + d4 * d4 + d5 * d5 + d6 * d6 + d7 * d7;
        }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) err += __shfl_xor_sync(kFullMask, err, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = err;
    __syncthreads();
    if (threadIdx.x == 0) {
        float s = 0.0f;
        for (int i = 0; i < 8; ++i) s += s_red[i];
        part[(size_t)r * gridDim.x + blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(256)
mse_finish_kernel(const float *__restrict__ part, int nblk, int T, const int32_t *__restrict__ w,
                  const int32_t *__restrict__ gmap, int E, int G, float *__restrict__ mse,
                  float *__restrict__ mse_total) {
    __shared__ double s_term[BM_MAX_G];
    long long wall = 0;
    for (int e = 0; e < E; ++e) wall += w[e];
    for (int r = threadIdx.x; r < G; r += blockDim.x) {
        double s = 0.0;
        for (int b = 0; b < nblk; ++b) s += (double)part[(size_t)r * nblk + b];
        const double m = T > 0 ? s / (double)T : 0.0;
        long long wr = 0;
        for (int e = 0; e < E; ++e)
            if (gmap[e] == r) wr += w[e];
        mse[r] = (float)m;
        s_term[r] = wall > 0 ? (double)wr / (double)wall * m : 0.0;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int r = 0; r < G; ++r) tot += s_term[r];        // group order
        *mse_total = (float)tot;
    }
}

}  // namespace

cudaError_t launch_expert_hist(const int32_t *expert_ids, long long items, int E, int32_t *w, cudaStream_t stream) {
    cudaError_t e = cudaMemsetAsync(w, 0, sizeof(int32_t) * E, stream);
    if (e != cudaSuccess || items == 0) return e;
    long long grid = (items + 255) / 256;
    if (grid > num_sms() * 4) grid = num_sms() * 4;
    expert_hist_kernel<<<(unsigned)grid, 256, 0, stream>>>(expert_ids, items, E, w);
    count_launch();
    return cudaGetLastError();
}

size_t gram_workspace_bytes(int E) { return (size_t)num_sms() * E * E * sizeof(float); }

cudaError_t launch_gram(const bm_bf16 *Y, int E, int T, int D, float *gram, float *cosine, float *partial,
                        cudaStream_t stream) {
    // Y [T, E, D]: a tile = the E rows of one token (4 KB apart at D = 2048) x 64 columns; rows >= E are out of bounds -> zeros
    CUtensorMap tm;
    if (!make_map_3d_sw128(&tm, Y, (uint64_t)T, (uint64_t)E, (uint64_t)D, 128)) return cudaErrorInvalidValue;
    const int kpt = (D + 63) / 64;
    const long long nkb = (long long)T * kpt;
    const int grid = (int)(nkb < num_sms() ? nkb : num_sms());
    const size_t smem = 1024 + (size_t)kGramStages * kGramTile + 256;
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(gram_kernel), smem); ea != cudaSuccess) return ea;
    gram_kernel<<<grid, kGramThreads, smem, stream>>>(tm, E, (int)nkb, kpt, partial);
    gram_finish_kernel<<<E, 128, 0, stream>>>(partial, grid, E, gram, cosine);
    count_launch(2);
    return cudaGetLastError();
}

int mse_blocks() { return num_sms() * 8; }

cudaError_t launch_group_mse(const bm_bf16 *Y, const bm_bf16 *U, int T, int D, const int32_t *w, const int32_t *gmap,
                             int E, int G, float *mse, float *mse_total, float *part, cudaStream_t stream) {
    const size_t n8 = (size_t)T * D / 8;
    int nblk = (int)((n8 + 255) / 256);
    const int cap = mse_blocks() / G + 1;
    if (nblk > cap) nblk = cap;
    if (nblk < 1) nblk = 1;
    mse_partial_kernel<<<dim3(nblk, G), 256, 0, stream>>>(Y, U, n8, (size_t)(D / 8), w, gmap, E, G, part);
    mse_finish_kernel<<<1, 256, 0, stream>>>(part, nblk, T, w, gmap, E, G, mse, mse_total);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace bm
