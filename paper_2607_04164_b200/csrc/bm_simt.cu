// bm_simt.cu -- BM_PATH_SIMT: the forward pass on plain CUDA cores (fp32 FMA, one warp per output
// element).  A debugging cross-check for the tensor-core paths; never selected by BM_PATH_AUTO and never
// benchmarked as the product.  Same math as steps 10-12 (A3, A11, A12),
// including the bf16 rounding of the intermediate h.
#include "bm_common.cuh"

namespace bm {

namespace {

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
    return v;
}

__device__ __forceinline__ void dot8(const uint4 &a, const uint4 &b, float &acc) {
    acc = fmaf(bf16_lo(a.x), bf16_lo(b.x), acc); acc = fmaf(bf16_hi(a.x), bf16_hi(b.x), acc);
    acc = fmaf(bf16_lo(a.y), bf16_lo(b.y), acc); acc = fmaf(bf16_hi(a.y), bf16_hi(b.y), acc);
    acc = fmaf(bf16_lo(a.z), bf16_lo(b.z), acc); acc = fmaf(bf16_hi(a.z), bf16_hi(b.z), acc);
    acc = fmaf(bf16_lo(a.w), bf16_lo(b.w), acc); acc = fmaf(bf16_hi(a.w), bf16_hi(b.w), acc);
}

// H[hrow, f] for every routed row (hrow = permuted row) and every shared row (hrow = TK + j*T + t)
__global__ void __launch_bounds__(256)
simt_gemm1_kernel(const bm_bf16 *__restrict__ x, int T, int D, int F, int K, int G, int S,
                  const int32_t *__restrict__ offsets, const int32_t *__restrict__ row_token,
                  const bm_bf16 *__restrict__ W1, const bm_bf16 *__restrict__ W3, bm_bf16 *__restrict__ h) {
    const int lane = threadIdx.x & 31;
    const int TK = T * K;
    const int A = min(offsets[G], TK);
    const long long n_rows = (long long)A + (long long)S * T;
    const long long total = n_rows * F;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < total; w += warps) {
        const long long ri = w / F;
        const int f = (int)(w % F);
        int u, t;
        long long hrow;
        if (ri < A) {
            hrow = ri;
            t = row_token[ri];
            int lo = 0, hi = G - 1;                 // group of row ri: last u with offsets[u] <= ri
            while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (offsets[mid] <= ri) lo = mid; else hi = mid - 1; }
            u = lo;
        } else {
            const long long si = ri - A;
            u = G + (int)(si / T);
            t = (int)(si % T);
            hrow = (long long)TK + si;
        }
        const uint4 *xv = reinterpret_cast<const uint4 *>(x + (size_t)t * D);
        const uint4 *w1 = reinterpret_cast<const uint4 *>(W1 + ((size_t)u * F + f) * D);
        const uint4 *w3 = reinterpret_cast<const uint4 *>(W3 + ((size_t)u * F + f) * D);
        float a = 0.f, b = 0.f;
        for (int i = lane; i < D / 8; i += 32) {
            const uint4 xx = __ldg(xv + i);
            dot8(xx, __ldg(w1 + i), a);
            dot8(xx, __ldg(w3 + i), b);
        }
        a = warp_sum(a);
        b = warp_sum(b);
        if (lane == 0) h[(size_t)hrow * F + f] = (bm_bf16)f32_to_bf16_bits(a / (1.0f + expf(-a)) * b);
    }
}

// out[t, d] = sum_s gate_w[t,s] * (H[slot_row[t,s]] . W2[group_ids[t,s]]_d) + sum_j H[TK + j*T + t] . W2[G+j]_d
__global__ void __launch_bounds__(256)
simt_gemm2_kernel(int T, int D, int F, int K, int G, int S, const int32_t *__restrict__ group_ids,
                  const float *__restrict__ gate_w, const int32_t *__restrict__ n_slots,
                  const int32_t *__restrict__ slot_row, const bm_bf16 *__restrict__ W2,
                  const bm_bf16 *__restrict__ h, bm_bf16 *__restrict__ out) {
    const int lane = threadIdx.x & 31;
    const long long total = (long long)T * D;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < total; w += warps) {
        const int t = (int)(w / D), d = (int)(w % D);
        float o = 0.f;
        const int n = min(max(n_slots[t], 0), K);
        for (int s = 0; s < n + S; ++s) {
            int u;
            long long hrow;
            float gw;
            if (s < n) {
                u = group_ids[(size_t)t * K + s];
                hrow = slot_row[(size_t)t * K + s];
                gw = gate_w[(size_t)t * K + s];
                if (u < 0 || u >= G || hrow < 0 || hrow >= (long long)T * K) continue;
            } else {
                u = G + (s - n);
                hrow = (long long)T * K + (long long)(s - n) * T + t;
                gw = 1.0f;
            }
            const uint4 *hv = reinterpret_cast<const uint4 *>(h + (size_t)hrow * F);
            const uint4 *w2 = reinterpret_cast<const uint4 *>(W2 + ((size_t)u * D + d) * F);
            float y = 0.f;
            for (int i = lane; i < F / 8; i += 32) dot8(__ldg(hv + i), __ldg(w2 + i), y);
            y = warp_sum(y);
            o = fmaf(gw, y, o);
        }
        if (lane == 0) out[(size_t)t * D + d] = (bm_bf16)f32_to_bf16_bits(o);
    }
}

}  // namespace

cudaError_t launch_forward_simt(const ForwardArgs &a, cudaStream_t stream) {
    const int grid = num_sms() * 8;
    simt_gemm1_kernel<<<grid, 256, 0, stream>>>(a.x, a.T, a.D, a.F, a.K, a.G, a.S, a.r.offsets, a.r.row_token,
                                                a.W1, a.W3, a.h);
    simt_gemm2_kernel<<<grid, 256, 0, stream>>>(a.T, a.D, a.F, a.K, a.G, a.S, a.r.group_ids, a.r.gate_w,
                                                a.r.n_slots, a.r.slot_row, a.W2, a.h, a.out);
    count_launch(2);
    return cudaGetLastError();
}

}  // namespace bm
