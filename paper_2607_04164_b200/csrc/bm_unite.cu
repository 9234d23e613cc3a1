// bm_unite.cu -- united-weight construction: the parameter average of the member
// experts of every group, the initialisation of a united expert before distillation.
//
// Cite: "The united expert is initialized as the parameter average of member experts";
// PAPER.md:118-122 (Eq. 2) for the group map.  out[u, i] = (1/|G_u|) * sum_{e: gmap[e] = u} W[e, i]:
// members added in ascending e in fp32, one division, one rounding to bf16.  A bandwidth kernel: each
// weight element is read once and each united element written once (E + G elements of traffic per G written).
#include "bm_common.cuh"

namespace bm {

namespace {

__global__ void __launch_bounds__(256)
unite_kernel(const bm_bf16 *__restrict__ W, int E, size_t n8, const int32_t *__restrict__ gmap, int G,
             bm_bf16 *__restrict__ out) {
    __shared__ int32_t s_members[BM_MAX_E];
    __shared__ int s_count;
    grid_dep_wait();
    grid_dep_launch();
    const int u = blockIdx.y;
    if (threadIdx.x == 0) {
        int c = 0;
        for (int e = 0; e < E; ++e)
            if (gmap[e] == u) s_members[c++] = e;       // ascending e
        s_count = c;
    }
    __syncthreads();
    const int cnt = s_count;
    const float inv = cnt > 0 ? 1.0f : 0.0f;
    const uint4 *W4 = reinterpret_cast<const uint4 *>(W);
    uint4 *o4 = reinterpret_cast<uint4 *>(out) + (size_t)u * n8;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
        float acc[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = 0.0f;
        int m = 0;
        for (; m + 4 <= cnt; m += 4) {                   // four members in flight
            uint4 v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) v[q] = __ldg(W4 + (size_t)s_members[m + q] * n8 + i);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                acc[0] += bf16_lo(v[q].x); acc[1] += bf16_hi(v[q].x); acc[2] += bf16_lo(v[q].y); acc[3] += bf16_hi(v[q].y);
                acc[4] += bf16_lo(v[q].z); acc[5] += bf16_hi(v[q].z); acc[6] += bf16_lo(v[q].w); acc[7] += bf16_hi(v[q].w);
            }
        }
        for (; m < cnt; ++m) {
            const uint4 v = __ldg(W4 + (size_t)s_members[m] * n8 + i);
            acc[0] += bf16_lo(v.x); acc[1] += bf16_hi(v.x); acc[2] += bf16_lo(v.y); acc[3] += bf16_hi(v.y);
            acc[4] += bf16_lo(v.z); acc[5] += bf16_hi(v.z); acc[6] += bf16_lo(v.w); acc[7] += bf16_hi(v.w);
        }
        const float d = cnt > 0 ? (float)cnt : 1.0f;
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = inv * (acc[k] / d);
        o4[i] = make_uint4(pack_bf16x2(acc[0], acc[1]), pack_bf16x2(acc[2], acc[3]), pack_bf16x2(acc[4], acc[5]),
                           pack_bf16x2(acc[6], acc[7]));
    }
}

}  // namespace

cudaError_t launch_unite(const bm_bf16 *W, int E, size_t n, const int32_t *gmap, int G, bm_bf16 *out,
                         cudaStream_t stream) {
    const size_t n8 = n / 8;
    size_t gx = (n8 + 255) / 256;
    const size_t cap = (size_t)num_sms() * 16 / (size_t)G + 1;
    if (gx > cap) gx = cap;
    if (gx < 1) gx = 1;
    return launch_kernel(unite_kernel, dim3((unsigned)gx, (unsigned)G), dim3(256), 0, stream, W, E, n8, gmap, G, out);
}

}  // namespace bm
