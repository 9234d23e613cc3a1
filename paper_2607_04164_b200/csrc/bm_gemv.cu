// bm_gemv.cu -- BM_PATH_GEMV: steps 10-12 for very small batches (a weight set meets about one token row:
// single-token decode; BM_PATH_AUTO: T <= 2 and T*K <= G) as weight-streaming matrix-vector products on the CUDA cores.
//
// Cite: PAPER.md:42 (expert FFN, gate-weighted sum), PAPER.md:46 (united experts cut "the number of experts
// loaded during inference": at these sizes the layer IS the weight load), A3, A11, A12.
//
// Why not the tcgen05 decode path here: its k-block loop has a floor of ~0.3 us per 64 columns whatever
// the tile holds, so one token on four groups costs 12 + 7 us of MMA pipeline for 7 + 3.5 us of HBM time,
// plus a gather/schedule kernel and TMEM/tensor-map set-up in each GEMM.  With <= 8 rows per weight set the
// FMA work is a few percent of the CUDA cores' rate, so plain 128-bit streaming loads with FFMA2 keep up
// with HBM and the kernels start at once.
//
// Both products are one kernel template.  A "unit" q of a weight set u is a pair of weight rows that
// share one FFMA2 per element:
//   SWIGLU:  rows W1[u][q,:] and W3[u][q,:]  (q < F, input x rows, length D)   -> h[r,q] = SiLU(a) * b
//   plain :  rows W2[u][2q,:] and W2[u][2q+1,:] (q < D/2, input h rows, length F) -> y[r,2q], y[r,2q+1]
// The active sets' units form one index space that is cut into equal contiguous ranges, one per CTA (the
// counts are read on the device; the host never sees them).  A CTA stages the <= 8 input rows of the set
// in shared memory, then each warp takes units q, q + warps, ...: lane l streams the 16-byte chunks l,
// l+32, ... of both weight rows (software-pipelined, see warp_units), multiplies them into one fp32 accumulator
// pair per input row, and the warp adds the lane partials with a shuffle butterfly.  A set with more than
// 8 rows takes several passes over its weights (correct, slower; BM_PATH_AUTO does not send such shapes
// here).  The W2 stage is normally the fused token-major kernel below (gemv2_combine_kernel); the set-major plain
// kernel writing bf16 y rows + the prefill path's combine_kernel remain as the fallback for huge K + S or F.
#include <algorithm>

#include "bm_common.cuh"
#include "bm_ptx.cuh"
#include "bm_router.cuh"

namespace bm {

namespace {

constexpr int kGvThreads = 512;
constexpr int kGvWarps = kGvThreads / 32;
constexpr int kGvRows = 8;          // input rows staged per pass

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void fma2(float &d0, float &d1, float x, float w0, float w1) {
    uint64_t a, b, c;
    asm("mov.b64 %0, {%1, %1};" : "=l"(a) : "f"(x));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(w0), "f"(w1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(d0), "f"(d1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(c));
}

// One warp's units q0, q0 + warps, ... < qb of one weight set against the R staged input rows (R: compile time).
// The weight stream is software-pipelined: the loads of step s + 1 (a step = U chunks per lane of both rows;
// the next step may belong to the next unit) are issued before the multiply of step s, from two register
// buffers, so a warp always has a step of loads in flight -- without it every step paid a full HBM latency
// (measured: 3 TB/s instead of 6 at T = 16, G = 60).  Staging the stream through per-lane cp.async rings in shared memory (8 KB
// per warp in flight instead of 4 KB) was measured too and was slower (single-token layer 26.6 -> 28 us).
template <int R, bool SWIGLU, typename StageFn>
__device__ __forceinline__ void warp_units(StageFn stage_rows, const bm_bf16 *__restrict__ base_a, const bm_bf16 *__restrict__ base_b,
                                           size_t stride_q, int n8, int q0, int qb, const uint8_t *s_in, int in_bytes,
                                           int lane, int nr, bm_bf16 *__restrict__ outp, size_t orow0, int OUT) {
    constexpr int U = R <= 4 ? 4 : 2;           // chunks of each row per lane and step (fewer with 8 rows: registers)
    const int iters = (n8 + 32 * U - 1) / (32 * U);
    float acc[R][2];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r][0] = acc[r][1] = 0.0f;

    // (always writes the buffers -- a conditionally written register array ends up in local memory)
    auto load = [&](bool on, int q, int it, uint4 (&va)[U], uint4 (&vb)[U]) {
        const uint4 *wa = reinterpret_cast<const uint4 *>(base_a + (size_t)q * stride_q);
        const uint4 *wb = reinterpret_cast<const uint4 *>(base_b + (size_t)q * stride_q);
#pragma unroll
        for (int i = 0; i < U; ++i) {
            const int c = (it * U + i) * 32 + lane;
            const bool ok = on && c < n8;
            va[i] = ok ? ld_stream(wa + c) : make_uint4(0u, 0u, 0u, 0u);
            vb[i] = ok ? ld_stream(wb + c) : make_uint4(0u, 0u, 0u, 0u);
        }
    };
    auto compute = [&](int it, const uint4 (&va)[U], const uint4 (&vb)[U]) {
#pragma unroll
        for (int i = 0; i < U; ++i) {
            const int c = (it * U + i) * 32 + lane;
            if (c < n8) {
                const uint32_t a[4] = {va[i].x, va[i].y, va[i].z, va[i].w};
                const uint32_t b[4] = {vb[i].x, vb[i].y, vb[i].z, vb[i].w};
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const uint4 xv = *reinterpret_cast<const uint4 *>(s_in + (size_t)r * in_bytes + (size_t)c * 16);
                    const uint32_t x[4] = {xv.x, xv.y, xv.z, xv.w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        fma2(acc[r][0], acc[r][1], bf16_lo(x[k]), bf16_lo(a[k]), bf16_lo(b[k]));
                        fma2(acc[r][0], acc[r][1], bf16_hi(x[k]), bf16_hi(a[k]), bf16_hi(b[k]));
                    }
                }
            }
        }
    };
    auto finish = [&](int q) {          // lane r keeps and stores the sums of row r; rows past nr are dropped
        float ma = 0.0f, mb = 0.0f;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float a = acc[r][0], b = acc[r][1];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) {
                a += __shfl_xor_sync(kFullMask, a, o);
                b += __shfl_xor_sync(kFullMask, b, o);
            }
            if (lane == r) { ma = a; mb = b; }
            acc[r][0] = acc[r][1] = 0.0f;
        }
        if (lane < nr) {
            const size_t orow = (orow0 + (size_t)lane) * (size_t)OUT;
            if (SWIGLU) outp[orow + q] = (bm_bf16)f32_to_bf16_bits(ma / (1.0f + expf(-ma)) * mb);
            else *reinterpret_cast<uint32_t *>(outp + orow + 2 * (size_t)q) = pack_bf16x2(ma, mb);
        }
    };

    uint4 a0[U], b0[U], a1[U], b1[U];
    int q = q0, it = 0;
    load(q < qb, q, 0, a0, b0);
    // the input rows are staged (by all threads of the CTA) while this first step of weight loads is in flight: the
    // weights do not depend on them, and the staging is two dependent global round trips (row_token -> x row)
    stage_rows();
    while (q < qb) {
        int qn = q, itn = it + 1;
        if (itn == iters) { itn = 0; qn += kGvWarps; }
        load(qn < qb, qn, itn, a1, b1);
        compute(it, a0, b0);
        if (it == iters - 1) finish(q);
        q = qn; it = itn;
        if (q >= qb) break;
        qn = q; itn = it + 1;
        if (itn == iters) { itn = 0; qn += kGvWarps; }
        load(qn < qb, qn, itn, a0, b0);
        compute(it, a1, b1);
        if (it == iters - 1) finish(q);
        q = qn; it = itn;
    }
}

struct GemvArgs {
    const bm_bf16 *in;          // SWIGLU: x [T, IN]; plain: h [TK + S*T, IN]
    const bm_bf16 *Wa, *Wb;     // SWIGLU: W1, W3 [G+S, F, D]; plain: W2 twice [G+S, D, F]
    bm_bf16 *outp;              // SWIGLU: h [TK + S*T, F]; plain: y [TK + S*T, D]
    const int32_t *offsets;     // [G+1]
    const int32_t *row_token;   // [TK]
    int T, TK, G, S;
    int IN;                     // length of an input row (D or F)
    int OUT;                    // length of an output row (F or D)
    int NQ;                     // units per set (F or D/2)
};

// (body of gemv_kernel; also one phase of layer_small_kernel, where p.offsets / p.row_token point into shared memory)
template <bool SWIGLU>
__device__ __forceinline__ void gemv_body(const GemvArgs &p, int rows_cap, uint8_t *gv_smem) {
    __shared__ int s_nact;
    const int in_bytes = p.IN * 2, n8 = p.IN / 8;
    uint8_t *s_in = gv_smem;                                              // [rows_cap][IN] bf16
    int *s_set = reinterpret_cast<int *>(gv_smem + (size_t)rows_cap * in_bytes);   // active sets, ascending
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nsets = p.G + p.S;

    if (warp == 0) {
        int n = 0;
        for (int base = 0; base < nsets; base += 32) {
            const int u = base + lane;
            bool act = false;
            if (u < nsets) act = (u < p.G ? p.offsets[u + 1] - p.offsets[u] : p.T) > 0;
            const unsigned m = __ballot_sync(kFullMask, act);
            if (act) s_set[n + __popc(m & ((1u << lane) - 1u))] = u;
            n += __popc(m);
        }
        if (lane == 0) s_nact = n;
    }
    __syncthreads();
    const long long total = (long long)s_nact * p.NQ;
    const long long per = (total + gridDim.x - 1) / gridDim.x;
    const long long lo = (long long)blockIdx.x * per;
    const long long hi = lo + per < total ? lo + per : total;

    for (long long pos = lo; pos < hi;) {
        const int k = (int)(pos / p.NQ);
        const int u = s_set[k];
        const int qa = (int)(pos - (long long)k * p.NQ);
        const int qb = (int)((hi - pos) < (long long)(p.NQ - qa) ? qa + (hi - pos) : p.NQ);
        long long row0;
        int cnt;
        if (u < p.G) {
            row0 = p.offsets[u];
            cnt = p.offsets[u + 1] - (int)row0;
            if (row0 < 0 || row0 > p.TK) cnt = 0;
            if (cnt > p.TK - (int)row0) cnt = p.TK - (int)row0;
        } else {
            row0 = (long long)p.TK + (long long)(u - p.G) * p.T;
            cnt = p.T;
        }
        for (int base = 0; base < cnt; base += rows_cap) {
            const int nr = cnt - base < rows_cap ? cnt - base : rows_cap;
            auto stage_rows = [&]() {
                __syncthreads();                               // the readers of the rows staged before are done
                for (int idx = tid; idx < nr * n8; idx += kGvThreads) {
                    const int r = idx / n8, c = idx - r * n8;
                    long long src;
                    if (SWIGLU) {
                        int tok = u < p.G ? p.row_token[row0 + base + r] : base + r;
                        tok = tok < 0 ? 0 : (tok >= p.T ? p.T - 1 : tok);
                        src = tok;
                    } else {
                        src = row0 + base + r;
                    }
                    *reinterpret_cast<uint4 *>(s_in + (size_t)r * in_bytes + (size_t)c * 16) =
                        __ldg(reinterpret_cast<const uint4 *>(p.in + (size_t)src * p.IN) + c);
                }
                __syncthreads();
            };
            const bm_bf16 *base_a, *base_b;
            size_t stride_q;
            if (SWIGLU) {
                base_a = p.Wa + (size_t)u * p.NQ * p.IN;
                base_b = p.Wb + (size_t)u * p.NQ * p.IN;
                stride_q = (size_t)p.IN;
            } else {
                base_a = p.Wa + (size_t)u * p.OUT * p.IN;
                base_b = base_a + p.IN;
                stride_q = 2 * (size_t)p.IN;
            }
            const size_t orow0 = (size_t)(row0 + base);
            // rows past nr (up to the next power of two) are stale shared memory: computed, never stored
            if (nr == 1) warp_units<1, SWIGLU>(stage_rows, base_a, base_b, stride_q, n8, qa + warp, qb, s_in, in_bytes, lane, nr, p.outp, orow0, p.OUT);
            else if (nr == 2) warp_units<2, SWIGLU>(stage_rows, base_a, base_b, stride_q, n8, qa + warp, qb, s_in, in_bytes, lane, nr, p.outp, orow0, p.OUT);
            else if (nr <= 4) warp_units<4, SWIGLU>(stage_rows, base_a, base_b, stride_q, n8, qa + warp, qb, s_in, in_bytes, lane, nr, p.outp, orow0, p.OUT);
            else warp_units<8, SWIGLU>(stage_rows, base_a, base_b, stride_q, n8, qa + warp, qb, s_in, in_bytes, lane, nr, p.outp, orow0, p.OUT);
        }
        pos += qb - qa;
    }
}

template <bool SWIGLU>
__global__ void __launch_bounds__(kGvThreads, 1)
gemv_kernel(GemvArgs p, int rows_cap) {
    extern __shared__ __align__(16) uint8_t gv_smem[];
    grid_dep_wait();      // routing arrays, x / h come from predecessors
    grid_dep_launch();
    gemv_body<SWIGLU>(p, rows_cap, gv_smem);
}

template <bool SWIGLU>
cudaError_t launch_gemv(const GemvArgs &p, int kid, cudaStream_t stream) {
    int rows_cap = kGvRows;
    while (rows_cap > 1 && (size_t)rows_cap * p.IN * 2 > 200 * 1024) rows_cap >>= 1;
    const size_t smem = (size_t)rows_cap * p.IN * 2 + (size_t)(p.G + p.S) * sizeof(int);
    if (smem > 220 * 1024) return cudaErrorInvalidValue;
    auto kern = gemv_kernel<SWIGLU>;
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(kern), smem); ea != cudaSuccess) return ea;
    profile_begin(kid, stream);
    cudaError_t e = launch_kernel(kern, dim3(num_sms()), dim3(kGvThreads), smem, stream, p, rows_cap);
    profile_end(kid, stream);
    return e;
}

// -------------------------------------------------------------------------------------------------
// W2 stage and gate-weighted combine in one kernel (token-major): a CTA owns a range of output column pairs of
// one token; its units are (source s, column pair q): rows W2[u_s][2q], W2[u_s][2q+1] against the source's h row.
// A warp walks its units in one software-pipelined stream (as warp_units), parks (y[2q], y[2q+1]) of every
// source in shared memory as fp32, and after a barrier the CTA adds them in slot order with the gate weights
// and stores bf16 out (or the fp32 sums for the tensor-parallel partial) -- no y rows in global memory and no
// combine launch (3 of the ~30 us of a single-token step).  Deterministic: fixed slot order, one warp per unit.
// -------------------------------------------------------------------------------------------------
struct Gemv2Args {
    const bm_bf16 *h;           // [TK + S*T, F]
    const bm_bf16 *W2;          // [G+S, D, F]
    bm_bf16 *out;               // [T, D] or nullptr
    float *out_f32;             // [T, D] or nullptr
    const int32_t *group_ids, *slot_row, *n_slots;
    const float *gate_w;
    int T, K, G, S, D, F;
};

// (body of gemv2_combine_kernel; also one phase of layer_small_kernel.  COHERENT_H: h was written earlier in the SAME
//  kernel by other CTAs, so it must not be read through the non-coherent path)
template <bool COHERENT_H, int U = 4>
__device__ __forceinline__ void gemv2_combine_body(const Gemv2Args &p, int max_src, int max_q, uint8_t *gv_smem) {
    __shared__ int s_u[32], s_row[32];
    __shared__ float s_gw[32];
    const int in_bytes = p.F * 2, n8 = p.F / 8, NQ = p.D / 2;
    uint8_t *s_in = gv_smem;                                                   // [max_src][F] bf16
    float *s_y = reinterpret_cast<float *>(gv_smem + (size_t)max_src * in_bytes);   // [max_src][2 * max_q]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long TK = (long long)p.T * p.K;
    const long long total = (long long)p.T * NQ;
    const long long per = (total + gridDim.x - 1) / gridDim.x;      // <= max_q by the host's choice
    const long long lo = (long long)blockIdx.x * per;
    const long long hi = lo + per < total ? lo + per : total;
    // U = chunks of each row per lane and step.  With F <= 1536 (n8 <= 192) U = 6 makes a unit one step, so a warp -- which
    // only has one or two units here -- has all of a unit's loads in flight at once
    const int iters = (n8 + 32 * U - 1) / (32 * U);

    for (long long pos = lo; pos < hi;) {
        const int t = (int)(pos / NQ);
        const int qa = (int)(pos - (long long)t * NQ);
        const int qb = (int)((hi - pos) < (long long)(NQ - qa) ? qa + (hi - pos) : NQ);
        const int nq = qb - qa;
        __syncthreads();                                   // the previous segment's tables and buffers are free
        int n_src = min(max(p.n_slots[t], 0), p.K) + p.S;
        n_src = n_src < max_src ? n_src : max_src;
        if (tid < 32) {
            const int n = n_src - p.S;
            int u = 0, row = -1;
            float gw = 0.0f;
            if (tid < n) {
                u = p.group_ids[(size_t)t * p.K + tid];
                row = p.slot_row[(size_t)t * p.K + tid];
                gw = p.gate_w[(size_t)t * p.K + tid];
                if (u < 0 || u >= p.G || row < 0 || row >= TK) { u = 0; row = -1; gw = 0.0f; }
            } else if (tid < n_src) {
                u = p.G + (tid - n);
                row = (int)(TK + (long long)(tid - n) * p.T + t);
                gw = 1.0f;
            }
            s_u[tid] = u; s_row[tid] = row; s_gw[tid] = gw;
        }
        __syncthreads();
        const int n_units = n_src * nq;                    // unit v = (source v / nq, column pair qa + v % nq)
        float acc0 = 0.0f, acc1 = 0.0f;
        auto load = [&](bool on, int v, int it, uint4 (&va)[U], uint4 (&vb)[U]) {
            const int sidx = on ? v / nq : 0;
            const int q = qa + v - sidx * nq;
            const uint4 *wa = reinterpret_cast<const uint4 *>(p.W2 + ((size_t)s_u[sidx] * p.D + 2 * (size_t)q) * p.F);
            const uint4 *wb = wa + n8;
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int c = (it * U + i) * 32 + lane;
                const bool ok = on && c < n8 && s_row[sidx] >= 0;
                va[i] = ok ? ld_stream(wa + c) : make_uint4(0u, 0u, 0u, 0u);
                vb[i] = ok ? ld_stream(wb + c) : make_uint4(0u, 0u, 0u, 0u);
            }
        };
        auto compute = [&](int v, int it, const uint4 (&va)[U], const uint4 (&vb)[U]) {
            const int sidx = v / nq;
            const uint8_t *xrow = s_in + (size_t)sidx * in_bytes;
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int c = (it * U + i) * 32 + lane;
                if (c < n8) {
                    const uint32_t a[4] = {va[i].x, va[i].y, va[i].z, va[i].w};
                    const uint32_t b[4] = {vb[i].x, vb[i].y, vb[i].z, vb[i].w};
                    const uint4 xv = *reinterpret_cast<const uint4 *>(xrow + (size_t)c * 16);
                    const uint32_t x[4] = {xv.x, xv.y, xv.z, xv.w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        fma2(acc0, acc1, bf16_lo(x[k]), bf16_lo(a[k]), bf16_lo(b[k]));
                        fma2(acc0, acc1, bf16_hi(x[k]), bf16_hi(a[k]), bf16_hi(b[k]));
                    }
                }
            }
        };
        auto finish = [&](int v) {
            float a = acc0, b = acc1;
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) {
                a += __shfl_xor_sync(kFullMask, a, o);
                b += __shfl_xor_sync(kFullMask, b, o);
            }
            if (lane == 0) {
                const int sidx = v / nq;
                *reinterpret_cast<float2 *>(s_y + ((size_t)sidx * max_q + (v - sidx * nq)) * 2) = make_float2(a, b);
            }
            acc0 = acc1 = 0.0f;
        };
        uint4 a0[U], b0[U], a1[U], b1[U];
        int v = warp, it = 0;
        load(v < n_units, v, 0, a0, b0);
        // stage the sources' h rows while the first weight loads are in flight (invalid sources: zeros)
        for (int idx = tid; idx < n_src * n8; idx += kGvThreads) {
            const int r = idx / n8, c = idx - r * n8;
            const int row = s_row[r];
            const uint4 *hp = reinterpret_cast<const uint4 *>(p.h + (size_t)(row >= 0 ? row : 0) * p.F) + c;
            *reinterpret_cast<uint4 *>(s_in + (size_t)r * in_bytes + (size_t)c * 16) =
                row >= 0 ? (COHERENT_H ? __ldcg(hp) : __ldg(hp)) : make_uint4(0u, 0u, 0u, 0u);
        }
        __syncthreads();
        while (v < n_units) {
            int vn = v, itn = it + 1;
            if (itn == iters) { itn = 0; vn += kGvWarps; }
            load(vn < n_units, vn, itn, a1, b1);
            compute(v, it, a0, b0);
            if (it == iters - 1) finish(v);
            v = vn; it = itn;
            if (v >= n_units) break;
            vn = v; itn = it + 1;
            if (itn == iters) { itn = 0; vn += kGvWarps; }
            load(vn < n_units, vn, itn, a0, b0);
            compute(v, it, a1, b1);
            if (it == iters - 1) finish(v);
            v = vn; it = itn;
        }
        __syncthreads();
        // F2: slot order, fp32
        for (int i = tid; i < 2 * nq; i += kGvThreads) {
            float o = 0.0f;
            for (int sidx = 0; sidx < n_src; ++sidx) o = fmaf(s_gw[sidx], s_y[((size_t)sidx * max_q) * 2 + i], o);
            const size_t oi = (size_t)t * p.D + 2 * (size_t)qa + i;
            if (p.out_f32) p.out_f32[oi] = o;
            else p.out[oi] = (bm_bf16)f32_to_bf16_bits(o);
        }
        pos += nq;
    }
}

__global__ void __launch_bounds__(kGvThreads, 1)
gemv2_combine_kernel(Gemv2Args p, int max_src, int max_q) {
    extern __shared__ __align__(16) uint8_t gv_smem[];
    grid_dep_wait();      // h comes from the W1/W3 stage, the routing arrays from bm_route
    grid_dep_launch();
    gemv2_combine_body<false>(p, max_src, max_q, gv_smem);
}

// -------------------------------------------------------------------------------------------------
// The whole layer for one or two tokens in ONE persistent kernel (bm_moe_layer, T <= 2, T*K <= G): single-token decode is
// a chain of four dependent steps -- router logits, selection, W1/W3 stream, W2 stream + combine -- each a few
// microseconds long, and as three launches every arrow costs a kernel boundary.  Here the arrows are two grid-wide
// barriers (cooperative launch: all CTAs are resident):
//   A  canonical router dots (A1), one warp per (token, expert), spread over the grid        -> logits scratch
//   -- barrier --
//   B  every CTA selects for itself (R2-R5, R6-R8 on <= 32 items, in shared memory); CTA 0 also writes the routing arrays
//   C  gemv_body<SWIGLU> with offsets / row_token in shared memory                            -> h
//   -- barrier --
//   D  gemv2_combine_body (h read with ld.global.cg: written in this kernel)                  -> out
// Barrier counters live in the zero-once head of the workspace and are put back to zero by the last CTA to leave.
// -------------------------------------------------------------------------------------------------
struct SmallArgs {
    const bm_bf16 *x, *Wr;
    const float *bias;
    const int32_t *gmap;
    const bm_bf16 *W1, *W3, *W2;
    bm_bf16 *h, *out;
    bm_routing r;
    float *logits;          // [T][E] scratch
    int32_t *status;        // workspace head: [0] status bits, [1] A, [8], [9], [10] barrier counters
    int T, D, E, K, G, S, F;
    int rows_cap, max_src, max_q;
};
constexpr int kSmallBar = 8;        // status[8], status[9]: the two grid barriers; status[10]: CTAs that have left

__device__ __forceinline__ void grid_barrier(int32_t *ctr, int n_cta) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1);
        uint32_t spins = 0;
        uint64_t t0 = 0;
        int v;
        do {
            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
            if (v < n_cta && (++spins & 0x3ffu) == 0) {
                const uint64_t now = ptx::globaltimer_ns();
                if (t0 == 0) t0 = now;
                else if (now - t0 > ptx::kWaitTimeoutNs) __trap();
            }
        } while (v < n_cta);
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kGvThreads, 1)
layer_small_kernel(SmallArgs a) {
    extern __shared__ __align__(16) uint8_t gv_smem[];
    __shared__ int32_t s_eid[2 * BM_MAX_K], s_gid[2 * BM_MAX_K], s_rtok[2 * BM_MAX_K], s_rslot[2 * BM_MAX_K], s_srow[2 * BM_MAX_K];
    __shared__ int32_t s_ns[2], s_off[BM_MAX_G + 1], s_A;
    __shared__ float s_gw[2 * BM_MAX_K];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_cta = (int)gridDim.x;
    const int T = a.T, E = a.E, K = a.K, G = a.G, D = a.D;

    // ---- A: router logits in the canonical order (A1), bit for bit as router_kernel ------------------------------
    for (int i = (int)blockIdx.x + warp * n_cta; i < T * E; i += n_cta * kGvWarps) {
        const int t = i / E, e = i - t * E;
        const bm_bf16 *xrow = a.x + (size_t)t * D, *wrow = a.Wr + (size_t)e * D;
        float p = 0.0f;
#pragma unroll 8
        for (int k = lane * 8; k < D; k += 256) {
            const uint4 xv = __ldg(reinterpret_cast<const uint4 *>(xrow + k));
            const uint4 wv = __ldg(reinterpret_cast<const uint4 *>(wrow + k));
            p = __fmaf_rn(bf16_lo(xv.x), bf16_lo(wv.x), p);
            p = __fmaf_rn(bf16_hi(xv.x), bf16_hi(wv.x), p);
            p = __fmaf_rn(bf16_lo(xv.y), bf16_lo(wv.y), p);
            p = __fmaf_rn(bf16_hi(xv.y), bf16_hi(wv.y), p);
            p = __fmaf_rn(bf16_lo(xv.z), bf16_lo(wv.z), p);
            p = __fmaf_rn(bf16_hi(xv.z), bf16_hi(wv.z), p);
            p = __fmaf_rn(bf16_lo(xv.w), bf16_lo(wv.w), p);
            p = __fmaf_rn(bf16_hi(xv.w), bf16_hi(wv.w), p);
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) p = __fadd_rn(p, __shfl_xor_sync(kFullMask, p, o));
        if (lane == 0) {
            if (a.bias) p = __fadd_rn(p, a.bias[e]);
            __stcg(a.logits + i, p);
        }
    }
    grid_barrier(a.status + kSmallBar, n_cta);

    // ---- B: selection and the (tiny) permutation, by every CTA for itself ----------------------------------------
    float *s_l = reinterpret_cast<float *>(gv_smem);
    for (int i = tid; i < T * E; i += kGvThreads) s_l[i] = __ldcg(a.logits + i);
    __syncthreads();
    if (warp < T) select_and_write(s_l + warp * E, warp, lane, E, K, GroupMap{a.gmap, nullptr, G}, s_eid, s_gid, s_gw, s_ns, a.status);
    __syncthreads();
    const int items = T * K;                      // <= 32
    for (int u = tid; u <= G; u += kGvThreads) {
        int less = 0;
        for (int j = 0; j < items; ++j) { const int kj = s_gid[j]; less += (kj >= 0 && kj < u) ? 1 : 0; }
        s_off[u] = less;
        if (u == G) s_A = less;
    }
    if (tid < items) {
        const int k = s_gid[tid];
        int row = 0;
        for (int j = 0; j < items; ++j) { const int kj = s_gid[j]; row += (kj >= 0 && (kj < k || (kj == k && j < tid))) ? 1 : 0; }
        s_srow[tid] = k >= 0 ? row : -1;
    }
    __syncthreads();
    if (tid < items) { s_rtok[tid] = -1; s_rslot[tid] = -1; }
    __syncthreads();
    if (tid < items && s_srow[tid] >= 0) { s_rtok[s_srow[tid]] = tid / K; s_rslot[s_srow[tid]] = tid % K; }
    __syncthreads();
    if (blockIdx.x == 0) {                         // the routing arrays of the API (fully written, pads included)
        if (tid < items) {
            a.r.expert_ids[tid] = s_eid[tid]; a.r.group_ids[tid] = s_gid[tid]; a.r.gate_w[tid] = s_gw[tid];
            a.r.row_token[tid] = s_rtok[tid]; a.r.row_slot[tid] = s_rslot[tid]; a.r.slot_row[tid] = s_srow[tid];
        }
        if (tid < T) a.r.n_slots[tid] = s_ns[tid];
        for (int u = tid; u <= G; u += kGvThreads) {
            a.r.offsets[u] = s_off[u];
            if (u < G) a.r.counts[u] = s_off[u + 1] - s_off[u];
        }
        if (tid == 0) a.status[1] = s_A;
    }

    // ---- C: W1 / W3 stream ------------------------------------------------------------------------------------------
    {
        GemvArgs p{};
        p.in = a.x; p.Wa = a.W1; p.Wb = a.W3; p.outp = a.h; p.offsets = s_off; p.row_token = s_rtok;
        p.T = T; p.TK = items; p.G = G; p.S = a.S; p.IN = D; p.OUT = a.F; p.NQ = a.F;
        gemv_body<true>(p, a.rows_cap, gv_smem);
    }
    grid_barrier(a.status + kSmallBar + 1, n_cta);

    // ---- D: W2 stream + gate-weighted combine ------------------------------------------------------------------
    {
        Gemv2Args q{};
        q.h = a.h; q.W2 = a.W2; q.out = a.out; q.out_f32 = nullptr;
        q.group_ids = s_gid; q.slot_row = s_srow; q.n_slots = s_ns; q.gate_w = s_gw;
        q.T = T; q.K = K; q.G = G; q.S = a.S; q.D = D; q.F = a.F;
        if (q.F <= 1536) gemv2_combine_body<true, 6>(q, a.max_src, a.max_q, gv_smem);
        else gemv2_combine_body<true>(q, a.max_src, a.max_q, gv_smem);
    }
    // barrier counters back to zero: the first is free once everybody is past the second; the second (and the exit
    // counter) once everybody has left it
    if (tid == 0) {
        if (blockIdx.x == 0) a.status[kSmallBar] = 0;
        if (atomicAdd(a.status + kSmallBar + 2, 1) == n_cta - 1) { a.status[kSmallBar + 1] = 0; a.status[kSmallBar + 2] = 0; }
    }
}

}  // namespace

// One cooperative launch for the whole layer on T <= 2 tokens; *handled = false when the shape does not fit (the caller
// then takes the separate kernels).
cudaError_t launch_layer_small(const bm_bf16 *x, int T, int D, const bm_bf16 *Wr, const float *bias, int E, int K,
                               const int32_t *gmap, int G, const bm_bf16 *W1, const bm_bf16 *W3, const bm_bf16 *W2, int F, int S,
                               bm_bf16 *out, const bm_routing &r, bm_bf16 *h, float *logits, int32_t *status, bool *handled,
                               cudaStream_t stream) {
    *handled = false;
    const int sms = num_sms();
    int rows_cap = 2;                            // a set meets at most T <= 2 rows here
    while (rows_cap > 1 && (size_t)rows_cap * D * 2 > 200 * 1024) rows_cap >>= 1;
    const size_t smem1 = (size_t)rows_cap * D * 2 + (size_t)(G + S) * sizeof(int);
    const int max_src = K + S;
    const long long total = (long long)T * (D / 2);
    const int max_q = (int)((total + sms - 1) / sms);
    const size_t smem2 = (size_t)max_src * F * 2 + (size_t)max_src * max_q * 2 * sizeof(float);
    const size_t smem = std::max(std::max(smem1, smem2), (size_t)T * E * sizeof(float));
    if (T < 1 || T > 2 || max_src > 32 || smem > 200 * 1024 || T * E > sms * kGvWarps) return cudaSuccess;
    if (cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void *>(layer_small_kernel), smem); ea != cudaSuccess) return ea;
    SmallArgs a{};
    a.x = x; a.Wr = Wr; a.bias = bias; a.gmap = gmap; a.W1 = W1; a.W3 = W3; a.W2 = W2; a.h = h; a.out = out; a.r = r;
    a.logits = logits; a.status = status;
    a.T = T; a.D = D; a.E = E; a.K = K; a.G = G; a.S = S; a.F = F;
    a.rows_cap = rows_cap; a.max_src = max_src; a.max_q = max_q;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(sms); cfg.blockDim = dim3(kGvThreads); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    count_launch();
    profile_begin(BM_KERNEL_GEMM1, stream);
    const cudaError_t e = cudaLaunchKernelEx(&cfg, layer_small_kernel, a);
    profile_end(BM_KERNEL_GEMM1, stream);
    if (e == cudaSuccess) *handled = true;
    return e;
}

cudaError_t launch_forward_gemv(const ForwardArgs &a, cudaStream_t stream) {
    GemvArgs p{};
    p.offsets = a.r.offsets; p.row_token = a.r.row_token;
    p.T = a.T; p.TK = a.T * a.K; p.G = a.G; p.S = a.S;
    p.in = a.x; p.Wa = a.W1; p.Wb = a.W3; p.outp = a.h; p.IN = a.D; p.OUT = a.F; p.NQ = a.F;
    cudaError_t e = launch_gemv<true>(p, BM_KERNEL_GEMM1, stream);
    if (e != cudaSuccess) return e;
    // W2 stage: fused with the combine when the per-CTA buffers fit (they do unless K + S or F is huge)
    const int max_src = a.K + a.S;
    const long long total = (long long)a.T * (a.D / 2);
    const int max_q = (int)((total + num_sms() - 1) / num_sms());
    const size_t smem2 = (size_t)max_src * a.F * 2 + (size_t)max_src * max_q * 2 * sizeof(float);
    if (max_src <= 32 && smem2 <= 200 * 1024 && opt(OPT_GEMV_FUSE) != 0) {
        Gemv2Args q{};
        q.h = a.h; q.W2 = a.W2; q.out = a.out_f32 ? nullptr : a.out; q.out_f32 = a.out_f32;
        q.group_ids = a.r.group_ids; q.slot_row = a.r.slot_row; q.n_slots = a.r.n_slots; q.gate_w = a.r.gate_w;
        q.T = a.T; q.K = a.K; q.G = a.G; q.S = a.S; q.D = a.D; q.F = a.F;
        if ((e = ensure_dyn_smem(reinterpret_cast<const void *>(gemv2_combine_kernel), smem2)) != cudaSuccess) return e;
        profile_begin(BM_KERNEL_GEMM2, stream);
        e = launch_kernel(gemv2_combine_kernel, dim3(num_sms()), dim3(kGvThreads), smem2, stream, q, max_src, max_q);
        profile_end(BM_KERNEL_GEMM2, stream);
        return e;
    }
    p.in = a.h; p.Wa = a.W2; p.Wb = a.W2; p.outp = a.y; p.IN = a.F; p.OUT = a.D; p.NQ = a.D / 2;
    e = launch_gemv<false>(p, BM_KERNEL_GEMM2, stream);
    if (e != cudaSuccess) return e;
    return launch_combine(a, stream);
}

}  // namespace bm
