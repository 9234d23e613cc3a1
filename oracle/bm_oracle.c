/*
 * bm_oracle.c -- the CPU ORACLE for the grouped MoE-layer forward pass (BrownoutMoE full-brownout path; also
 *               partial brownout, SURVEY 8(f) NEXT-1, and the united-weight average, NEXT-3).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code with the CUDA
 * path under paper_2607_04164_b200/ (no headers, helpers, tables or constants) and neither imports
 * the other.  It is deliberately plain and slow: one loop per sentence of the algorithm, no blocking,
 * no BLAS.  OpenMP is used over the outermost independent loop only.
 *
 * What it computes (citations: PAPER.md line numbers = P:NN; readings = A1..A14):
 *   R1  router logits    l[t,e] = x_t . Wr_e (+ bias_e)                       P:42 "gating function"
 *       in fp32 with the CANONICAL summation order of reading A1 (it decides integers, so both
 *       sides must take the decision in the same precision and order).
 *   R2  top-K            K largest logits, ties -> lower expert index, ranked  P:42 "top-K routing"; A4
 *   R3  gate weights     softmax over the K selected logits, fp32              P:42 "gating score"; A2
 *   R4  group remap      u_i = gmap[e_i]                                       P:118-122 (Eq. 2)
 *   R5  dedup + merge    equal groups of one token collapse, weights summed    A5 (linearity of P:42 under P:46)
 *   R6  histogram, exclusive scan
 *   R7  stable permutation: rows ordered by (group, token ascending)           A7
 *   F1  per row: a = W1[u] x_t, b = W3[u] x_t, h = SiLU(a)*b, y = W2[u] h       P:42 FFN_i; A3 (SwiGLU)
 *   F2  out[t] = sum_s gw[t,s] * y_{slot_row[t,s]}  +  sum_j FFN_{G+j}(x_t)     P:42; A11 (shared experts)
 *       F1/F2 in fp64 (inputs are bf16, so every product is exact in fp64); the paper fixes no precision.
 *
 * bf16 crosses this ABI as uint16_t storage.  All pointers are HOST pointers.
 * Pins (tests/test_oracle_*.py): definition-form evaluator, replicated-weights equivalence, gate-sum
 * invariants, brute-force top-K, fp64 logits vs canonical, permutation inverses, G=1 vs library matmul,
 * closed forms, equivariances.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline float bf16_to_f32(uint16_t h) {
    uint32_t u = ((uint32_t)h) << 16;   /* bf16 is the top half of an IEEE binary32: exact */
    float f;
    memcpy(&f, &u, sizeof f);
    return f;
}

/* Reading A1: the canonical fp32 dot product.
 * 32 partial sums; element j belongs to partial (j/8) mod 32; inside a partial, ascending j with a
 * correctly rounded fused multiply-add from p = 0; then the butterfly p_l <- p_l + p_(l xor o) for
 * o = 16, 8, 4, 2, 1 (all l at once); the result is p_0. */
float oracle_canon_dot(const uint16_t *x, const uint16_t *w, int D) {
    float p[32], q[32];
    for (int l = 0; l < 32; ++l) p[l] = 0.0f;
    for (int j = 0; j < D; ++j) {
        int l = (j / 8) % 32;
        p[l] = fmaf(bf16_to_f32(x[j]), bf16_to_f32(w[j]), p[l]);
    }
    for (int o = 16; o >= 1; o >>= 1) {
        for (int l = 0; l < 32; ++l) q[l] = p[l] + p[l ^ o];
        for (int l = 0; l < 32; ++l) p[l] = q[l];
    }
    return p[0];
}

/* R1..R7.  Output arrays are caller-allocated at their maximum size:
 *   expert_ids, group_ids, slot_row [T*K] i32; gate_w [T*K] f32; n_slots [T]; counts [G]; offsets [G+1];
 *   row_token, row_slot [T*K] (first A = offsets[G] valid, rest -1); logits [T*E] f32 or NULL.
 * Returns 0, or -1 on a bad shape / group_map entry outside [0,G). */
/* Partial brownout ("partial-brownout delegates only cold expert tokens to united experts"; P:172
 * "the original gate still determines the ac[tivated experts]"; "the grouping map determines which
 * united expert handles tokens originally routed to each cold expert"; A9: the caller says which
 * experts are cold).  Weight sets are numbered  [0, G) = united experts,  G + e = original expert e.
 * R4 becomes   u_i = cold[e_i] ? gmap[e_i] : G + e_i   and everything after it runs over NS = G + E sets
 * (counts [NS], offsets [NS+1]).  cold == NULL is full brownout over NS = G sets (oracle_route). */
static int route_impl(const uint16_t *x, int T, int D, const uint16_t *Wr, const float *bias, int E, int K,
                 const int32_t *gmap, int G, const int32_t *cold,
                 int32_t *expert_ids, int32_t *group_ids, float *gate_w, int32_t *n_slots,
                 int32_t *counts, int32_t *offsets, int32_t *row_token, int32_t *row_slot,
                 int32_t *slot_row, float *logits_out) {
    if (T < 0 || D < 8 || D % 8 != 0 || E < 1 || K < 1 || K > E || G < 1) return -1;
    for (int e = 0; e < E; ++e)
        if (gmap[e] < 0 || gmap[e] >= G) return -1;
    const int NS = cold ? G + E : G;      /* number of weight sets the routing arrays range over */

#pragma omp parallel for schedule(static)
    for (int t = 0; t < T; ++t) {
        float *l = (float *)malloc(sizeof(float) * (size_t)E);
        char *taken = (char *)calloc((size_t)E, 1);
        /* R1 */
        for (int e = 0; e < E; ++e) {
            float v = oracle_canon_dot(x + (size_t)t * D, Wr + (size_t)e * D, D);
            if (bias) v = v + bias[e];
            l[e] = v;
            if (logits_out) logits_out[(size_t)t * E + e] = v;
        }
        /* R2: rank i takes the largest remaining logit; scanning e upwards with a strict '>' keeps
         * the lower index on exact ties (+0 == -0 is a tie). */
        int32_t *eid = expert_ids + (size_t)t * K;
        for (int i = 0; i < K; ++i) {
            int best = -1;
            for (int e = 0; e < E; ++e) {
                if (taken[e]) continue;
                if (best < 0 || l[e] > l[best]) best = e;
            }
            taken[best] = 1;
            eid[i] = best;
        }
        /* R3: softmax over the K selected logits, sum taken in rank order */
        float w[64];
        float *wk = (K <= 64) ? w : (float *)malloc(sizeof(float) * (size_t)K);
        float m = l[eid[0]];
        float sum = 0.0f;
        for (int i = 0; i < K; ++i) {
            wk[i] = expf(l[eid[i]] - m);
            sum = sum + wk[i];
        }
        for (int i = 0; i < K; ++i) wk[i] = wk[i] / sum;
        /* R4 + R5: remap, then dedup in rank order (first occurrence keeps the slot; A6) */
        int32_t *gid = group_ids + (size_t)t * K;
        float *gw = gate_w + (size_t)t * K;
        int n = 0;
        for (int i = 0; i < K; ++i) {
            int32_t u = (!cold || cold[eid[i]]) ? gmap[eid[i]] : G + eid[i];
            int s;
            for (s = 0; s < n; ++s)
                if (gid[s] == u) break;
            if (s < n) {
                gw[s] = gw[s] + wk[i];
            } else {
                gid[n] = u;
                gw[n] = wk[i];
                n++;
            }
        }
        for (int s = n; s < K; ++s) {
            gid[s] = -1;
            gw[s] = 0.0f;
        }
        n_slots[t] = n;
        if (wk != w) free(wk);
        free(taken);
        free(l);
    }

    /* R6: histogram and exclusive scan */
    for (int u = 0; u < NS; ++u) counts[u] = 0;
    for (int t = 0; t < T; ++t)
        for (int s = 0; s < K; ++s) {
            int32_t u = group_ids[(size_t)t * K + s];
            if (u >= 0) counts[u]++;
        }
    offsets[0] = 0;
    for (int u = 0; u < NS; ++u) offsets[u + 1] = offsets[u] + counts[u];

    /* R7: rows ordered by (group, token ascending) */
    for (size_t i = 0; i < (size_t)T * K; ++i) {
        row_token[i] = -1;
        row_slot[i] = -1;
        slot_row[i] = -1;
    }
    for (int u = 0; u < NS; ++u) {
        int32_t r = offsets[u];
        for (int t = 0; t < T; ++t)
            for (int s = 0; s < K; ++s)
                if (group_ids[(size_t)t * K + s] == u) {
                    row_token[r] = t;
                    row_slot[r] = s;
                    slot_row[(size_t)t * K + s] = r;
                    r++;
                }
    }
    return 0;
}

int oracle_route(const uint16_t *x, int T, int D, const uint16_t *Wr, const float *bias, int E, int K,
                 const int32_t *gmap, int G,
                 int32_t *expert_ids, int32_t *group_ids, float *gate_w, int32_t *n_slots,
                 int32_t *counts, int32_t *offsets, int32_t *row_token, int32_t *row_slot,
                 int32_t *slot_row, float *logits_out) {
    return route_impl(x, T, D, Wr, bias, E, K, gmap, G, NULL, expert_ids, group_ids, gate_w, n_slots, counts,
                      offsets, row_token, row_slot, slot_row, logits_out);
}

/* cold [E]: non-zero = cold expert (served by its group's united expert).  counts [G+E], offsets [G+E+1]. */
int oracle_route_partial(const uint16_t *x, int T, int D, const uint16_t *Wr, const float *bias, int E, int K,
                         const int32_t *gmap, int G, const int32_t *cold,
                         int32_t *expert_ids, int32_t *group_ids, float *gate_w, int32_t *n_slots,
                         int32_t *counts, int32_t *offsets, int32_t *row_token, int32_t *row_slot,
                         int32_t *slot_row, float *logits_out) {
    if (!cold) return -1;
    return route_impl(x, T, D, Wr, bias, E, K, gmap, G, cold, expert_ids, group_ids, gate_w, n_slots, counts,
                      offsets, row_token, row_slot, slot_row, logits_out);
}

/* United-weight initialisation ("The united expert is initialized as the parameter average of member
 * experts"; the same average is the convex target of Eq. 5 with uniform weights):
 *   Wu[u, i] = (1 / |G_u|) * sum_{e : gmap[e] == u} W[e, i]      in fp64, one plain sum in ascending e.
 * W: [E, n] bf16 (uint16 storage), out: [G, n] fp64; an empty group gives zeros.  Returns 0 or -1. */
int oracle_unite_weights(const uint16_t *W, int E, long long n, const int32_t *gmap, int G, double *out) {
    if (E < 1 || G < 1 || n < 0) return -1;
    for (int e = 0; e < E; ++e)
        if (gmap[e] < 0 || gmap[e] >= G) return -1;
#pragma omp parallel for schedule(static)
    for (int u = 0; u < G; ++u) {
        int members = 0;
        for (int e = 0; e < E; ++e) members += (gmap[e] == u);
        for (long long i = 0; i < n; ++i) {
            double acc = 0.0;
            for (int e = 0; e < E; ++e)
                if (gmap[e] == u) acc += (double)bf16_to_f32(W[(size_t)e * n + i]);
            out[(size_t)u * n + i] = members ? acc / (double)members : 0.0;
        }
    }
    return 0;
}

/* One expert FFN on one token, fp64:  y = W2 . ( SiLU(W1 x) * (W3 x) )      (A3: SwiGLU, no biases)
 * W1, W3: [F, D] row-major; W2: [D, F] row-major.  a_buf: scratch [F]. */
static void ffn_f64(const uint16_t *xt, const uint16_t *W1, const uint16_t *W3, const uint16_t *W2,
                    int D, int F, double *h, double *y) {
    for (int f = 0; f < F; ++f) {
        const uint16_t *w1 = W1 + (size_t)f * D;
        const uint16_t *w3 = W3 + (size_t)f * D;
        double a = 0.0, b = 0.0;
        /* `omp simd reduction` only lets the compiler keep several fp64 partial sums of this one
         * dot product (a 1e-16-relative reassociation); it is still one plain sum per output. */
#pragma omp simd reduction(+ : a)
        for (int j = 0; j < D; ++j) a += (double)bf16_to_f32(w1[j]) * (double)bf16_to_f32(xt[j]);
#pragma omp simd reduction(+ : b)
        for (int j = 0; j < D; ++j) b += (double)bf16_to_f32(w3[j]) * (double)bf16_to_f32(xt[j]);
        h[f] = a / (1.0 + exp(-a)) * b;
    }
    for (int d = 0; d < D; ++d) {
        const uint16_t *w2 = W2 + (size_t)d * F;
        double acc = 0.0;
#pragma omp simd reduction(+ : acc)
        for (int f = 0; f < F; ++f) acc += (double)bf16_to_f32(w2[f]) * h[f];
        y[d] = acc;
    }
}

/* F1 + F2.  Weights hold the G united experts first, then the S shared experts (A11).
 * sel_tokens: ascending list of n_sel token indices to evaluate, or NULL for all T tokens (n_sel = T).
 * out: [n_sel, D] fp64, row i belongs to token sel_tokens[i].
 * Rows are walked in permuted (group-major) order as R7 produced them; a row whose token is not
 * selected is skipped.  Returns 0 or -1. */
int oracle_moe_forward(const uint16_t *x, int T, int D, int K, int G,
                       const int32_t *group_ids, const float *gate_w, const int32_t *n_slots,
                       const int32_t *offsets, const int32_t *row_token, const int32_t *slot_row,
                       const uint16_t *W1, const uint16_t *W3, const uint16_t *W2, int F, int S,
                       const int32_t *sel_tokens, int n_sel, double *out) {
    if (T < 0 || D < 1 || F < 1 || K < 1 || G < 1 || S < 0) return -1;
    if (!sel_tokens) n_sel = T;
    int32_t *sel_index = (int32_t *)malloc(sizeof(int32_t) * (size_t)(T > 0 ? T : 1));
    for (int t = 0; t < T; ++t) sel_index[t] = sel_tokens ? -1 : t;
    if (sel_tokens)
        for (int i = 0; i < n_sel; ++i) {
            if (sel_tokens[i] < 0 || sel_tokens[i] >= T) { free(sel_index); return -1; }
            sel_index[sel_tokens[i]] = i;
        }
    const int A = offsets[G];
    const size_t wsz = (size_t)F * D;

    /* F1: y_r for every (selected) row r, group u = the group whose offset range holds r */
    double *Y = (double *)malloc(sizeof(double) * (size_t)(A > 0 ? A : 1) * D);
    int32_t *row_group = (int32_t *)malloc(sizeof(int32_t) * (size_t)(A > 0 ? A : 1));
    for (int u = 0; u < G; ++u)
        for (int r = offsets[u]; r < offsets[u + 1]; ++r) row_group[r] = u;
#pragma omp parallel
    {
        double *h = (double *)malloc(sizeof(double) * (size_t)F);
#pragma omp for schedule(dynamic, 1)
        for (int r = 0; r < A; ++r) {
            int t = row_token[r];
            if (sel_index[t] < 0) continue;
            int u = row_group[r];
            ffn_f64(x + (size_t)t * D, W1 + u * wsz, W3 + u * wsz, W2 + u * wsz, D, F, h,
                    Y + (size_t)r * D);
        }
        free(h);
    }

    /* F2: combine in slot order, then the shared experts with weight 1 */
#pragma omp parallel
    {
        double *h = (double *)malloc(sizeof(double) * (size_t)F);
        double *y = (double *)malloc(sizeof(double) * (size_t)D);
#pragma omp for schedule(dynamic, 1)
        for (int i = 0; i < n_sel; ++i) {
            int t = sel_tokens ? sel_tokens[i] : i;
            double *o = out + (size_t)i * D;
            for (int d = 0; d < D; ++d) o[d] = 0.0;
            for (int s = 0; s < n_slots[t]; ++s) {
                int r = slot_row[(size_t)t * K + s];
                double gw = (double)gate_w[(size_t)t * K + s];
                for (int d = 0; d < D; ++d) o[d] += gw * Y[(size_t)r * D + d];
            }
            for (int j = 0; j < S; ++j) {
                size_t u = (size_t)G + j;
                ffn_f64(x + (size_t)t * D, W1 + u * wsz, W3 + u * wsz, W2 + u * wsz, D, F, h, y);
                for (int d = 0; d < D; ++d) o[d] += y[d];
            }
        }
        free(y);
        free(h);
    }
    (void)group_ids;
    free(row_group);
    free(Y);
    free(sel_index);
    return 0;
}

/* Calibration forward: the output of EVERY original expert on every calibration token,
 * f_e(x_t) = FFN_e(x_t), the quantity P:147-149 (Eq. 5) averages and P:170 takes cosine similarities of.
 * W1, W3: [E, F, D]; W2: [E, D, F]; out: [E, T, D] fp64. */
int oracle_expert_outputs(const uint16_t *x, int T, int D, const uint16_t *W1, const uint16_t *W3,
                          const uint16_t *W2, int E, int F, double *out) {
    if (T < 0 || D < 1 || F < 1 || E < 1) return -1;
    const size_t wsz = (size_t)F * D;
#pragma omp parallel
    {
        double *h = (double *)malloc(sizeof(double) * (size_t)F);
#pragma omp for schedule(dynamic, 1) collapse(2)
        for (int e = 0; e < E; ++e)
            for (int t = 0; t < T; ++t)
                ffn_f64(x + (size_t)t * D, W1 + e * wsz, W3 + e * wsz, W2 + e * wsz, D, F, h,
                        out + ((size_t)e * T + t) * D);
        free(h);
    }
    return 0;
}
