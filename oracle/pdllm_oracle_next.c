/*
 * pdllm_oracle_next.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU oracle for the rows SURVEY.md section 8(f) lists after the hot path
 * (NEXT-1 .. NEXT-3), written from /root/reference/PAPER.md ("P:<line>") and the
 * readings of DESIGN.md ("R<n>").  Same rules as pdllm_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's oracle legs may load it; it shares nothing
 * with paper_2606_10537_b200/csrc and neither includes the other.
 *
 *   NEXT-1  oracle_token_scores   Eq. 5, query->chunk term only (Table 7 "query-to-chunk",
 *                                 P:457-465); R22   [parity unpinned by the paper: the softmax is taken
 *                                 inside the chunk, the cache holds no query / pseudo-label keys]
 *           oracle_topb           "only the top-B KV entries per chunk are retained"; R7, R22
 *   NEXT-2  oracle_prefill_attn   chunk prefill attention, Eq. 2: N independent bidirectional
 *                                 sequences [BOS; c_i; q; m]; plain softmax attention per sequence
 *   NEXT-3  oracle_compact_kv     static cache assembly: the selected rows copied once
 *           oracle_pooled_keys / oracle_pooled_scores   R23 (ours): mean-key chunk scorer
 *                                 [parity unpinned by the paper]
 *
 * Conventions as in pdllm_oracle.c: bf16 bit patterns widened exactly to fp64, kv(h) = h / G,
 * natural log, cache rows per chunk Cp = C + 1 with slot 0 = BOS.
 * Pins: tests/test_oracle_next.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef uint16_t bf16_bits;

static double widen(bf16_bits v) {
    uint32_t u = ((uint32_t)v) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* ------------------------------------------------------------------------
 * NEXT-1 (Eq. 5; R22): eviction score of cache slot j of chunk n,
 *   e[b,g,n,j] = sum_{h in group g} sum_{i<L_q} softmax_j( scale * <Q[b,h,i,:], Kcache[b,g,n,j,:]> ),
 * the softmax running over the chunk's own C+1 slots (BOS included).  Only the
 * query->chunk term of Eq. 5; the chunk->query term needs chunk-token queries (model).
 *   Q addressed as in oracle_scores; e fp64 [B,H_kv,N,C+1].
 * ------------------------------------------------------------------------ */
int oracle_token_scores(const bf16_bits *Q, int64_t q_batch_stride, int64_t q_head_stride,
                        const bf16_bits *Kcache, int B, int H, int H_kv, int d, int N, int C, int L_q,
                        double scale, double *e)
{
    if (H_kv <= 0 || H % H_kv != 0 || L_q <= 0) return -1;
    const int G = H / H_kv, Cp = C + 1;
    #pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < B; ++b)
    for (int gn = 0; gn < H_kv * N; ++gn) {
        const int g = gn / N, n = gn % N;
        const bf16_bits *Kn = Kcache + ((((int64_t)b * H_kv + g) * N + n) * Cp) * (int64_t)d;
        double *out = e + (((int64_t)b * H_kv + g) * N + n) * Cp;
        double *z = (double *)malloc(sizeof(double) * (size_t)Cp);
        for (int j = 0; j < Cp; ++j) out[j] = 0.0;
        for (int hh = 0; hh < G; ++hh) {
            const int h = g * G + hh;
            for (int i = 0; i < L_q; ++i) {
                const bf16_bits *q = Q + (int64_t)b * q_batch_stride + (int64_t)h * q_head_stride + (int64_t)i * d;
                double zmax = -INFINITY;
                for (int j = 0; j < Cp; ++j) {
                    double acc = 0.0;
                    for (int c = 0; c < d; ++c) acc += widen(q[c]) * widen(Kn[(int64_t)j * d + c]);
                    z[j] = scale * acc;
                    if (z[j] > zmax) zmax = z[j];
                }
                double sum = 0.0;
                for (int j = 0; j < Cp; ++j) { z[j] = exp(z[j] - zmax); sum += z[j]; }
                for (int j = 0; j < Cp; ++j) out[j] += z[j] / sum;      /* Attn(q_i, c_j) */
            }
        }
        free(z);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * NEXT-1 (R7, R22): per chunk keep slot 0 (BOS, always) and the Bk-1 slots of
 * 1..C with the highest eviction score; ties go to the lower slot; NaN counts as
 * -inf; the kept slots are emitted in ascending order (slot 0 first).
 *   e fp64 [chunks, C+1] -> keep int32 [chunks, Bk], 1 <= Bk <= C+1.
 * Written as Bk-1 passes of "take the best remaining" followed by an index sort.
 * ------------------------------------------------------------------------ */
int oracle_topb(const double *e, int64_t chunks, int C, int Bk, int32_t *keep)
{
    const int Cp = C + 1;
    if (Bk < 1 || Bk > Cp) return -1;
    for (int64_t r = 0; r < chunks; ++r) {
        const double *s = e + r * Cp;
        char *taken = (char *)calloc((size_t)Cp, 1);
        taken[0] = 1;
        for (int k = 1; k < Bk; ++k) {
            int best = -1;
            double bestv = 0.0;
            for (int j = 1; j < Cp; ++j) {
                if (taken[j]) continue;
                double v = s[j];
                if (v != v) v = -INFINITY;
                if (best < 0 || v > bestv) { best = j; bestv = v; }
            }
            taken[best] = 1;
        }
        int w = 0;
        for (int j = 0; j < Cp; ++j) if (taken[j]) keep[r * Bk + w++] = j;
        free(taken);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * NEXT-2 (Eq. 2; Fig. 5(a)): attention of the chunk prefill.  Each of
 * the S = B*N sequences [BOS; c_i; q; m] (T rows) attends to itself, bidirectionally,
 * no mask, independently of every other sequence ("chunks are independent").
 *   Q bf16 [S,H,T,d]; K,V bf16 [S,H_kv,T,d] -> O fp64 [S,H,T,d], LSE fp64 [S,H,T].
 * ------------------------------------------------------------------------ */
int oracle_prefill_attn(const bf16_bits *Q, const bf16_bits *K, const bf16_bits *V,
                        int S, int H, int H_kv, int T, int d, double scale, double *O, double *LSE)
{
    if (H_kv <= 0 || H % H_kv != 0 || T <= 0) return -1;
    const int G = H / H_kv;
    #pragma omp parallel for collapse(2) schedule(dynamic)
    for (int s = 0; s < S; ++s)
    for (int h = 0; h < H; ++h) {
        const int g = h / G;
        const bf16_bits *Ks = K + ((int64_t)s * H_kv + g) * T * (int64_t)d;
        const bf16_bits *Vs = V + ((int64_t)s * H_kv + g) * T * (int64_t)d;
        double *z = (double *)malloc(sizeof(double) * (size_t)T);
        for (int i = 0; i < T; ++i) {
            const int64_t row = ((int64_t)s * H + h) * T + i;
            const bf16_bits *q = Q + row * d;
            double zmax = -INFINITY;
            for (int j = 0; j < T; ++j) {
                double acc = 0.0;
                for (int c = 0; c < d; ++c) acc += widen(q[c]) * widen(Ks[(int64_t)j * d + c]);
                z[j] = scale * acc;
                if (z[j] > zmax) zmax = z[j];
            }
            double l = 0.0;
            for (int j = 0; j < T; ++j) { z[j] = exp(z[j] - zmax); l += z[j]; }
            for (int c = 0; c < d; ++c) O[row * d + c] = 0.0;
            for (int j = 0; j < T; ++j) {
                const double p = z[j] / l;
                for (int c = 0; c < d; ++c) O[row * d + c] += p * widen(Vs[(int64_t)j * d + c]);
            }
            LSE[row] = zmax + log(l);
        }
        free(z);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * NEXT-3 ("assembled directly from the retained KV entries of the selected chunks",
 * P:116 "static cache that is reused across all T denoising steps"): row r of the compact
 * cache of (b,g) is cache row gather_idx[b,g,r] (= ids[k]*Cp + keep slot, R7) -- a copy of
 * the bf16 bit patterns, nothing else.
 *   Kcache,Vcache bf16 [B,H_kv,N*Cp,d]; gather_idx int32 [B,H_kv,S_pre] -> Kc,Vc bf16 [B,H_kv,S_pre,d].
 * ------------------------------------------------------------------------ */
int oracle_compact_kv(const bf16_bits *Kcache, const bf16_bits *Vcache, const int32_t *gather_idx,
                      int B, int H_kv, int64_t cache_rows, int S_pre, int d, bf16_bits *Kc, bf16_bits *Vc)
{
    for (int64_t bg = 0; bg < (int64_t)B * H_kv; ++bg)
        for (int r = 0; r < S_pre; ++r) {
            const int64_t src = gather_idx[bg * S_pre + r];
            if (src < 0 || src >= cache_rows) return -2;
            for (int c = 0; c < d; ++c) {
                Kc[(bg * S_pre + r) * d + c] = Kcache[(bg * cache_rows + src) * d + c];
                Vc[(bg * S_pre + r) * d + c] = Vcache[(bg * cache_rows + src) * d + c];
            }
        }
    return 0;
}

/* ------------------------------------------------------------------------
 * NEXT-3 (R23, ours): pooled (mean) key of every chunk, kbar[b,g,n,:] = 1/(C+1) * sum_j Kcache[b,g,n,j,:]
 * (BOS included, as in R3), fp64 [B,H_kv,N,d].
 * ------------------------------------------------------------------------ */
int oracle_pooled_keys(const bf16_bits *Kcache, int B, int H_kv, int N, int C, int d, double *kbar)
{
    const int Cp = C + 1;
    for (int64_t c0 = 0; c0 < (int64_t)B * H_kv * N; ++c0)
        for (int c = 0; c < d; ++c) {
            double acc = 0.0;
            for (int j = 0; j < Cp; ++j) acc += widen(Kcache[(c0 * Cp + j) * d + c]);
            kbar[c0 * d + c] = acc / (double)Cp;
        }
    return 0;
}

/* ------------------------------------------------------------------------
 * NEXT-3 (R23, ours): pooled-key chunk score
 *   s_pool[b,g,n] = log(C+1) + 1/(G*L_q) * sum_{h in g} sum_{i<L_q} scale * <Q[b,h,i,:], kbar[b,g,n,:]>,
 * i.e. the R1 score with every chunk row replaced by the chunk's mean key; by Jensen it never
 * exceeds the R1 score and equals it when the rows of a chunk are identical.
 *   kbar fp64 [B,H_kv,N,d] (as the caller holds it, e.g. the GPU's fp32 values widened) -> fp64 [B,H_kv,N].
 * ------------------------------------------------------------------------ */
int oracle_pooled_scores(const bf16_bits *Q, int64_t q_batch_stride, int64_t q_head_stride, const double *kbar,
                         int B, int H, int H_kv, int d, int N, int C, int L_q, double scale, double *scores)
{
    if (H_kv <= 0 || H % H_kv != 0 || L_q <= 0) return -1;
    const int G = H / H_kv;
    for (int b = 0; b < B; ++b)
    for (int g = 0; g < H_kv; ++g)
    for (int n = 0; n < N; ++n) {
        const double *kb = kbar + ((((int64_t)b * H_kv + g) * N) + n) * d;
        double total = 0.0;
        for (int hh = 0; hh < G; ++hh)
            for (int i = 0; i < L_q; ++i) {
                const bf16_bits *q = Q + (int64_t)b * q_batch_stride + (int64_t)(g * G + hh) * q_head_stride + (int64_t)i * d;
                double acc = 0.0;
                for (int c = 0; c < d; ++c) acc += widen(q[c]) * kb[c];
                total += scale * acc;
            }
        scores[((int64_t)b * H_kv + g) * N + n] = log((double)(C + 1)) + total / ((double)G * (double)L_q);
    }
    return 0;
}
