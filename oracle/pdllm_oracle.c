/*
 * pdllm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the decode-stage hot path of Prefilling-dLLM
 * (arxiv/paper_2606_10537), written from /root/reference/PAPER.md ("P:<line>")
 * and SURVEY.md section 8(c) ("R<n>" = a reading listed there and in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header,
 * table or helper with paper_2606_10537_b200/csrc (the CUDA path) and
 * neither includes the other.
 *
 * What it computes, in the paper's order:
 *   step 1  chunk scores        oracle_scores      (Eq. 5; R1-R3)   [parity unpinned by the paper: R1]
 *   step 2  top-K chunks        oracle_topk        (R6)
 *   step 3  gather indices      oracle_gather_idx  (R7)
 *   step 4  explicit concat     inside oracle_attn ("concatenated with the cached KV")
 *   step 5  naive softmax attn  oracle_attn        (bidirectional, no mask; R9)
 *   step 6  Split-S + LSE merge oracle_attn_split  (self-check path only; R10)
 *
 * Conventions (R4, R5, R14): inputs are bf16 bit patterns (uint16) widened
 * exactly to fp64; all arithmetic is fp64; kv(h) = h / G with G = H / H_kv;
 * scale multiplies q.k; log is natural; cache rows per chunk Cp = C + 1 with
 * slot 0 = that chunk's BOS token.
 *
 * Pins: tests/test_oracle_*.py (dense-attention reduction, closed forms,
 * brute force, library SDPA, split independence, subset enumeration).
 * The definition of the chunk score itself (R1) is ours, not the paper's:
 * "parity unpinned" for oracle_scores w.r.t. the paper; its arithmetic is
 * pinned by closed forms and the chain rule against step 5.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef uint16_t bf16_bits;

/* bf16 -> fp64, exact: bf16 is the upper 16 bits of an IEEE-754 binary32. */
static double widen(bf16_bits v) {
    uint32_t u = ((uint32_t)v) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

static double dot_bf16(const bf16_bits *a, const bf16_bits *b, int d) {
    double acc = 0.0;
    for (int c = 0; c < d; ++c) acc += widen(a[c]) * widen(b[c]);
    return acc;
}

/* ------------------------------------------------------------------------
 * Step 1 (R1): scores[b,g,n] = 1/(G*L_q) * sum_{h in group g} sum_{i<L_q}
 *              log sum_{j<=C} exp(scale * <Q[b,h,i,:], Kcache[b,g,n,j,:]>)
 * BOS (slot 0) included, keep mask not applied (R3; Fig. 3 caption P:108).
 * Q is addressed as Q[b*q_batch_stride + h*q_head_stride + i*d + c] (elements)
 * so that the first L_q rows of Q_dec can be used in place (R8).
 * row_lse (optional, may be NULL): [B,H,L_q,N] the per-row per-chunk log-mass.
 * ------------------------------------------------------------------------ */
int oracle_scores(const bf16_bits *Q, int64_t q_batch_stride, int64_t q_head_stride,
                  const bf16_bits *Kcache,
                  int B, int H, int H_kv, int d, int N, int C, int L_q, double scale,
                  double *scores, double *row_lse)
{
    if (H_kv <= 0 || H % H_kv != 0 || L_q <= 0) return -1;
    const int G = H / H_kv, Cp = C + 1;
    #pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < B; ++b)
    for (int gn = 0; gn < H_kv * N; ++gn) {
        const int g = gn / N, n = gn % N;
        const bf16_bits *Kn = Kcache + ((((int64_t)b * H_kv + g) * N + n) * Cp) * (int64_t)d;
        double *z = (double *)malloc(sizeof(double) * (size_t)Cp);
        double total = 0.0;
        for (int hh = 0; hh < G; ++hh) {
            const int h = g * G + hh;
            for (int i = 0; i < L_q; ++i) {
                const bf16_bits *q = Q + (int64_t)b * q_batch_stride + (int64_t)h * q_head_stride + (int64_t)i * d;
                double zmax = -INFINITY;
                for (int j = 0; j < Cp; ++j) {
                    z[j] = scale * dot_bf16(q, Kn + (int64_t)j * d, d);
                    if (z[j] > zmax) zmax = z[j];
                }
                double sum = 0.0;
                for (int j = 0; j < Cp; ++j) sum += exp(z[j] - zmax);
                const double ell = zmax + log(sum);
                if (row_lse) row_lse[(((int64_t)b * H + h) * L_q + i) * N + n] = ell;
                total += ell;
            }
        }
        scores[((int64_t)b * H_kv + g) * N + n] = total / ((double)G * (double)L_q);
        free(z);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Step 2 (R6): per row of `scores` keep the K highest; ties go to the
 * lower index; NaN counts as -inf; the K ids are emitted in ascending index
 * order.  Written as K passes of "take the best remaining", which is the
 * stable (score desc, index asc) order, followed by an index sort.
 * ------------------------------------------------------------------------ */
int oracle_topk(const double *scores, int64_t rows, int N, int K, int32_t *ids)
{
    if (K < 1 || K > N) return -1;
    for (int64_t r = 0; r < rows; ++r) {
        const double *s = scores + r * N;
        char *taken = (char *)calloc((size_t)N, 1);
        for (int k = 0; k < K; ++k) {
            int best = -1;
            double bestv = 0.0;
            for (int n = 0; n < N; ++n) {
                if (taken[n]) continue;
                double v = s[n];
                if (v != v) v = -INFINITY;          /* NaN -> -inf */
                if (best < 0 || v > bestv) { best = n; bestv = v; }   /* strict '>' keeps the lower index on ties */
            }
            taken[best] = 1;
        }
        int w = 0;
        for (int n = 0; n < N; ++n) if (taken[n]) ids[r * K + w++] = n;   /* ascending index order */
        free(taken);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Step 3 (R7): row r = k*Bk + t of the virtual selected prefix is
 * cache row ids[k]*Cp + keep[b,g,ids[k],t]; keep == NULL means slot t itself
 * (then Bk must equal Cp).  keep is int32 [B,H_kv,N,Bk], ascending, keep[..,0]=0.
 * ------------------------------------------------------------------------ */
int oracle_gather_idx(const int32_t *ids, const int32_t *keep,
                      int B, int H_kv, int N, int C, int K, int Bk, int32_t *gather_idx)
{
    const int Cp = C + 1;
    if (!keep && Bk != Cp) return -1;
    for (int b = 0; b < B; ++b)
    for (int g = 0; g < H_kv; ++g) {
        const int64_t bg = (int64_t)b * H_kv + g;
        for (int k = 0; k < K; ++k) {
            const int n = ids[bg * K + k];
            if (n < 0 || n >= N) return -2;
            for (int t = 0; t < Bk; ++t) {
                const int slot = keep ? keep[((bg * N + n) * (int64_t)Bk) + t] : t;
                if (slot < 0 || slot > C) return -3;
                gather_idx[bg * ((int64_t)K * Bk) + (int64_t)k * Bk + t] = n * Cp + slot;
            }
        }
    }
    return 0;
}

/* Steps 3+4 for one (b,g): build Kx, Vx = [gathered prefix rows || decode rows] in fp64. */
static int concat_kv(const bf16_bits *Kcache, const bf16_bits *Vcache,
                     const int32_t *ids, const int32_t *keep,
                     const bf16_bits *K_dec, const bf16_bits *V_dec,
                     int b, int g, int H_kv, int d, int N, int C, int K, int Bk, int L_s,
                     double *Kx, double *Vx)
{
    const int Cp = C + 1;
    const int64_t bg = (int64_t)b * H_kv + g;
    const bf16_bits *Kc = Kcache + bg * (int64_t)N * Cp * d;
    const bf16_bits *Vc = Vcache + bg * (int64_t)N * Cp * d;
    int64_t r = 0;
    for (int k = 0; k < K; ++k) {
        const int n = ids[bg * K + k];
        if (n < 0 || n >= N) return -2;
        for (int t = 0; t < Bk; ++t, ++r) {
            const int slot = keep ? keep[((bg * N + n) * (int64_t)Bk) + t] : t;
            if (slot < 0 || slot > C) return -3;
            const int64_t src = ((int64_t)n * Cp + slot) * d;
            for (int c = 0; c < d; ++c) {
                Kx[r * d + c] = widen(Kc[src + c]);
                Vx[r * d + c] = widen(Vc[src + c]);
            }
        }
    }
    for (int j = 0; j < L_s; ++j, ++r)
        for (int c = 0; c < d; ++c) {
            Kx[r * d + c] = widen(K_dec[(bg * L_s + j) * (int64_t)d + c]);
            Vx[r * d + c] = widen(V_dec[(bg * L_s + j) * (int64_t)d + c]);
        }
    return 0;
}

/* Step 5 on rows [j0, j1) of Kx/Vx for one query row: returns lse, writes the
 * NORMALISED partial output; an empty range gives lse = -inf and zeros (R10). */
static double attend_range(const double *q, const double *Kx, const double *Vx,
                           int64_t j0, int64_t j1, int d, double scale,
                           double *s_buf, double *o, double *p_out)
{
    for (int c = 0; c < d; ++c) o[c] = 0.0;
    if (j1 <= j0) return -INFINITY;
    double m = -INFINITY;
    for (int64_t j = j0; j < j1; ++j) {
        double acc = 0.0;
        for (int c = 0; c < d; ++c) acc += q[c] * Kx[j * d + c];
        s_buf[j - j0] = scale * acc;
        if (s_buf[j - j0] > m) m = s_buf[j - j0];
    }
    double l = 0.0;
    for (int64_t j = j0; j < j1; ++j) { s_buf[j - j0] = exp(s_buf[j - j0] - m); l += s_buf[j - j0]; }
    for (int64_t j = j0; j < j1; ++j) {
        const double p = s_buf[j - j0] / l;
        if (p_out) p_out[j] = p;
        for (int c = 0; c < d; ++c) o[c] += p * Vx[j * d + c];
    }
    return m + log(l);
}

/* ------------------------------------------------------------------------
 * Steps 3-5 (R8, R9) and, when n_splits > 1, step 6 (R10).
 *   Q_dec bf16 [B,H,L,d]; Kcache,Vcache bf16 [B,H_kv,N,Cp,d]; ids int32 [B,H_kv,K];
 *   keep int32 [B,H_kv,N,Bk] or NULL; K_dec,V_dec bf16 [B,H_kv,L_s,d].
 *   O fp64 [B,H,L,d]; LSE fp64 [B,H,L]; P (optional) fp64 [B,H,L,S_kv] softmax rows
 *   (only filled when n_splits <= 1).
 *   head_mask (optional) uint8 [B,H]: heads with 0 are skipped (outputs untouched).
 * n_splits <= 1: one pass over all S_kv = K*Bk + L_s rows (the definition).
 * n_splits  > 1: cut [0,S_kv) at floor(s*S_kv/n_splits), attend per range with its
 *   own (m,l), merge: LSE = log sum_s exp(lse_s), O = sum_s exp(lse_s-LSE) O_s.
 * ------------------------------------------------------------------------ */
int oracle_attn(const bf16_bits *Q_dec, const bf16_bits *Kcache, const bf16_bits *Vcache,
                const int32_t *ids, const int32_t *keep,
                const bf16_bits *K_dec, const bf16_bits *V_dec,
                int B, int H, int H_kv, int d, int N, int C, int K, int Bk, int L, int L_s,
                double scale, int n_splits, const uint8_t *head_mask,
                double *O, double *LSE, double *P)
{
    if (H_kv <= 0 || H % H_kv != 0) return -1;
    if (!keep && Bk != C + 1) return -1;
    const int G = H / H_kv;
    const int64_t S_kv = (int64_t)K * Bk + L_s;
    int err = 0;
    #pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < B; ++b)
    for (int g = 0; g < H_kv; ++g) {
        int any = 0;
        for (int hh = 0; hh < G; ++hh) if (!head_mask || head_mask[b * H + g * G + hh]) any = 1;
        if (!any) continue;
        double *Kx = (double *)malloc(sizeof(double) * (size_t)S_kv * d);
        double *Vx = (double *)malloc(sizeof(double) * (size_t)S_kv * d);
        double *s_buf = (double *)malloc(sizeof(double) * (size_t)S_kv);
        double *q = (double *)malloc(sizeof(double) * (size_t)d);
        double *o_s = (double *)malloc(sizeof(double) * (size_t)d);
        double *lse_s = (double *)malloc(sizeof(double) * (size_t)(n_splits > 1 ? n_splits : 1));
        double *o_all = (double *)malloc(sizeof(double) * (size_t)(n_splits > 1 ? n_splits : 1) * d);
        int rc = concat_kv(Kcache, Vcache, ids, keep, K_dec, V_dec, b, g, H_kv, d, N, C, K, Bk, L_s, Kx, Vx);
        if (rc) {
            #pragma omp atomic write
            err = rc;
        } else
        for (int hh = 0; hh < G; ++hh) {
            const int h = g * G + hh;
            if (head_mask && !head_mask[b * H + h]) continue;
            for (int i = 0; i < L; ++i) {
                const int64_t row = ((int64_t)b * H + h) * L + i;
                for (int c = 0; c < d; ++c) q[c] = widen(Q_dec[row * d + c]);
                if (n_splits <= 1) {
                    LSE[row] = attend_range(q, Kx, Vx, 0, S_kv, d, scale, s_buf, O + row * d,
                                            P ? P + row * S_kv : NULL);
                } else {
                    double big = -INFINITY;
                    for (int s = 0; s < n_splits; ++s) {
                        const int64_t j0 = (int64_t)s * S_kv / n_splits, j1 = (int64_t)(s + 1) * S_kv / n_splits;
                        lse_s[s] = attend_range(q, Kx, Vx, j0, j1, d, scale, s_buf, o_all + (int64_t)s * d, NULL);
                        if (lse_s[s] > big) big = lse_s[s];
                    }
                    double tot = 0.0;
                    for (int s = 0; s < n_splits; ++s) if (lse_s[s] > -INFINITY) tot += exp(lse_s[s] - big);
                    const double lse = big + log(tot);
                    for (int c = 0; c < d; ++c) o_s[c] = 0.0;
                    for (int s = 0; s < n_splits; ++s) {
                        if (!(lse_s[s] > -INFINITY)) continue;          /* empty split contributes nothing */
                        const double w = exp(lse_s[s] - lse);
                        for (int c = 0; c < d; ++c) o_s[c] += w * o_all[(int64_t)s * d + c];
                    }
                    for (int c = 0; c < d; ++c) O[row * d + c] = o_s[c];
                    LSE[row] = lse;
                }
            }
        }
        free(Kx); free(Vx); free(s_buf); free(q); free(o_s); free(lse_s); free(o_all);
    }
    return err;
}

/* ------------------------------------------------------------------------
 * Step 6's merge alone: combine S normalised partials.
 *   O_part fp64 [S,rows,d], lse_part fp64 [S,rows] -> O [rows,d], LSE [rows].
 * Used to check the GPU combine kernel in isolation.
 * ------------------------------------------------------------------------ */
int oracle_lse_combine(const double *O_part, const double *lse_part, int S, int64_t rows, int d,
                       double *O, double *LSE)
{
    for (int64_t r = 0; r < rows; ++r) {
        double big = -INFINITY;
        for (int s = 0; s < S; ++s) if (lse_part[s * rows + r] > big) big = lse_part[s * rows + r];
        for (int c = 0; c < d; ++c) O[r * d + c] = 0.0;
        if (!(big > -INFINITY)) { LSE[r] = -INFINITY; continue; }
        double tot = 0.0;
        for (int s = 0; s < S; ++s) if (lse_part[s * rows + r] > -INFINITY) tot += exp(lse_part[s * rows + r] - big);
        LSE[r] = big + log(tot);
        for (int s = 0; s < S; ++s) {
            if (!(lse_part[s * rows + r] > -INFINITY)) continue;
            const double w = exp(lse_part[s * rows + r] - LSE[r]);
            for (int c = 0; c < d; ++c) O[r * d + c] += w * O_part[((int64_t)s * rows + r) * d + c];
        }
    }
    return 0;
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
