/*
 * pdllm.h -- C ABI of the B200-native (sm_100a) decode-stage hot path of
 * Prefilling-dLLM (arxiv/paper_2606_10537).
 *
 * Citations: "P:<line>" = /root/reference/PAPER.md line; "R<n>" = a reading of the
 * paper listed in DESIGN.md; "S8(x)" = SURVEY.md section 8.
 *
 * The path (S8(a)): at every denoising step the decode-block rows attend,
 * bidirectionally and unmasked, over
 *     [ selected prefix KV  ||  the decode block's own KV ]
 * where the prefix was prefilled once as N chunks of C tokens, each with a BOS
 * token prepended, only the top-K chunks are read, each thinned to
 * Bk kept slots by a token-keep index list (top-B retention), the selected
 * KV sequence is cut into Split-S shards whose partial softmax results are merged
 * by a log-sum-exp reduction.  Chunk relevance scoring and the top-K
 * selection are part of the same path (R1).
 *
 * General rules for every entry point unless stated otherwise
 *   - extern "C"; returns int: 0 = PDLLM_OK, < 0 = error (see pdllm_status).
 *   - ENQUEUE-ONLY on the given stream: never synchronises, never allocates or
 *     frees device memory, keeps no state between calls (TMA descriptors are
 *     passed to kernels by value; the only thing the library remembers is the
 *     SM count of each device, an immutable hardware fact read on first use;
 *     launches set the kernels' dynamic shared-memory attribute each call).
 *   - "device" pointers are caller-owned device memory (e.g. a torch allocation),
 *     16-byte aligned, dense row-major in the stated shape; inputs are read-only;
 *     outputs are fully overwritten; buffers must stay alive until the stream has
 *     run the enqueued work.
 *   - Validation is host-side only (null pointer, misalignment, unsupported shape,
 *     workspace too small): the call returns an error and enqueues nothing.
 *     Device-side data errors (chunk id outside [0,N), keep slot outside [0,C],
 *     unsorted keep list, keep[..,0] != 0) are undefined behaviour in normal
 *     operation: the kernels address the cache with 32-bit offsets formed from them.
 *   - DEBUG SWITCH: with the environment variable PDLLM_DEBUG_VALIDATE=1 the calls
 *     that take chunk_ids / token_keep_idx (pdllm_gather_idx, pdllm_sparse_attn,
 *     pdllm_step*, pdllm_compact_kv, pdllm_score_tokens consumers) first run a
 *     checking kernel over those lists on `stream`, SYNCHRONISE the stream, and
 *     return PDLLM_ERR_DATA with nothing else enqueued on the first violation
 *     (this mode allocates and frees a 4-byte device flag per call: the one
 *     exception to the rules above; for pdllm_step* the ids are produced
 *     internally, so only the keep list is checked).
 *   - STREAM ORDER: the kernels are launched with programmatic stream
 *     serialisation: a kernel's set-up may run under the tail of the kernel before
 *     it in the stream (yours included), but it touches no global memory before
 *     that kernel has completed and its writes are visible
 *     (griddepcontrol.wait), so the usual in-stream ordering holds for every
 *     buffer you pass.
 *   - bf16 = IEEE bfloat16 bit patterns; O is rounded to bf16 round-to-nearest-even
 *     from the fp32 accumulator (R11).
 *   - GQA: query head h reads KV head h / (H / H_kv) (R4).
 *   - scale multiplies q.k before the softmax; LSE and scores are natural logs (R5).
 */
#ifndef PDLLM_H_
#define PDLLM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* A CUDA stream handle (cudaStream_t / CUstream) passed as an opaque pointer;
 * NULL is the legacy default stream. */
typedef void *pdllm_stream_t;

typedef enum {
    PDLLM_OK = 0,
    PDLLM_ERR_NULL = -1,        /* a required pointer is NULL */
    PDLLM_ERR_ALIGN = -2,       /* a device pointer or stride is not 16-byte aligned */
    PDLLM_ERR_SHAPE = -3,       /* a shape field is out of range (see pdllm_shape) */
    PDLLM_ERR_WORKSPACE = -4,   /* workspace_bytes smaller than pdllm_workspace_bytes() */
    PDLLM_ERR_UNSUPPORTED = -5, /* valid request that this build does not implement */
    PDLLM_ERR_CUDA = -6,        /* a CUDA runtime / driver call or a launch failed */
    PDLLM_ERR_DATA = -7,        /* PDLLM_DEBUG_VALIDATE=1 only: a device-side index list is malformed */
    PDLLM_ERR_SCRATCH_LIMIT = -8 /* pdllm_sparse_attn_noalloc: the request needs more than PDLLM_NOALLOC_SCRATCH_BYTES */
} pdllm_status;

/* Shapes shared by all calls (S8 symbols).
 *   Cp   = C + 1 cache rows per chunk, slot 0 = the chunk's BOS (R14)
 *   S_pre = K * Bk selected prefix rows, S_kv = S_pre + L_s                     */
typedef struct {
    int32_t B;      /* batch, >= 1 */
    int32_t H;      /* query heads, H % H_kv == 0 */
    int32_t H_kv;   /* KV heads */
    int32_t d;      /* head dim, 64 or 128 */
    int32_t N;      /* chunks in the cached prefix, 1..4096 */
    int32_t C;      /* tokens per chunk (cache rows per chunk = C + 1) */
    int32_t K;      /* chunks selected, 1 <= K <= min(N, 64) */
    int32_t Bk;     /* kept rows per chunk incl. BOS, 1..C+1; must be C+1 when token_keep_idx == NULL */
    int32_t L_q;    /* rows of Q used for scoring (the query window), >= 1 */
    int32_t L;      /* rows of Q_dec / O / LSE per head, >= 1 */
    int32_t L_s;    /* rows of K_dec / V_dec per KV head, >= 1 (R8) */
    float   scale;  /* softmax scale; <= 0 selects 1/sqrt(d) (R5) */
} pdllm_shape;

/* ---- host-only, pure helpers (no CUDA call, usable without a GPU) ---------- */

int pdllm_version(void);                       /* 200 = 0.2.0 (round 2: pdllm_step_host takes the side stream) */
const char *pdllm_strerror(int status);        /* static string, never NULL */

/* a6 (S8(a); P:189-191 fixes S = 4, NS: "chosen from N*K*C and the number of
 * SMs"): the split count a cost model of the persistent attention kernel picks
 * for num_sms SMs (<= 0: the current device's count).  Per candidate S in
 * 1..min(KV tiles, 64) the model takes the busiest CTA's KV-tile steps under the
 * kernel's item order (plus a fixed cost per work item) and, for S > 1, the
 * combine step's launch and its 2*S*rows*d*4 bytes of partial traffic (at L2
 * speed while they fit L2, at HBM speed beyond); the constants are fitted to
 * measured split sweeps; the cheapest S wins, a larger S only by a 3 % margin.  A split may be a single
 * 128-row KV tile; never more splits than KV tiles.  >= 1. */
int32_t pdllm_auto_splits(const pdllm_shape *shape, int32_t num_sms);

/* Bytes of scratch pdllm_sparse_attn / pdllm_step need for n_splits splits
 * (n_splits == 0: the auto choice for num_sms; num_sms <= 0: the current device's
 * SM count.  Should the auto choice of the device that later runs the call differ,
 * the call takes the largest split count this many bytes hold): always >= 256 (the
 * persistent attention kernel's work-item counter, cleared by the call itself), plus
 * the fp32 partials when there is more than one split, plus -- when G*L_q > 128 --
 * the per-M-tile chunk-score partials of pdllm_step.  Returns 0 for an invalid shape. */
size_t pdllm_workspace_bytes(const pdllm_shape *shape, int32_t n_splits, int32_t num_sms);

/* Bytes of device scratch pdllm_step_host needs (staging of the per-step tensors
 * + pdllm_workspace_bytes). */
size_t pdllm_step_host_scratch_bytes(const pdllm_shape *shape, int32_t n_splits, int32_t num_sms);

/* ---- a1: chunk-score reduction (Eq. 5; R1, R2, R3) ----------
 * scores[b,g,n] = mean over the G*L_q rows (h in group g, i < L_q) of
 *                 log sum_{j=0..C} exp(scale * <Q[b,h,i,:], Kcache[b,g,n,j,:]>)
 * BOS included, keep mask not applied; higher = more relevant.
 *   Q       device bf16, row (b,h,i) at Q + b*q_batch_stride + h*q_head_stride + i*d
 *           (strides in elements, multiples of 8) -- lets the first L_q rows of
 *           Q_dec [B,H,L,d] be scored in place
 *   Kcache  device bf16 [B,H_kv,N,C+1,d]
 *   scores  device fp32 [B,H_kv,N] (out)
 * Reproducibility: bit-identical from run to run when G*L_q <= 128.  Above that the
 * scoring rows span several 128-row M tiles whose contributions this standalone call
 * adds with float atomics (last bits may vary); pdllm_step and pdllm_score_tokens sum
 * them in a fixed order through their scratch and are bit-reproducible.            */
int pdllm_score_chunks(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride,
                       int64_t q_head_stride, const void *Kcache, float *scores,
                       pdllm_stream_t stream);

/* ---- a2: warp-level top-K (R6) ----------------------------------------
 * Per (b,g): the K highest scores, ties to the lower index, NaN treated as -inf;
 * the K chunk ids are written in ascending index order.
 *   scores    device fp32 [B,H_kv,N];  chunk_ids  device int32 [B,H_kv,K] (out)   */
int pdllm_select_topk(const pdllm_shape *shape, const float *scores, int32_t *chunk_ids,
                      pdllm_stream_t stream);

/* ---- a3: gather-index build (R7) ----------------------------------
 * gather_idx[b,g,k*Bk+t] = chunk_ids[b,g,k]*(C+1) + token_keep_idx[b,g,chunk_ids[b,g,k],t]
 * (token_keep_idx == NULL: slot t).  The attention kernel evaluates the same
 * device function inline; this entry point exports the list.
 *   token_keep_idx  device int32 [B,H_kv,N,Bk] ascending slots in [0,C], [..,0]==0, or NULL
 *   gather_idx      device int32 [B,H_kv,K*Bk] (out)                              */
int pdllm_gather_idx(const pdllm_shape *shape, const int32_t *chunk_ids,
                     const int32_t *token_keep_idx, int32_t *gather_idx, pdllm_stream_t stream);

/* ---- a4 + a5: Split-S partial attention and LSE combine (R8-R11)
 * For every (b,h,i<L): softmax attention of Q_dec[b,h,i] over the S_kv rows
 *   [ Kcache/Vcache rows gather_idx[b,g,:]  ||  K_dec/V_dec[b,g,:] ],  g = h/(H/H_kv),
 * computed as n_splits partial softmax passes over contiguous ranges of those rows
 * merged by log-sum-exp (exactly the unsplit result up to fp32 rounding).
 *   Q_dec   device bf16 [B,H,L,d];   Kcache,Vcache device bf16 [B,H_kv,N,C+1,d]
 *   chunk_ids device int32 [B,H_kv,K];  token_keep_idx device int32 [B,H_kv,N,Bk] or NULL
 *   K_dec,V_dec device bf16 [B,H_kv,L_s,d]
 *   n_splits  >= 1, or 0 = pdllm_auto_splits (capped so that no split is empty)
 *   O       device bf16 [B,H,L,d] (out);  LSE device fp32 [B,H,L] (out)
 *   gather_idx_out  device int32 [B,H_kv,K*Bk] (out) or NULL
 *   workspace  device scratch of >= pdllm_workspace_bytes(shape, n_splits, num_sms) bytes
 *              (required; its contents need no initialisation)                     */
int pdllm_sparse_attn(const pdllm_shape *shape, const void *Q_dec, const void *Kcache,
                      const void *Vcache, const int32_t *chunk_ids, const int32_t *token_keep_idx,
                      const void *K_dec, const void *V_dec, int32_t n_splits,
                      void *O, float *LSE, int32_t *gather_idx_out,
                      void *workspace, size_t workspace_bytes, pdllm_stream_t stream);

/* ---- a5 alone: LSE combine of normalised partials ---------------------
 * LSE = log sum_s exp(lse_s);  O = sum_s exp(lse_s - LSE) * O_s;  a split with
 * lse_s = -inf contributes nothing; all -inf gives O = 0, LSE = -inf.
 *   O_part device fp32 [S,rows,d]; lse_part device fp32 [S,rows];
 *   O device bf16 [rows,d] (out); LSE device fp32 [rows] (out); d in {64,128}    */
int pdllm_lse_combine(const float *O_part, const float *lse_part, int32_t S, int64_t rows,
                      int32_t d, void *O, float *LSE, pdllm_stream_t stream);

/* ---- the per-step call: a1 -> a2 -> (a3) -> a4 -> a5 as one enqueue sequence ---
 * Rows 0..L_q-1 of every head of Q_dec are the scoring rows (R8).
 * scores_out [B,H_kv,N] fp32 and chunk_ids_out [B,H_kv,K] int32 are required
 * device outputs (they carry the data between the kernels).
 * With N <= PDLLM_FOLD_MAX_N chunks and gather_idx_out == NULL, a2 runs inside the
 * a4 kernel (each work item ranks its group's scores; same order, same ties, same
 * ids and scores written as pdllm_select_topk) and the sequence is one launch
 * shorter; otherwise a2 is a kernel of its own.  PDLLM_NO_FOLD=1 in the environment
 * (read once) keeps it apart always.                                              */
#define PDLLM_FOLD_MAX_N 128
int pdllm_step(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
               const int32_t *token_keep_idx, const void *K_dec, const void *V_dec, int32_t n_splits,
               float *scores_out, int32_t *chunk_ids_out, void *O, float *LSE,
               int32_t *gather_idx_out, void *workspace, size_t workspace_bytes,
               pdllm_stream_t stream);

/* ---- pdllm_step with per-stage timestamps (measurement aid, S8(d)) ---------------
 * Same enqueue sequence as pdllm_step; additionally records the given CUDA events
 * (cudaEvent_t handles created by the caller with timing enabled, passed as opaque
 * pointers; a NULL member is skipped) on `stream` at the stage boundaries, so that
 * a harness can attribute the step's device time to a1 / a2 / a3-a5 inside the same
 * timed region.  ev == NULL is exactly pdllm_step; with events a2 is always a
 * kernel of its own (there is a boundary to stamp). */
typedef struct {
    void *begin;         /* before a1 */
    void *after_score;   /* after a1 (chunk-score reduction) */
    void *after_topk;    /* after a2 (top-K) */
    void *after_attn;    /* after a3+a4 (Split-S partial attention), before a5 */
    void *end;           /* after a5 (LSE combine; == after_attn time when one split) */
} pdllm_stage_events;

int pdllm_step_profiled(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
                        const int32_t *token_keep_idx, const void *K_dec, const void *V_dec, int32_t n_splits,
                        float *scores_out, int32_t *chunk_ids_out, void *O, float *LSE,
                        int32_t *gather_idx_out, void *workspace, size_t workspace_bytes,
                        const pdllm_stage_events *ev, pdllm_stream_t stream);

/* ---- the per-step call with HOST per-step tensors ------------------------------
 * The prefix cache and keep lists are state that the prefill left on the device
 * ("static cache that is reused across all T denoising steps"); what
 * changes every step is the decode block.  This call enqueues, on `stream`:
 * the H2D copy of h_Q_dec (host, pinned for true async) into d_scratch, the
 * steps of pdllm_step, and D2H copies of O, LSE and chunk ids into the host
 * outputs.  h_K_dec / h_V_dec are read by the attention only: when the caller
 * passes a side stream (`side` != NULL: a second stream of the same device and
 * two events created with cudaEventDisableTiming, all caller-owned; the library
 * creates and keeps nothing) they are copied on it -- the side stream forks from
 * `stream` at the start of the call and joins it ahead of the attention kernel,
 * so those copies run under the scoring kernel.  side == NULL: every copy goes
 * on `stream` in order.  To the caller all work is ordered on `stream`, which it
 * synchronises before reading the outputs.
 *   d_scratch  device scratch of >= pdllm_step_host_scratch_bytes() bytes; one
 *              call at a time may use it                                          */
typedef struct {
    pdllm_stream_t stream;   /* the side stream */
    void *ev_fork;           /* cudaEvent_t, recorded on `stream`, waited on by the side stream */
    void *ev_join;           /* cudaEvent_t, recorded on the side stream, waited on by `stream` */
} pdllm_side_stream;

int pdllm_step_host(const pdllm_shape *shape, const void *h_Q_dec, const void *h_K_dec,
                    const void *h_V_dec, const void *d_Kcache, const void *d_Vcache,
                    const int32_t *d_token_keep_idx, int32_t n_splits,
                    void *h_O, float *h_LSE, int32_t *h_chunk_ids,
                    void *d_scratch, size_t scratch_bytes,
                    const pdllm_side_stream *side, pdllm_stream_t stream);

/* =========================================================================
 * Rows after the hot path.
 * ========================================================================= */

/* ---- NEXT-3: the static-selection fast path ---------------
 * The paper's selection is static: "the retained KV entries of the selected chunks
 * ... form a static cache that is reused across all T denoising steps";
 * its FlexAttention kernel reloads that cache every step.  Here the
 * selected, token-thinned rows are copied ONCE into a contiguous cache, and every
 * later step runs the same attention kernel over plain 128-row TMA tiles.
 *
 * pdllm_compact_kv: row r = k*Bk + t of (b,g) <- cache row
 * chunk_ids[b,g,k]*(C+1) + token_keep_idx[b,g,chunk_ids[b,g,k],t] (NULL: slot t);
 * a bit copy of K and V rows.
 *   Kcompact, Vcompact  device bf16 [B,H_kv,K*Bk,d] (out)                          */
int pdllm_compact_kv(const pdllm_shape *shape, const void *Kcache, const void *Vcache,
                     const int32_t *chunk_ids, const int32_t *token_keep_idx,
                     void *Kcompact, void *Vcompact, pdllm_stream_t stream);

/* Shapes of attention over CONTIGUOUS K/V (no chunk ids, no keep lists): S_pre
 * prefix rows per KV head followed by L_s decode rows (may be 0).               */
typedef struct {
    int32_t B;      /* batch (static cache) or number of independent sequences (prefill), >= 1 */
    int32_t H;      /* query heads, H % H_kv == 0 */
    int32_t H_kv;   /* KV heads */
    int32_t d;      /* head dim, 64 or 128 */
    int32_t S_pre;  /* contiguous prefix rows per KV head, >= 1 */
    int32_t L;      /* rows of Q / O / LSE per head, >= 1 */
    int32_t L_s;    /* rows of K_dec / V_dec per KV head, >= 0 */
    float   scale;  /* softmax scale; <= 0 selects 1/sqrt(d) */
} pdllm_dense_shape;

/* a6 for the contiguous kernels; the prefix and the decode rows are tiled separately
 * (ceil(S_pre/128) + ceil(L_s/128) KV tiles).  Host-only, pure. */
int32_t pdllm_dense_auto_splits(const pdllm_dense_shape *shape, int32_t num_sms);
size_t pdllm_dense_workspace_bytes(const pdllm_dense_shape *shape, int32_t n_splits, int32_t num_sms);

/* pdllm_static_attn: a4 + a5 over [ Kcompact/Vcompact rows || K_dec/V_dec rows ]:
 * exactly pdllm_sparse_attn's result for the chunk ids and keep lists the compact
 * cache was built from (same keys, same order).
 *   Q_dec device bf16 [B,H,L,d]; Kcompact,Vcompact device bf16 [B,H_kv,S_pre,d];
 *   K_dec,V_dec device bf16 [B,H_kv,L_s,d] (NULL allowed when L_s == 0);
 *   O device bf16 [B,H,L,d] (out); LSE device fp32 [B,H,L] (out);
 *   workspace >= pdllm_dense_workspace_bytes(shape, n_splits, num_sms) bytes       */
int pdllm_static_attn(const pdllm_dense_shape *shape, const void *Q_dec, const void *Kcompact,
                      const void *Vcompact, const void *K_dec, const void *V_dec, int32_t n_splits,
                      void *O, float *LSE, void *workspace, size_t workspace_bytes,
                      pdllm_stream_t stream);

/* Pooled-key chunk scorer (R23, ours; parity unpinned by the paper): a cheap
 * per-step re-selection score that reads N*d instead of N*(C+1)*d per KV head.
 * pdllm_pool_keys (once, after the prefill):
 *   kbar[b,g,n,:] = mean over the C+1 cached keys of chunk n (BOS included), fp32.
 * pdllm_score_chunks_pooled (per step):
 *   scores[b,g,n] = log(C+1) + scale * < mean of the G*L_q scoring rows, kbar[b,g,n,:] >,
 * the a1 score with every row of a chunk replaced by the chunk's mean key (by
 * Jensen's inequality a lower bound of it).  Feed it to pdllm_select_topk.
 *   kbar device fp32 [B,H_kv,N,d]; Q, strides as in pdllm_score_chunks;
 *   scores device fp32 [B,H_kv,N] (out)                                            */
int pdllm_pool_keys(const pdllm_shape *shape, const void *Kcache, float *kbar, pdllm_stream_t stream);
int pdllm_score_chunks_pooled(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride,
                              int64_t q_head_stride, const float *kbar, float *scores,
                              pdllm_stream_t stream);

/* ---- NEXT-1: intra-chunk token eviction scores and top-B retention ---------------
 * (Eq. 5, the query->chunk term -- Table 7's "query-to-chunk" variant,
 * P:457-465; "only the top-B KV entries per chunk are retained"; R7, R22.)
 * The step just before the hot path: it produces token_keep_idx on the device.
 *
 * pdllm_score_tokens:
 *   e[b,g,n,j] = sum over the G*L_q scoring rows (h in group g, i < L_q) of
 *                softmax_j( scale * <Q[b,h,i,:], Kcache[b,g,n,j,:]> ),
 * the softmax running over the chunk's own C+1 slots (the cache holds no query or
 * pseudo-label keys: R22; parity unpinned by the paper).  Every chunk's slots sum
 * to G*L_q.  Two streaming passes over the K cache (row log-masses, then scores).
 *   Q, strides, Kcache as in pdllm_score_chunks;
 *   token_scores device fp32 [B,H_kv,N,C+1] (out);
 *   workspace   device scratch >= pdllm_score_tokens_workspace_bytes(shape)
 * pdllm_select_topb: per chunk slot 0 (BOS, always) and the Bk-1 slots of 1..C with
 * the highest score, ties to the lower slot, NaN as -inf, emitted ascending --
 * exactly the list pdllm_sparse_attn / pdllm_step / pdllm_compact_kv take.
 *   token_scores device fp32 [B,H_kv,N,C+1]; token_keep_idx device int32 [B,H_kv,N,Bk] (out);
 *   C + 1 <= 8192, else PDLLM_ERR_UNSUPPORTED                                       */
size_t pdllm_score_tokens_workspace_bytes(const pdllm_shape *shape);
int pdllm_score_tokens(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride,
                       int64_t q_head_stride, const void *Kcache, float *token_scores,
                       void *workspace, size_t workspace_bytes, pdllm_stream_t stream);
int pdllm_select_topb(const pdllm_shape *shape, const float *token_scores, int32_t *token_keep_idx,
                      pdllm_stream_t stream);

/* ---- NEXT-2: attention of the chunk prefill (Eq. 2; Fig. 5(a)) --
 * Each of the shape->B = B*N sequences [BOS; c_i; q; m] (T = S_pre = L rows, L_s = 0)
 * attends to itself, bidirectionally and unmasked, independently of all
 * other sequences ("chunks are independent").  Same kernel as
 * pdllm_static_attn (GQA groups packed into the MMA M dimension, Split-S over the
 * KV tiles when the sequences alone do not fill the GPU).
 *   Q device bf16 [B,H,T,d]; K,V device bf16 [B,H_kv,T,d];
 *   O device bf16 [B,H,T,d] (out); LSE device fp32 [B,H,T] (out)                   */
int pdllm_prefill_attn(const pdllm_dense_shape *shape, const void *Q, const void *K, const void *V,
                       int32_t n_splits, void *O, float *LSE, void *workspace,
                       size_t workspace_bytes, pdllm_stream_t stream);

/* ---- a3 + a4 + a5 without a caller workspace: the call that allocates nothing -----
 * pdllm_sparse_attn (same arguments, same kernels, same results)
 * for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid allocation.  The scratch the path needs (the
 * persistent kernel's work-item counter; the fp32 Split-S partials when more than
 * one split runs) lives in ONE file-scope device array of
 * PDLLM_NOALLOC_SCRATCH_BYTES inside the library: every GPU that loads the library
 * holds those bytes until the process exits; the call itself calls no cudaMalloc,
 * cudaFree or allocating library routine.  Inputs and outputs are still the
 * caller's.
 *   limit     an explicit n_splits whose pdllm_workspace_bytes(shape, n_splits, 0)
 *             exceeds PDLLM_NOALLOC_SCRATCH_BYTES returns PDLLM_ERR_SCRATCH_LIMIT with
 *             nothing enqueued; n_splits == 0 takes the auto choice, lowered to the
 *             largest split count the array holds (one split always fits).  The
 *             limit covers every named workload (C3 at 3 splits: 16.6 MB).
 *   sharing   every call on a device uses the same array, which keeps the previous
 *             call's contents; what must start at zero (the work-item counter) is
 *             cleared on `stream` by the call, the partials are written in full
 *             before they are read.  Calls that OVERLAP on one GPU (different
 *             streams, or several host threads) race on the array: serialise them,
 *             or use pdllm_sparse_attn with a workspace per stream.
 *   debug     PDLLM_DEBUG_VALIDATE=1 makes pdllm_sparse_attn allocate a 4-byte flag
 *             and synchronise; under that switch this call returns
 *             PDLLM_ERR_UNSUPPORTED (debug with pdllm_sparse_attn instead).
 *   set-up    the array's device address is looked up once per device
 *             (cudaGetSymbolAddress with the caller's device current) on the first
 *             call there; make that first call outside a stream capture.          */
#define PDLLM_NOALLOC_SCRATCH_BYTES (32u << 20)
int pdllm_sparse_attn_noalloc(const pdllm_shape *shape, const void *Q_dec, const void *Kcache,
                              const void *Vcache, const int32_t *chunk_ids,
                              const int32_t *token_keep_idx, const void *K_dec, const void *V_dec,
                              int32_t n_splits, void *O, float *LSE, int32_t *gather_idx_out,
                              pdllm_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* PDLLM_H_ */
