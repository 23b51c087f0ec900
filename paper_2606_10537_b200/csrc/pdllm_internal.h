// pdllm_internal.h -- declarations shared by the translation units of libpdllm.so (not installed).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <cstring>

#include "../../include/pdllm.h"

namespace pdllm {

// pdllm_shape with the derived sizes of SURVEY 8 resolved once on the host.
struct Dims {
    int B, H, H_kv, G, d;
    int N, C, Cp, K, Bk;
    int L_q, L, L_s;
    int S_pre, S_kv;      // K*Bk, K*Bk + L_s
    int rows_g;           // G*L: rows of Q_dec that share one KV head (contiguous in [B,H,L,d])
    float scale;
    int contig;           // 1: the prefix is a contiguous [B*H_kv, S_pre, d] cache (compact static cache / chunk prefill)
};

constexpr int kTileM = 128;   // query rows per CTA tile (UMMA M)
constexpr int kTileN = 128;   // virtual KV rows per tile

// ---- a2
// partials / scores_out (optional, together): sum the chunk-score kernel's per-M-tile partials first (launch_score)
cudaError_t launch_topk(const Dims &s, const float *scores, int32_t *chunk_ids, cudaStream_t st,
                        const float *partials = nullptr, float *scores_out = nullptr);
// ---- a3
cudaError_t launch_gather_idx(const Dims &s, const int32_t *chunk_ids, const int32_t *keep, int32_t *gather_idx,
                              cudaStream_t st);
// ---- PDLLM_DEBUG_VALIDATE: *flag |= bits for malformed chunk_ids [B,H_kv,K] / keep [B,H_kv,N,Bk] (either may be NULL)
cudaError_t launch_validate(const Dims &s, const int32_t *chunk_ids, const int32_t *keep, int32_t *flag, cudaStream_t st);
// ---- a5
cudaError_t launch_combine(const float *O_part, const float *lse_part, int S, int64_t rows, int d, void *O, float *LSE,
                           cudaStream_t st);
// ---- a1: scores[b,g,n]
// row_lse (optional): [B*H_kv, N, G*L_q] fp32, every scoring row's log-mass per chunk
cudaError_t launch_score(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride, const void *Kcache,
                         float *scores, float *row_lse, float *partials, cudaStream_t st, int32_t *zero_counter = nullptr);
// ---- NEXT-1 (token_score.cu): e [B,H_kv,N,Cp] from row_lse; e_part: [m_tiles, B,H_kv,N,Cp] scratch when G*L_q > 128
cudaError_t launch_token_scores(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                                const void *Kcache, const float *row_lse, float *e, float *e_part, cudaStream_t st);
cudaError_t launch_topb(const Dims &s, const float *token_scores, int32_t *keep, cudaStream_t st);
int topb_max_cp();
// ---- a3+a4 into O / LSE (n_splits == 1) or into the partials (n_splits > 1: launch_combine follows);
// work_counter: one zeroed int32 (the persistent kernel's work-item counter)
// fold (optional): a2 inside the attention kernel -- the chunk ids are chosen from `scores` (or the per-M-tile
// `partials`, summed in M-tile order and written to scores_out) and written to ids_out; chunk_ids is then unused
struct AttnFold {
    const float *scores, *partials;
    int32_t *ids_out;
    float *scores_out;
};
bool attn_can_fold_topk(const Dims &d);
cudaError_t launch_attn(const Dims &s, const void *Q_dec, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                        const int32_t *keep, const void *K_dec, const void *V_dec, int n_splits, void *O, float *LSE,
                        float *O_part, float *lse_part, int32_t *work_counter, cudaStream_t st, const AttnFold *fold = nullptr);

int device_num_sms();
// KV tiles of 128 rows one query tile walks (gather mode: ceil(S_kv / 128); contiguous mode: prefix and decode rows
// are tiled separately)
int kv_tiles(const Dims &d);

// TMA descriptors (score.cu): bf16 [rows, d] row-major, box = [box_rows, 64 columns], 128-byte swizzle, OOB rows read as
// zero; the 3-D form adds an outermost index over `groups` matrices of `rows` rows each.
bool make_rows_tmap(CUtensorMap *tm, const void *base, uint64_t rows, int d, int box_rows);
bool make_rows_tmap3d(CUtensorMap *tm, const void *base, uint64_t groups, uint64_t rows, int d, int box_rows);

// ---- NEXT-3 (static_cache.cu)
cudaError_t launch_compact_kv(const Dims &s, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                              const int32_t *keep, void *Kcompact, void *Vcompact, cudaStream_t st);
cudaError_t launch_pool_keys(const Dims &s, const void *Kcache, float *kbar, cudaStream_t st);
cudaError_t launch_pooled_scores(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                                 const float *kbar, float *scores, cudaStream_t st);

}  // namespace pdllm
