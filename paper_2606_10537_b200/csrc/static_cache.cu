// static_cache.cu -- the static-selection fast path:
//   compact_kv_kernel    : the selected, token-thinned cache rows copied ONCE into a contiguous cache
//                          [B,H_kv,K*Bk,d], so that every later denoising step reads plain TMA tiles;
//   pool_keys_kernel     : mean key of every chunk (R23), computed once after the prefill;
//   pooled_score_kernel  : the mean-key chunk score (R23) -- reads N*d instead of N*(C+1)*d per KV head.
// All three are streaming kernels: coalesced 16-byte accesses, fp32 accumulation, no tensor cores (no contraction
// worth a tile: the pooled score is one d-vector against N d-vectors per KV head).
#include "pdllm_internal.h"

namespace pdllm {

namespace {

// One warp per destination row: row r of (b,g) <- cache row ids[k]*Cp + keep[ids[k], t], r = k*Bk + t (R7); K and V.
template <int D>
__global__ void __launch_bounds__(256) compact_kv_kernel(const uint16_t *__restrict__ Kc, const uint16_t *__restrict__ Vc,
                                                         const int32_t *__restrict__ ids, const int32_t *__restrict__ keep,
                                                         uint16_t *__restrict__ Ko, uint16_t *__restrict__ Vo, int64_t total_rows,
                                                         int N, int Cp, int K, int Bk) {
    constexpr int kLanesPerRow = D / 8;                       // 16-byte chunks per row: 16 (d = 128) or 8 (d = 64)
    constexpr int kRowsPerWarp = 32 / kLanesPerRow;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t r = ((int64_t)blockIdx.x * 8 + warp) * kRowsPerWarp + lane / kLanesPerRow;
    if (r >= total_rows) return;
    const int S_pre = K * Bk;
    const int64_t bg = r / S_pre;
    const int v = (int)(r - bg * S_pre), k = v / Bk, t = v - k * Bk;
    const int n = __ldg(ids + bg * K + k);
    const int slot = keep ? __ldg(keep + (bg * N + n) * (int64_t)Bk + t) : t;
    const int64_t src = ((bg * N + n) * (int64_t)Cp + slot) * D + (lane % kLanesPerRow) * 8;
    const int64_t dst = r * D + (lane % kLanesPerRow) * 8;
    *reinterpret_cast<uint4 *>(Ko + dst) = __ldg(reinterpret_cast<const uint4 *>(Kc + src));
    *reinterpret_cast<uint4 *>(Vo + dst) = __ldg(reinterpret_cast<const uint4 *>(Vc + src));
}

__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// One CTA per chunk: thread (w, l) sums rows w, w + kWarps, ... of its 16-byte column chunk; the warps' partial sums
// meet in shared memory in a fixed order (bit-reproducible).  kbar fp32 [chunks, d].
template <int D>
__global__ void __launch_bounds__(256) pool_keys_kernel(const uint16_t *__restrict__ Kc, float *__restrict__ kbar, int Cp) {
    constexpr int kLanesPerRow = D / 8;
    constexpr int kRowSlots = 256 / kLanesPerRow;             // rows in flight per pass
    __shared__ float part[kRowSlots][D];
    const int c8 = threadIdx.x % kLanesPerRow, rs = threadIdx.x / kLanesPerRow;
    const uint16_t *src = Kc + (int64_t)blockIdx.x * Cp * D + c8 * 8;
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int r = rs; r < Cp; r += kRowSlots) {
        const uint4 u = __ldg(reinterpret_cast<const uint4 *>(src + (int64_t)r * D));
        acc[0] += bf16_lo(u.x); acc[1] += bf16_hi(u.x); acc[2] += bf16_lo(u.y); acc[3] += bf16_hi(u.y);
        acc[4] += bf16_lo(u.z); acc[5] += bf16_hi(u.z); acc[6] += bf16_lo(u.w); acc[7] += bf16_hi(u.w);
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) part[rs][c8 * 8 + e] = acc[e];
    __syncthreads();
    if (threadIdx.x < D) {
        float s = 0.f;
        for (int i = 0; i < kRowSlots; ++i) s += part[i][threadIdx.x];
        kbar[(int64_t)blockIdx.x * D + threadIdx.x] = s / (float)Cp;
    }
}

// One CTA per (b,g): qbar = mean of the G*L_q scoring rows (16-byte loads, the row slots' partial sums meet in shared
// memory in a fixed order), then one warp per chunk: scores[n] = log(C+1) + scale * <qbar, kbar[n]>.
template <int D>
__global__ void __launch_bounds__(512) pooled_score_kernel(const uint16_t *__restrict__ Q, int64_t q_batch_stride,
                                                           int64_t q_head_stride, const float *__restrict__ kbar,
                                                           float *__restrict__ scores, int H_kv, int G, int N, int L_q,
                                                           float scale, float log_cp) {
    constexpr int kLanesPerRow = D / 8;
    constexpr int kSlots = 512 / kLanesPerRow;                // row slots: 32 (d = 128) or 64 (d = 64)
    __shared__ float part[kSlots][D];
    __shared__ float qbar[D];
    const int bg = blockIdx.x, b = bg / H_kv, g = bg % H_kv;
    const int c8 = threadIdx.x % kLanesPerRow, rs = threadIdx.x / kLanesPerRow;
    const int rows = G * L_q;
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int m = rs; m < rows; m += kSlots) {
        const int hh = m / L_q, i = m - hh * L_q;
        const uint4 u = __ldg(reinterpret_cast<const uint4 *>(Q + (int64_t)b * q_batch_stride +
                                                              (int64_t)(g * G + hh) * q_head_stride + (int64_t)i * D + c8 * 8));
        acc[0] += bf16_lo(u.x); acc[1] += bf16_hi(u.x); acc[2] += bf16_lo(u.y); acc[3] += bf16_hi(u.y);
        acc[4] += bf16_lo(u.z); acc[5] += bf16_hi(u.z); acc[6] += bf16_lo(u.w); acc[7] += bf16_hi(u.w);
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) part[rs][c8 * 8 + e] = acc[e];
    __syncthreads();
    if (threadIdx.x < D) {
        float s = 0.f;
        for (int i = 0; i < kSlots; ++i) s += part[i][threadIdx.x];
        qbar[threadIdx.x] = s / (float)rows;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int n = warp; n < N; n += 16) {
        const float *kb = kbar + ((int64_t)bg * N + n) * D;
        float s = 0.f;
        for (int e = lane; e < D; e += 32) s += qbar[e] * kb[e];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) scores[(int64_t)bg * N + n] = log_cp + scale * s;
    }
}

}  // namespace

cudaError_t launch_compact_kv(const Dims &s, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                              const int32_t *keep, void *Kcompact, void *Vcompact, cudaStream_t st) {
    const int64_t total = (int64_t)s.B * s.H_kv * s.S_pre;
    const int rows_per_block = 8 * (32 / (s.d / 8));
    const unsigned blocks = (unsigned)((total + rows_per_block - 1) / rows_per_block);
    auto Kc = static_cast<const uint16_t *>(Kcache), Vc = static_cast<const uint16_t *>(Vcache);
    auto Ko = static_cast<uint16_t *>(Kcompact), Vo = static_cast<uint16_t *>(Vcompact);
    if (s.d == 128) compact_kv_kernel<128><<<blocks, 256, 0, st>>>(Kc, Vc, chunk_ids, keep, Ko, Vo, total, s.N, s.Cp, s.K, s.Bk);
    else compact_kv_kernel<64><<<blocks, 256, 0, st>>>(Kc, Vc, chunk_ids, keep, Ko, Vo, total, s.N, s.Cp, s.K, s.Bk);
    return cudaGetLastError();
}

cudaError_t launch_pool_keys(const Dims &s, const void *Kcache, float *kbar, cudaStream_t st) {
    const unsigned chunks = (unsigned)((int64_t)s.B * s.H_kv * s.N);
    if (s.d == 128) pool_keys_kernel<128><<<chunks, 256, 0, st>>>(static_cast<const uint16_t *>(Kcache), kbar, s.Cp);
    else pool_keys_kernel<64><<<chunks, 256, 0, st>>>(static_cast<const uint16_t *>(Kcache), kbar, s.Cp);
    return cudaGetLastError();
}

cudaError_t launch_pooled_scores(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                                 const float *kbar, float *scores, cudaStream_t st) {
    const unsigned groups = (unsigned)(s.B * s.H_kv);
    const float log_cp = logf((float)s.Cp);
    if (s.d == 128)
        pooled_score_kernel<128><<<groups, 512, 0, st>>>(static_cast<const uint16_t *>(Q), q_batch_stride, q_head_stride, kbar,
                                                         scores, s.H_kv, s.G, s.N, s.L_q, s.scale, log_cp);
    else
        pooled_score_kernel<64><<<groups, 512, 0, st>>>(static_cast<const uint16_t *>(Q), q_batch_stride, q_head_stride, kbar,
                                                        scores, s.H_kv, s.G, s.N, s.L_q, s.scale, log_cp);
    return cudaGetLastError();
}

}  // namespace pdllm
