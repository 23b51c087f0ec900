// select.cu -- a2 warp-level top-K (R6) and a3 gather-index build (R7).
#include "pdllm_internal.h"

namespace pdllm {

namespace {

constexpr int kTopkWarps = 4;          // warps (= score rows) per block
constexpr int kTopkMaxN = 4096;        // pdllm_shape bound on N

// (value, index) order of R6: higher value first, ties to the lower index.
__device__ __forceinline__ bool better(float v, int i, float bv, int bi) { return v > bv || (v == bv && i < bi); }

// One warp per (b,g) row.  The row is staged in shared memory with 128-bit loads; K rounds of
// "best remaining" (lane-local scan + shuffle arg-max) mark a bitmask; the mask is then emitted
// in ascending index order (R6).  NaN is read as -inf.
// `partials` (optional): [m_tiles, rows*N] per-M-tile score contributions of the chunk-score kernel; the row is then
// their sum in M-tile order (bit-reproducible, unlike float atomics) and is also written to scores_out.
__global__ void __launch_bounds__(kTopkWarps * 32) topk_kernel(const float *__restrict__ scores, int32_t *__restrict__ ids,
                                                               int rows, int N, int K, const float *__restrict__ partials,
                                                               int m_tiles, float *__restrict__ scores_out) {
    extern __shared__ float smem_f[];
    // this kernel may have been launched under the kernel that writes the scores (programmatic dependent launch):
    // wait for that grid's completion and flush before the scores are read
    // ... and lets its own dependent (the attention kernel in pdllm_step) be scheduled as SMs fall free: that kernel
    // does its set-up, then waits for this grid in turn
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = blockIdx.x * kTopkWarps + warp;
    if (row >= rows) return;
    const int Npad = (N + 3) & ~3;
    const int words = (N + 31) >> 5;
    float *v = smem_f + (size_t)warp * (Npad + words);
    uint32_t *taken = reinterpret_cast<uint32_t *>(v + Npad);
    const float *src = scores + (size_t)row * N;

    if (partials) {
        for (int i = lane; i < N; i += 32) {
            float x = 0.f;
            for (int mt = 0; mt < m_tiles; ++mt) x += partials[((size_t)mt * rows + row) * N + i];
            scores_out[(size_t)row * N + i] = x;
            v[i] = x == x ? x : -INFINITY;
        }
    } else if ((N & 3) == 0 && ((reinterpret_cast<uintptr_t>(src) & 15) == 0)) {
        for (int i = lane * 4; i < N; i += 128) {
            float4 x = *reinterpret_cast<const float4 *>(src + i);
            v[i] = x.x == x.x ? x.x : -INFINITY;
            v[i + 1] = x.y == x.y ? x.y : -INFINITY;
            v[i + 2] = x.z == x.z ? x.z : -INFINITY;
            v[i + 3] = x.w == x.w ? x.w : -INFINITY;
        }
    } else {
        for (int i = lane; i < N; i += 32) { float x = src[i]; v[i] = x == x ? x : -INFINITY; }
    }
    for (int w = lane; w < words; w += 32) taken[w] = 0u;
    __syncwarp();

    for (int k = 0; k < K; ++k) {
        float bv = -INFINITY;
        int bi = 0x7fffffff;
        for (int i = lane; i < N; i += 32) {
            const bool free_ = ((taken[i >> 5] >> (i & 31)) & 1u) == 0u;
            const float x = v[i];
            if (free_ && better(x, i, bv, bi)) { bv = x; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) taken[bi >> 5] |= 1u << (bi & 31);
        __syncwarp();
    }

    // ascending emission: exclusive prefix of popcounts over the mask words
    int base = 0;
    for (int w0 = 0; w0 < words; w0 += 32) {
        const int w = w0 + lane;
        const uint32_t m = w < words ? taken[w] : 0u;
        const int cnt = __popc(m);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        int pos = base + incl - cnt;
        uint32_t mm = m;
        while (mm) {
            const int b = __ffs(mm) - 1;
            mm &= mm - 1;
            ids[(size_t)row * K + pos++] = w * 32 + b;
        }
        base += __shfl_sync(0xffffffffu, incl, 31);
    }
}

__global__ void gather_idx_kernel(const int32_t *__restrict__ ids, const int32_t *__restrict__ keep,
                                  int32_t *__restrict__ out, int64_t total, int N, int Cp, int K, int Bk) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int64_t per = (int64_t)K * Bk;
    const int64_t bg = i / per;
    const int r = (int)(i - bg * per);
    const int k = r / Bk, t = r - k * Bk;
    const int n = ids[bg * K + k];
    const int slot = keep ? keep[(bg * N + n) * (int64_t)Bk + t] : t;
    out[i] = n * Cp + slot;
}

// PDLLM_DEBUG_VALIDATE (include/pdllm.h): bit 0 = a chunk id outside [0, N); bit 1 = keep[..,0] != 0 (the BOS slot, R7);
// bit 2 = a keep slot outside [0, C]; bit 3 = a keep list that is not strictly ascending.
__global__ void validate_kernel(const int32_t *__restrict__ ids, int64_t n_ids, int N, const int32_t *__restrict__ keep,
                                int64_t n_keep, int Bk, int C, int32_t *flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int bad = 0;
    if (ids && i < n_ids) {
        const int n = ids[i];
        if (n < 0 || n >= N) bad |= 1;
    }
    if (keep && i < n_keep) {
        const int t = (int)(i % Bk), v = keep[i];
        if (t == 0 && v != 0) bad |= 2;
        if (v < 0 || v > C) bad |= 4;
        if (t > 0 && keep[i - 1] >= v) bad |= 8;
    }
    if (bad) atomicOr(flag, bad);
}

}  // namespace

cudaError_t launch_validate(const Dims &s, const int32_t *chunk_ids, const int32_t *keep, int32_t *flag, cudaStream_t st) {
    const int64_t n_ids = chunk_ids ? (int64_t)s.B * s.H_kv * s.K : 0;
    const int64_t n_keep = keep ? (int64_t)s.B * s.H_kv * s.N * s.Bk : 0;
    const int64_t total = n_ids > n_keep ? n_ids : n_keep;
    if (total == 0) return cudaSuccess;
    validate_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(chunk_ids, n_ids, s.N, keep, n_keep, s.Bk, s.C, flag);
    return cudaGetLastError();
}

cudaError_t launch_topk(const Dims &s, const float *scores, int32_t *chunk_ids, cudaStream_t st, const float *partials,
                        float *scores_out) {
    const int rows = s.B * s.H_kv;
    const int Npad = (s.N + 3) & ~3, words = (s.N + 31) >> 5;
    const size_t smem = (size_t)kTopkWarps * (Npad + words) * sizeof(float);
    static_assert((size_t)kTopkWarps * (kTopkMaxN + kTopkMaxN / 32) * 4 <= 100 * 1024, "top-K staging must fit");
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // programmatic dependent launch: its blocks fit beside the score kernel's CTAs and start the moment it ends
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((rows + kTopkWarps - 1) / kTopkWarps), 1, 1);
    cfg.blockDim = dim3(kTopkWarps * 32, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const int N = s.N, K = s.K;
    const int m_tiles = (s.G * s.L_q + kTileM - 1) / kTileM;
    return cudaLaunchKernelEx(&cfg, topk_kernel, scores, chunk_ids, rows, N, K, partials, m_tiles, scores_out);
}

cudaError_t launch_gather_idx(const Dims &s, const int32_t *chunk_ids, const int32_t *keep, int32_t *gather_idx,
                              cudaStream_t st) {
    const int64_t total = (int64_t)s.B * s.H_kv * s.K * s.Bk;
    const int threads = 256;
    gather_idx_kernel<<<(unsigned)((total + threads - 1) / threads), threads, 0, st>>>(chunk_ids, keep, gather_idx, total,
                                                                                      s.N, s.Cp, s.K, s.Bk);
    return cudaGetLastError();
}

}  // namespace pdllm
