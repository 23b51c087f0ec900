// combine.cu -- a5: log-sum-exp merge of the Split-S partials (R10, R11).
//   LSE = log sum_s exp(lse_s);  O = sum_s exp(lse_s - LSE) * O_s   (O_s normalised per split)
// Pure streaming: one warp per output row, 128-bit loads of the fp32 partial rows, bf16 RNE store.
#include "pdllm_internal.h"
#include "ptx.cuh"

namespace pdllm {

namespace {

constexpr int kCombineWarps = 8;

template <int D>
__global__ void __launch_bounds__(kCombineWarps * 32) combine_kernel(const float *__restrict__ O_part,
                                                                     const float *__restrict__ lse_part, int S, int64_t rows,
                                                                     uint16_t *__restrict__ O, float *__restrict__ LSE) {
    constexpr int NB = 4;                          // partial rows in flight per lane (8 measured: no different)
    constexpr int V = D / 32;                      // floats per lane: 4 (d=128) or 2 (d=64)
    // launched as a programmatic dependent of the kernel that writes the partials (its launch is processed while that
    // kernel still runs): wait for that grid's completion and flush before reading them
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");      // (the next step's score kernel)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kCombineWarps + warp;
    if (row >= rows) return;

    // every split's log-mass of this row in ONE round trip (lane s holds splits s and s + 32; splits beyond 64 by plain loops), the weights by
    // shuffles, then the partial rows NB loads at a time: 1 + ceil(S / NB) dependent round trips per row, not 1 + S
    const float x0 = lane < S ? lse_part[(int64_t)lane * rows + row] : -INFINITY;
    const float x1 = lane + 32 < S ? lse_part[(int64_t)(lane + 32) * rows + row] : -INFINITY;
    float big = fmaxf(x0, x1);
    for (int sp = lane + 64; sp < S; sp += 32) big = fmaxf(big, lse_part[(int64_t)sp * rows + row]);   // (S > 64: never the library's own choice)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = fmaxf(big, __shfl_xor_sync(0xffffffffu, big, o));

    float acc[V];
#pragma unroll
    for (int i = 0; i < V; ++i) acc[i] = 0.f;
    float lse = -INFINITY;
    if (big > -INFINITY) {
        float tot = (x0 > -INFINITY ? __expf(x0 - big) : 0.f) + (x1 > -INFINITY ? __expf(x1 - big) : 0.f);
        for (int sp = lane + 64; sp < S; sp += 32) {
            const float x = lse_part[(int64_t)sp * rows + row];
            if (x > -INFINITY) tot += __expf(x - big);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
        lse = big + __logf(tot);
        const float w0 = x0 > -INFINITY ? __expf(x0 - lse) : 0.f;       // an empty split contributes nothing
        const float w1 = x1 > -INFINITY ? __expf(x1 - lse) : 0.f;
        const float *src = O_part + row * D + lane * V;
        for (int s0 = 0; s0 < S; s0 += NB) {
            float v[NB][V];
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const bool on = s0 + k < S;
                const float *ptr = src + (int64_t)(on ? s0 + k : s0) * rows * D;
                if (V == 4) {
                    const float4 t = *reinterpret_cast<const float4 *>(ptr);
                    v[k][0] = t.x; v[k][1] = t.y; v[k][V - 2] = t.z; v[k][V - 1] = t.w;
                } else {
                    const float2 t = *reinterpret_cast<const float2 *>(ptr);
                    v[k][0] = t.x; v[k][1] = t.y;
                }
            }
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int sp = s0 + k;
                float w = __shfl_sync(0xffffffffu, sp < 32 ? w0 : w1, sp & 31);
                if (sp >= 64 && sp < S) {
                    const float x = lse_part[(int64_t)sp * rows + row];
                    w = x > -INFINITY ? __expf(x - lse) : 0.f;
                }
                if (sp >= S) w = 0.f;
                if (w > 0.f) {                                          // (an empty split's partial row may hold anything)
#pragma unroll
                    for (int i = 0; i < V; ++i) acc[i] += w * v[k][i];
                }
            }
        }
    }
    if (lane == 0) LSE[row] = lse;
    uint16_t *dst = O + row * D + lane * V;
    if (V == 4) {
        uint2 u;
        u.x = pack_bf16x2(acc[0], acc[1]);
        u.y = pack_bf16x2(acc[V - 2], acc[V - 1]);
        *reinterpret_cast<uint2 *>(dst) = u;
    } else {
        *reinterpret_cast<uint32_t *>(dst) = pack_bf16x2(acc[0], acc[1]);
    }
}

}  // namespace

cudaError_t launch_combine(const float *O_part, const float *lse_part, int S, int64_t rows, int d, void *O, float *LSE,
                           cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((rows + kCombineWarps - 1) / kCombineWarps), 1, 1);
    cfg.blockDim = dim3(kCombineWarps * 32, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    uint16_t *Ob = static_cast<uint16_t *>(O);
    if (d == 128) return cudaLaunchKernelEx(&cfg, combine_kernel<128>, O_part, lse_part, S, rows, Ob, LSE);
    return cudaLaunchKernelEx(&cfg, combine_kernel<64>, O_part, lse_part, S, rows, Ob, LSE);
}

}  // namespace pdllm
