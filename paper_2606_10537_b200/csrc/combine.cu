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
    constexpr int V = D / 32;                      // floats per lane: 4 (d=128) or 2 (d=64)
    // launched as a programmatic dependent of the kernel that writes the partials (its launch is processed while that
    // kernel still runs): wait for that grid's completion and flush before reading them
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kCombineWarps + warp;
    if (row >= rows) return;

    float big = -INFINITY;
    for (int s = lane; s < S; s += 32) big = fmaxf(big, lse_part[(int64_t)s * rows + row]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = fmaxf(big, __shfl_xor_sync(0xffffffffu, big, o));

    float acc[V];
#pragma unroll
    for (int i = 0; i < V; ++i) acc[i] = 0.f;
    float lse = -INFINITY;
    if (big > -INFINITY) {
        float tot = 0.f;
        for (int s = lane; s < S; s += 32) {
            const float x = lse_part[(int64_t)s * rows + row];
            if (x > -INFINITY) tot += __expf(x - big);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
        lse = big + __logf(tot);
        for (int s = 0; s < S; ++s) {
            const float x = lse_part[(int64_t)s * rows + row];         // warp-uniform broadcast load
            if (!(x > -INFINITY)) continue;                             // empty split contributes nothing
            const float w = __expf(x - lse);
            const float *src = O_part + ((int64_t)s * rows + row) * D + lane * V;
            if (V == 4) {
                const float4 v = *reinterpret_cast<const float4 *>(src);
                acc[0] += w * v.x; acc[1] += w * v.y; acc[V - 2] += w * v.z; acc[V - 1] += w * v.w;
            } else {
                const float2 v = *reinterpret_cast<const float2 *>(src);
                acc[0] += w * v.x; acc[1] += w * v.y;
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
