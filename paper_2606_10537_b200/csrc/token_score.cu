// token_score.cu -- SURVEY 8(f) NEXT-1: intra-chunk token eviction scores and top-B retention on the device
// (Eq. 5, query->chunk term, Table 7 "query-to-chunk" P:457-465; readings R7, R22).
//
//   e[b,g,n,j] = sum over the G*L_q scoring rows m of  exp( scale * q_m . Kcache[b,g,n,j]  -  ell[m,n] ),
//   ell[m,n]   = log sum_{j'<=C} exp(scale * q_m . Kcache[b,g,n,j'])      (the row's log-mass inside chunk n)
//
// Two passes over the K cache: the chunk-score kernel (score.cu) exports ell[m,n] -- it computes it anyway --, then
// token_score_kernel streams every cached K row once more with the SAME persistent TMA -> tcgen05 -> TMEM pipeline,
// the MMA operands swapped: S^T = K_tile (A, M = 128 cache slots) x Q_tile^T (B, N = 128 scoring rows), so that a
// cache slot is a TMEM lane and its score is a row sum -- no reduction across threads.  Two threads per slot (column
// halves, as in score.cu); the per-column subtrahend ell comes from shared memory as broadcast 128-bit loads; a quarter
// of the exponentials run as the FMA-pipe polynomial.  HBM-bound at MHA shapes like the chunk-score kernel.
// topb_kernel: one CTA per chunk, MSB-first radix select on order-preserving integer keys, ties to the lower slot,
// ascending emission, slot 0 (BOS) always kept; topb_warp_kernel: one warp per chunk (C <= 1024, many chunks).
#include <cuda.h>

#include "pdllm_internal.h"
#include "ptx.cuh"

namespace pdllm {

namespace {

constexpr int kTokThreads = 320;          // 8 softmax warps (two column halves) + TMA warp + MMA warp
constexpr int kTokTmaWarp = 8, kTokMmaWarp = 9;
constexpr int kTokTailGroup = 4;         // one-row tails (Cp = 128 t + 1) of this many consecutive chunks share a tile step (as in score.cu)

struct TokParams {
    const uint16_t *Q;
    int64_t q_batch_stride, q_head_stride;
    const float *row_lse;                 // [B*H_kv, N, rows] natural log
    float *e;                             // [m_tiles (only when > 1), B*H_kv, N, Cp]
    int H_kv, G, N, Cp, L_q, rows, m_tiles;
    int64_t units, part_stride;           // part_stride = B*H_kv*N*Cp
    float c2;
};

template <int D>
struct TokCfg {
    static constexpr int kPanels = D / 64;
    static constexpr uint32_t kPanelBytes = 128 * 128;
    static constexpr uint32_t kTileBytes = kPanels * kPanelBytes;
    static constexpr int kStages = (D == 128) ? 2 : 4;
    static constexpr size_t kSmem = 1024 + (size_t)(1 + kStages) * kTileBytes;
};

template <int D>
__global__ void __launch_bounds__(kTokThreads, 2)
token_score_kernel(const TokParams p, const __grid_constant__ CUtensorMap tmap128, const __grid_constant__ CUtensorMap tmap16) {
    using Cfg = TokCfg<D>;
    constexpr int ST = Cfg::kStages;
    constexpr int kChunksPerRow = D / 8;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;
    auto sK = [&](int stage) { return smem_base + Cfg::kTileBytes * (uint32_t)(1 + stage); };

    __shared__ uint64_t bars[2 * ST + 4];     // k_full[ST], k_free[ST], s_ready[2], s_free[2]
    __shared__ uint32_t tmem_slot;
    __shared__ __align__(16) float s_l2[2][kTileM];      // -ell * log2(e) per scoring row of the tile (+inf beyond the rows)
    __shared__ float s_e1[2][kTileM];         // column half 1's partial sums, double-buffered by tile parity
    __shared__ __align__(16) float s_l2t[kTokTailGroup][kTileM];   // -ell * log2(e) of a tail group's chunks (the shared tail step)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t u_lo = p.units * blockIdx.x / gridDim.x, u_hi = p.units * (blockIdx.x + 1) / gridDim.x;
    const int tiles_per_chunk = (p.Cp + kTileN - 1) / kTileN;
    // chunks of 128 t + 1 rows: the one-row tails of kTokTailGroup consecutive chunks of a segment are taken in ONE tile step
    // behind the main tiles of the group's first chunk (16-row TMA boxes side by side: chunk n + k's tail slot is tile row 16 k)
    const bool tail_groups = tiles_per_chunk > 1 && p.Cp - (tiles_per_chunk - 1) * kTileN == 1;
    const int main_tiles = tail_groups ? tiles_per_chunk - 1 : tiles_per_chunk;

    const uint32_t bar0 = smem_u32(&bars[0]);
    auto k_full = [&](int s) { return bar0 + 8u * s; };
    auto k_free = [&](int s) { return bar0 + 8u * (ST + s); };
    auto s_ready = [&](int i) { return bar0 + 8u * (2 * ST + i); };
    auto s_free = [&](int i) { return bar0 + 8u * (2 * ST + 2 + i); };

    if (tid == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(k_full(s), 1); mbar_init(k_free(s), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(s_ready(i), 1); mbar_init(s_free(i), 256); }
        fence_mbar_init();
        tma_prefetch_desc(&tmap128);
        tma_prefetch_desc(&tmap16);
    }
    if (warp == kTokMmaWarp) {
        tmem_alloc(smem_u32(&tmem_slot), 256);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_slot;
    int q = 0;                                // tile-step counter of the K ring / S buffers (every role counts alike)

    for (int64_t u = u_lo; u < u_hi;) {
    // ---- one segment: consecutive chunks n0..n1-1 of one (bg, M tile of scoring rows); units as in score.cu
    const int64_t bgm = u / p.N;
    const int n0 = (int)(u - bgm * p.N);
    const int n1 = (int)min((int64_t)p.N, (int64_t)n0 + (u_hi - u));
    const int bg = (int)(bgm / p.m_tiles), mt = (int)(bgm % p.m_tiles);
    const int b = bg / p.H_kv, g = bg % p.H_kv;
    for (int i = tid; i < kTileM * kChunksPerRow; i += kTokThreads) {
        const int r = i / kChunksPerRow, c = i % kChunksPerRow;
        const int m = mt * kTileM + r;
        const bool ok = m < p.rows;
        const int hh = ok ? m / p.L_q : 0, qi = ok ? m % p.L_q : 0;
        const uint16_t *src = p.Q + (int64_t)b * p.q_batch_stride + (int64_t)(g * p.G + hh) * p.q_head_stride +
                              (int64_t)qi * D + c * 8;
        cp_async16_zfill(sQ + (uint32_t)(c >> 3) * Cfg::kPanelBytes + sw128_off(r, c & 7), src, ok ? 16u : 0u);
    }
    cp_async_commit();
    cp_async_wait<0>();
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (warp == kTokTmaWarp) {
        if (lane == 0) {
            const uint64_t policy = l2_policy_evict_first();
            for (int n = n0; n < n1; ++n) {
                const int64_t row0 = ((int64_t)bg * p.N + n) * p.Cp;
                const bool leader = tail_groups && (n - n0) % kTokTailGroup == 0;
                for (int tt = 0; tt < main_tiles + (leader ? 1 : 0); ++tt, ++q) {
                    const int stage = q % ST;
                    const int valid = min(kTileN, p.Cp - tt * kTileN);
                    const bool small = valid <= 16;
                    mbar_wait(k_free(stage), ((q / ST) & 1) ^ 1);
                    if (tt == main_tiles && tail_groups) {
                        const int g = min(kTokTailGroup, n1 - n);
                        mbar_arrive_expect_tx(k_full(stage), (uint32_t)(16 * g) * D * 2);
                        for (int k = 0; k < g; ++k) {
                            const int32_t trow = (int32_t)(row0 + (int64_t)k * p.Cp + (int64_t)main_tiles * kTileN);
#pragma unroll
                            for (int pn = 0; pn < Cfg::kPanels; ++pn)
                                tma_load_2d(sK(stage) + pn * Cfg::kPanelBytes + (uint32_t)k * 2048u, &tmap16, pn * 64, trow, k_full(stage));
                        }
                        continue;
                    }
                    mbar_arrive_expect_tx(k_full(stage), (uint32_t)(small ? 16 : 128) * D * 2);
                    const CUtensorMap *tm = small ? &tmap16 : &tmap128;
                    const int32_t row = (int32_t)(row0 + (int64_t)tt * kTileN);
#pragma unroll
                    for (int pn = 0; pn < Cfg::kPanels; ++pn) {
                        if (p.m_tiles == 1)
                            tma_load_2d_hint(sK(stage) + pn * Cfg::kPanelBytes, tm, pn * 64, row, k_full(stage), policy);
                        else
                            tma_load_2d(sK(stage) + pn * Cfg::kPanelBytes, tm, pn * 64, row, k_full(stage));
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == kTokMmaWarp) {
        // S^T[slot, scoring row] = K_tile . Q_tile^T: the K tile is the A operand (M = 128 cache slots; slots past the
        // tile's valid rows hold stale shared memory and only ever reach their own, unread lanes), Q the B operand
        if (lane == 0) {
            constexpr uint32_t idesc = umma_idesc_bf16(kTileM, kTileN, 0, 0);
            for (int n = n0; n < n1; ++n) {
                const bool leader = tail_groups && (n - n0) % kTokTailGroup == 0;
                for (int tt = 0; tt < main_tiles + (leader ? 1 : 0); ++tt, ++q) {
                    const int stage = q % ST, buf = q & 1;
                    mbar_wait(k_full(stage), (q / ST) & 1);
                    mbar_wait(s_free(buf), ((q >> 1) & 1) ^ 1);
                    tc_fence_after();
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t off = (uint32_t)(ks >> 2) * Cfg::kPanelBytes + (uint32_t)(ks & 3) * 32u;
                        umma_ss(tmem + 128u * buf, umma_desc_sw128(sK(stage) + off, 16, 1024),
                                umma_desc_sw128(sQ + off, 16, 1024), idesc, ks > 0);
                    }
                    umma_commit(s_ready(buf));
                    umma_commit(k_free(stage));
                }
            }
        }
        __syncwarp();
    } else {
        // =============================== row sums of exp(z - ell) (two threads per cache slot) ===============================
        const int half = warp >> 2, row = tid & (kTileM - 1);
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32) << 16) + 64u * (uint32_t)half;
        const uint32_t pair_bar = 2u + (uint32_t)(warp & 3);
        const float kLog2e = 1.4426950408889634f;
        auto load_l2 = [&](int n) -> float {           // -ell in log2 units for column `tid` of chunk n (threads 0..127)
            const int m = mt * kTileM + tid;
            return m < p.rows ? -__ldg(p.row_lse + ((int64_t)bg * p.N + n) * p.rows + m) * kLog2e : -INFINITY;
        };
        float l2_next = tid < kTileM ? load_l2(n0) : 0.f;
        float lt[kTokTailGroup];                       // the next tail group's values (threads 0..127), one group ahead
#pragma unroll
        for (int k = 0; k < kTokTailGroup; ++k) lt[k] = (tail_groups && tid < kTileM && n0 + k < n1) ? load_l2(n0 + k) : 0.f;
        float *e_out = p.e + (int64_t)mt * p.part_stride;
        for (int n = n0; n < n1; ++n) {
            const int par = (n - n0) & 1;
            const bool leader = tail_groups && (n - n0) % kTokTailGroup == 0;
            const int g = min(kTokTailGroup, n1 - n);      // chunks in the group this chunk leads
            if (tid < kTileM) {
                s_l2[par][tid] = l2_next;
                if (n + 1 < n1) l2_next = load_l2(n + 1);       // in flight under this chunk's tiles
                if (leader) {
#pragma unroll
                    for (int k = 0; k < kTokTailGroup; ++k) {
                        s_l2t[k][tid] = lt[k];
                        if (n + kTokTailGroup + k < n1) lt[k] = load_l2(n + kTokTailGroup + k);
                    }
                }
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");
            const float4 *l2v = reinterpret_cast<const float4 *>(&s_l2[par][64 * half]);
            // sum over 32 columns of 2^(c2*x - ell2[col]): packed f32x2 arithmetic, a quarter of the exponentials as polynomial
            auto block_sum = [&](const uint32_t(&v)[32], int c0, const float4 *l2v) {
                const uint64_t c2v = pack_f32x2(p.c2, p.c2);
                uint64_t acc0 = 0ull, acc1 = 0ull;
#pragma unroll
                for (int e = 0; e < 32; e += 4) {
                    const float4 m4 = l2v[(c0 + e) >> 2];
                    float x0, x1, x2, x3, p0, p1;
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e], v[e + 1]), c2v, pack_f32x2(m4.x, m4.y)), x0, x1);
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e + 2], v[e + 3]), c2v, pack_f32x2(m4.z, m4.w)), x2, x3);
                    if ((e & 4) == 0) {
                        ex2_poly_x2(x0, x1, p0, p1);
                    } else {
                        p0 = ex2_approx(x0);
                        p1 = ex2_approx(x1);
                    }
                    acc0 = add_f32x2(acc0, pack_f32x2(p0, p1));
                    acc1 = add_f32x2(acc1, pack_f32x2(ex2_approx(x2), ex2_approx(x3)));
                }
                float s0, s1, s2, s3;
                unpack_f32x2(acc0, s0, s1);
                unpack_f32x2(acc1, s2, s3);
                return (s0 + s1) + (s2 + s3);
            };
            for (int tt = 0; tt < main_tiles + (leader ? 1 : 0); ++tt, ++q) {
                const int buf = q & 1;
                const bool group_tail = tail_groups && tt == main_tiles;
                // rows of the tile that are cache slots: a tile's first `valid` rows, or, in a group's tail step, rows 0, 16, ..
                const int valid = group_tail ? 16 * (g - 1) + 1 : min(kTileN, p.Cp - tt * kTileN);
                const uint32_t tS = tmem + 128u * buf + lane_base;
                mbar_wait(s_ready(buf), (q >> 1) & 1);
                tc_fence_after();
                if ((warp & 3) * 32 >= valid) {           // ragged tail tile: none of this warp's 32 slots is a cache row
                    tc_fence_before();
                    mbar_arrive(s_free(buf));
                    asm volatile("bar.sync %0, 64;" ::"r"(pair_bar) : "memory");
                    continue;
                }
                uint32_t va[32], vb[32];
                tmem_ld32(tS, va);
                tmem_wait_ld();
                tmem_ld32(tS + 32u, vb);
                // the subtrahends: this chunk's, or in a group's tail step those of the chunk whose tail this slot is
                const int kk = group_tail ? min(row >> 4, g - 1) : 0;
                const float4 *lv = group_tail ? reinterpret_cast<const float4 *>(&s_l2t[kk][64 * half]) : l2v;
                float sum = block_sum(va, 0, lv);
                tmem_wait_ld();
                tc_fence_before();
                mbar_arrive(s_free(buf));
                sum += block_sum(vb, 32, lv);
                if (half == 1) s_e1[q & 1][row] = sum;
                asm volatile("bar.sync %0, 64;" ::"r"(pair_bar) : "memory");
                if (half == 0) {
                    if (group_tail) {
                        if ((row & 15) == 0 && (row >> 4) < g)
                            e_out[((int64_t)bg * p.N + n + (row >> 4)) * p.Cp + tt * kTileN] = sum + s_e1[q & 1][row];
                    } else if (row < valid) {
                        e_out[((int64_t)bg * p.N + n) * p.Cp + tt * kTileN + row] = sum + s_e1[q & 1][row];
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    u += n1 - n0;
    }   // segments
    tc_fence_before();
    __syncthreads();
    if (warp == kTokMmaWarp) tmem_dealloc(tmem, 256);
}

// e[i] = sum over the M tiles' partials, in M-tile order (bit-reproducible)
__global__ void token_reduce_kernel(const float *__restrict__ part, float *__restrict__ e, int64_t n, int m_tiles) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s = 0.f;
    for (int mt = 0; mt < m_tiles; ++mt) s += part[(int64_t)mt * n + i];
    e[i] = s;
}

// ------------------------------------------------------------------ top-B retention (R7)
constexpr int kTopbThreads = 256;
constexpr int kTopbMaxCp = 8192;

// order-preserving key: larger float <=> larger key; NaN counts as -inf; -0 as +0
__device__ __forceinline__ uint32_t order_key(float x) {
    if (x != x) x = -INFINITY;
    uint32_t u = __float_as_uint(x);
    if (u == 0x80000000u) u = 0u;
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// exclusive prefix sum of one int per thread over the block (256 threads); returns the block total through `total`
__device__ __forceinline__ int block_excl_scan(int v, int *s_warp, int &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();                          // s_warp may still be read from the previous call
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int base = 0;
    total = 0;
#pragma unroll
    for (int w = 0; w < kTopbThreads / 32; ++w) {
        const int t = s_warp[w];
        if (w < warp) base += t;
        total += t;
    }
    return base + incl - v;
}

__global__ void __launch_bounds__(kTopbThreads) topb_kernel(const float *__restrict__ e, int32_t *__restrict__ keep, int Cp, int Bk) {
    extern __shared__ uint32_t s_key[];       // Cp keys
    __shared__ int s_hist[256];
    __shared__ int s_warp[kTopbThreads / 32];
    __shared__ uint32_t s_prefix;
    __shared__ int s_need;
    const int tid = threadIdx.x;
    const float *src = e + (int64_t)blockIdx.x * Cp;
    int32_t *dst = keep + (int64_t)blockIdx.x * Bk;
    for (int j = tid; j < Cp; j += kTopbThreads) s_key[j] = order_key(src[j]);
    if (tid == 0) {
        dst[0] = 0;                           // BOS is always kept (R7)
        s_prefix = 0u;
        s_need = Bk - 1;
    }
    __syncthreads();
    if (Bk == 1) return;
    // MSB-first radix select of the (Bk-1)-th largest key among slots 1..Cp-1
    for (int shift = 24; shift >= 0; shift -= 8) {
        s_hist[tid] = 0;
        __syncthreads();
        const uint32_t prefix = s_prefix;
        const uint32_t mask = shift == 24 ? 0u : (0xffffffffu << (shift + 8));
        for (int j = 1 + tid; j < Cp; j += kTopbThreads) {
            const uint32_t k = s_key[j];
            if ((k & mask) == prefix) atomicAdd(&s_hist[(k >> shift) & 0xffu], 1);
        }
        __syncthreads();
        if (tid < 32) {
            // warp 0 walks the 256 bins from the top: lane l owns bins 255 - 8l .. 248 - 8l; a suffix scan over the
            // lanes finds the lane in whose bins the need-th largest key falls, which then walks its eight bins
            const int need = s_need;
            int h[8], mine = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                h[i] = s_hist[255 - 8 * tid - i];
                mine += h[i];
            }
            int incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (tid >= o) incl += t;
            }
            const int before = incl - mine;                   // keys in the bins above this lane's
            if (before < need && need <= incl) {
                int left = need - before, d = 255 - 8 * tid;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (h[i] >= left) break;
                    left -= h[i];
                    --d;
                }
                s_prefix = prefix | ((uint32_t)d << shift);
                s_need = left;                // how many keys equal to the final threshold are taken (lowest slots first)
            }
        }
        __syncthreads();
    }
    const uint32_t T = s_prefix;
    const int need_eq = s_need;
    // ordered pass: keep key > T, and the first need_eq slots with key == T; emit ascending
    int run_eq = 0, run_out = 1;
    for (int base = 1; base < Cp; base += kTopbThreads) {
        const int j = base + tid;
        const uint32_t k = j < Cp ? s_key[j] : 0u;
        const int eq = (j < Cp && k == T) ? 1 : 0;
        int tot_eq, tot_sel;
        const int rank = block_excl_scan(eq, s_warp, tot_eq);
        const int sel = (j < Cp && (k > T || (eq && run_eq + rank < need_eq))) ? 1 : 0;
        const int pos = block_excl_scan(sel, s_warp, tot_sel);
        if (sel) dst[run_out + pos] = j;
        run_eq += tot_eq;
        run_out += tot_sel;
    }
}

template <int D>
cudaError_t launch_tok_d(const TokParams &p, const CUtensorMap &t128, const CUtensorMap &t16, cudaStream_t st) {
    using Cfg = TokCfg<D>;
    cudaError_t e = cudaFuncSetAttribute(token_score_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmem);
    if (e != cudaSuccess) return e;
    const int64_t slots = 2ll * device_num_sms();
    dim3 grid((unsigned)(p.units < slots ? p.units : slots), 1, 1);
    token_score_kernel<D><<<grid, kTokThreads, Cfg::kSmem, st>>>(p, t128, t16);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_token_scores(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                                const void *Kcache, const float *row_lse, float *e, float *e_part, cudaStream_t st) {
    TokParams p;
    p.Q = static_cast<const uint16_t *>(Q);
    p.q_batch_stride = q_batch_stride;
    p.q_head_stride = q_head_stride;
    p.row_lse = row_lse;
    p.H_kv = s.H_kv; p.G = s.G; p.N = s.N; p.Cp = s.Cp; p.L_q = s.L_q;
    p.rows = s.G * s.L_q;
    p.m_tiles = (p.rows + kTileM - 1) / kTileM;
    const int64_t BG = (int64_t)s.B * s.H_kv;
    p.units = BG * s.N * p.m_tiles;
    p.part_stride = BG * s.N * s.Cp;
    p.e = p.m_tiles > 1 ? e_part : e;
    p.c2 = s.scale * 1.4426950408889634f;
    CUtensorMap t128, t16;
    const uint64_t rows = (uint64_t)BG * s.N * s.Cp;
    if (!make_rows_tmap(&t128, Kcache, rows, s.d, 128) || !make_rows_tmap(&t16, Kcache, rows, s.d, 16))
        return cudaErrorInvalidValue;
    cudaError_t err = s.d == 128 ? launch_tok_d<128>(p, t128, t16, st) : launch_tok_d<64>(p, t128, t16, st);
    if (err != cudaSuccess || p.m_tiles == 1) return err;
    token_reduce_kernel<<<(unsigned)((p.part_stride + 255) / 256), 256, 0, st>>>(e_part, e, p.part_stride, p.m_tiles);
    return cudaGetLastError();
}

int topb_max_cp() { return kTopbMaxCp; }

// Chunks of up to 32 R + 1 slots: one WARP per chunk, the keys of slots 1..C in registers (lane l: slots 1 + l, 33 + l, ...).
// The threshold T = the (Bk-1)-th largest key is built bit by bit from the top (T |= bit whenever at least Bk-1 keys are
// >= the candidate: 32 rounds of R compares and one warp reduction), then one ordered pass emits the kept slots ascending
// with ballots and popcount prefixes.  No shared memory, no block barriers.  The search stops as soon as exactly Bk-1 keys
// lie at or above the candidate (distinct scores: after ~20 of the 32 rounds).
constexpr int kTopbWarps = 8;

template <int R>
__global__ void __launch_bounds__(kTopbWarps * 32) topb_warp_kernel(const float *__restrict__ e, int32_t *__restrict__ keep,
                                                                    int chunks, int Cp, int Bk) {
    const int lane = threadIdx.x & 31;
    const int chunk = blockIdx.x * kTopbWarps + (threadIdx.x >> 5);
    if (chunk >= chunks) return;
    const float *src = e + (int64_t)chunk * Cp;
    int32_t *dst = keep + (int64_t)chunk * Bk;
    uint32_t key[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = 1 + r * 32 + lane;
        key[r] = j < Cp ? order_key(__ldg(src + j)) : 0u;         // 0 is below every real key (order_key(-inf) = 0x007fffff)
    }
    if (lane == 0) dst[0] = 0;                                    // BOS is always kept (R7)
    const int want = Bk - 1;
    if (want == 0) return;
    uint32_t T = 0u;
#pragma unroll 1
    for (int bit = 31; bit >= 0; --bit) {
        const uint32_t cand = T | (1u << bit);
        int cnt = 0;
#pragma unroll
        for (int r = 0; r < R; ++r) cnt += key[r] >= cand ? 1 : 0;
        const int c = (int)__reduce_add_sync(0xffffffffu, (unsigned)cnt);
        if (c >= want) {
            T = cand;
            if (c == want) break;             // exactly the keys >= T: the lower bits cannot change the selection
        }
    }
    int above = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) above += key[r] > T ? 1 : 0;
    const int need_eq = want - (int)__reduce_add_sync(0xffffffffu, (unsigned)above);   // keys equal to T to take, lowest slots first
    const uint32_t lt = (1u << lane) - 1u;
    int out = 1, eq_seen = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = 1 + r * 32 + lane;
        const bool in = j < Cp;
        const bool eq = in && key[r] == T;
        const uint32_t eq_mask = __ballot_sync(0xffffffffu, eq);
        const bool sel = in && (key[r] > T || (eq && eq_seen + __popc(eq_mask & lt) < need_eq));
        const uint32_t sel_mask = __ballot_sync(0xffffffffu, sel);
        if (sel) dst[out + __popc(sel_mask & lt)] = j;
        out += __popc(sel_mask);
        eq_seen += __popc(eq_mask);
    }
}

cudaError_t launch_topb(const Dims &s, const float *token_scores, int32_t *keep, cudaStream_t st) {
    const unsigned chunks = (unsigned)((int64_t)s.B * s.H_kv * s.N);
    // one warp per chunk pays when there are warps enough to fill the GPU (C4: 8192 chunks, 53 -> 17 us); with few chunks
    // the CTA-per-chunk kernel below has more threads on each of them
    if (s.Cp - 1 <= 32 * 32 && chunks >= 1024u) {
        const unsigned grid = (chunks + kTopbWarps - 1) / kTopbWarps;
        if (s.Cp - 1 <= 32 * 4) topb_warp_kernel<4><<<grid, kTopbWarps * 32, 0, st>>>(token_scores, keep, (int)chunks, s.Cp, s.Bk);
        else if (s.Cp - 1 <= 32 * 16) topb_warp_kernel<16><<<grid, kTopbWarps * 32, 0, st>>>(token_scores, keep, (int)chunks, s.Cp, s.Bk);
        else topb_warp_kernel<32><<<grid, kTopbWarps * 32, 0, st>>>(token_scores, keep, (int)chunks, s.Cp, s.Bk);
        return cudaGetLastError();
    }
    const size_t smem = (size_t)s.Cp * sizeof(uint32_t);
    topb_kernel<<<chunks, kTopbThreads, smem, st>>>(token_scores, keep, s.Cp, s.Bk);
    return cudaGetLastError();
}

}  // namespace pdllm
