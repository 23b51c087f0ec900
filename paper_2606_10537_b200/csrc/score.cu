// score.cu -- a1: chunk-score reduction (Eq. 5; readings R1-R3), tcgen05 / TMEM / TMA.
//
//   scores[b,g,n] = mean over the G*L_q scoring rows of  log sum_{j<=C} exp(scale * q . Kcache[b,g,n,j])
//
// The kernel streams every cached K row exactly once (HBM-bound at MHA shapes).  Persistent CTAs (two per SM) each take
// an even share of the (b, g, M tile, chunk) units: a contiguous run of chunks, cut into segments of one (b, g, M tile)
// whose 128-row tile of scoring rows is staged in shared memory.  Each chunk is cut into 128-row K tiles (the tail
// tile is shortened to a multiple of 16 rows) that one thread fetches with TMA into a 2-stage ring of 128B-swizzled
// panels; one thread issues S = Q K^T (tcgen05.mma) into one of two TMEM accumulators; 256 softmax threads (two per
// row: columns 0-63 / 64-127 of every tile) fold the tile into their running (reference max, sum) of the current
// chunk with one exp pass -- a quarter of the exponentials as an FMA-pipe polynomial, the tile's row sum as the overflow
// detector -- and, at the chunk's last tile, merge the halves and reduce the log-masses over the rows.
#include <cuda.h>

#include "pdllm_internal.h"
#include "ptx.cuh"

namespace pdllm {

namespace {

constexpr int kScoreThreads = 320;        // 8 softmax warps (two column halves) + TMA warp + MMA warp
constexpr int kTmaWarp = 8, kMmaWarp = 9;
constexpr int kMaxChunksPerCta = 64;
constexpr int kTailGroup = 4;             // one-row tails (C = 2^k: Cp = 128 t + 1) of this many consecutive chunks share a tile step
constexpr bool kPolyShare = true;          // MUFU is co-critical with HBM here (538 M ex2 per C4 launch): offload 1/4

struct ScoreParams {
    const uint16_t *Q;
    int64_t q_batch_stride, q_head_stride;
    float *scores;
    float *row_lse;                       // optional export [B*H_kv, N, rows]: every scoring row's log-mass per chunk (NEXT-1)
    int H_kv, G, N, Cp, L_q, rows;        // rows = G * L_q
    int m_tiles;
    int64_t units;                        // (b, g, M tile, chunk) work units, split evenly over the persistent CTAs
    int64_t part_stride;                  // B*H_kv*N
    float c2, inv_rows;
    int use_atomic, evict_first;          // use_atomic: several M tiles add into scores[] (order not fixed)
    float *partials;                      // or, when given: [m_tiles, B*H_kv*N] plain stores, summed in M-tile order by the consumer
    int32_t *zero_counter;                // pdllm_step: the attention kernel's work-item counters, cleared here (no memset node)
};

template <int D>
struct ScoreCfg {
    static constexpr int kPanels = D / 64;
    static constexpr uint32_t kPanelBytes = 128 * 128;
    static constexpr uint32_t kTileBytes = kPanels * kPanelBytes;
    static constexpr int kStages = (D == 128) ? 2 : 4;
    static constexpr size_t kSmem = 1024 + (size_t)(1 + kStages) * kTileBytes;
};

template <int D>
__global__ void __launch_bounds__(kScoreThreads, 2)
score_kernel(const ScoreParams p, const __grid_constant__ CUtensorMap tmap128, const __grid_constant__ CUtensorMap tmap16) {
    using Cfg = ScoreCfg<D>;
    constexpr int ST = Cfg::kStages;
    constexpr int kChunksPerRow = D / 8;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;
    auto sK = [&](int stage) { return smem_base + Cfg::kTileBytes * (uint32_t)(1 + stage); };

    __shared__ uint64_t bars[2 * ST + 4];   // k_full[ST], k_free[ST], s_ready[2], s_free[2]
    __shared__ uint32_t tmem_slot;
    __shared__ float s_acc[kMaxChunksPerCta * 4];
    __shared__ float s_ml[2][kTileM][2];      // column half 1's (m_ref, l) per row, double-buffered by chunk parity
    __shared__ float s_tail[kTailGroup - 1][kTileM];   // tail logits (log2 units) of a group's later chunks, per row

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // a dependent kernel (top-K, launched with programmatic stream serialization) may become resident beside this one;
    // it waits for this grid's completion before it reads the scores
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // persistent CTA: a contiguous range of the units u = ((bg * m_tiles + mt) * N + n)
    const int64_t u_lo = p.units * blockIdx.x / gridDim.x, u_hi = p.units * (blockIdx.x + 1) / gridDim.x;
    const int tiles_per_chunk = (p.Cp + kTileN - 1) / kTileN;
    // A chunk of 128 t + 1 rows (C = 2^k plus the BOS row) ends in a one-row tile.  Such tails do not get a tile step each:
    // the chunks of a segment form groups of kTailGroup; after the main tiles of a group's FIRST chunk one step takes the
    // tail rows of all its chunks (a 16-row TMA box each, side by side in one ring stage, one MMA of N = 16 g) -- the
    // first chunk folds its tail in as before, the others start from theirs.  4 + 1/kTailGroup steps per chunk, not 5.
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
    if (warp == kMmaWarp) {
        tmem_alloc(smem_u32(&tmem_slot), 256);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_slot;
    int q = 0;                                // tile-step counter of the K ring / S buffers (every role counts alike)
    // The kernel is itself launched as a programmatic dependent of whatever precedes it in the stream (in a denoising loop:
    // the previous step's attention / combine kernel): the set-up above ran under that kernel's tail; nothing it may have
    // written (Q, the cache, the counters) is touched before this wait.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (p.zero_counter && blockIdx.x == 0 && tid == 0) {
        p.zero_counter[0] = 0;                // the attention kernel reads them behind its own wait on this grid
        p.zero_counter[1] = 0;
    }

    for (int64_t u = u_lo; u < u_hi;) {
    // ---- one segment: up to kMaxChunksPerCta consecutive chunks n0..n1-1 of one (bg, M tile)
    const int64_t bgm = u / p.N;
    const int n0 = (int)(u - bgm * p.N);
    const int n1 = (int)min((int64_t)p.N, (int64_t)n0 + min(u_hi - u, (int64_t)kMaxChunksPerCta));
    const int bg = (int)(bgm / p.m_tiles), mt = (int)(bgm % p.m_tiles);
    const int b = bg / p.H_kv, g = bg % p.H_kv;
    // TMA producer state of this segment; its first ST tiles go out BEFORE the Q tile is staged (every ring stage is
    // free at a segment start: the previous segment's MMAs are complete), so the two round trips overlap
    int pn = n0, ptt = 0;
    auto produce = [&](int max_tiles) {
        const uint64_t policy = l2_policy_evict_first();
        for (; pn < n1 && max_tiles > 0; --max_tiles, ++q) {
            const int64_t row0 = ((int64_t)bg * p.N + pn) * p.Cp;
            const int stage = q % ST;
            mbar_wait(k_free(stage), ((q / ST) & 1) ^ 1);
            if (ptt < main_tiles) {
                const int valid = min(kTileN, p.Cp - ptt * kTileN);
                const bool small = valid <= 16;
                mbar_arrive_expect_tx(k_full(stage), (uint32_t)(small ? 16 : 128) * D * 2);
                const CUtensorMap *tm = small ? &tmap16 : &tmap128;
                const int32_t row = (int32_t)(row0 + (int64_t)ptt * kTileN);
#pragma unroll
                for (int pnl = 0; pnl < Cfg::kPanels; ++pnl) {
                    if (p.evict_first)
                        tma_load_2d_hint(sK(stage) + pnl * Cfg::kPanelBytes, tm, pnl * 64, row, k_full(stage), policy);
                    else
                        tma_load_2d(sK(stage) + pnl * Cfg::kPanelBytes, tm, pnl * 64, row, k_full(stage));
                }
            } else {
                // the group's tail rows: chunk pn + k's last row (and the 15 rows behind it) at tile rows 16 k ..
                const int g = min(kTailGroup, n1 - pn);
                mbar_arrive_expect_tx(k_full(stage), (uint32_t)(16 * g) * D * 2);
                for (int k = 0; k < g; ++k) {
                    const int32_t row = (int32_t)(row0 + (int64_t)k * p.Cp + (int64_t)main_tiles * kTileN);
#pragma unroll
                    for (int pnl = 0; pnl < Cfg::kPanels; ++pnl)
                        tma_load_2d(sK(stage) + pnl * Cfg::kPanelBytes + (uint32_t)k * 2048u, &tmap16, pnl * 64, row, k_full(stage));
                }
            }
            // next step: the main tiles of every chunk, then -- behind a group's first chunk -- the group's tails
            const bool leader = tail_groups && (pn - n0) % kTailGroup == 0;
            if (++ptt == main_tiles + (leader ? 1 : 0)) { ptt = 0; ++pn; }
        }
    };
    if (warp == kTmaWarp && lane == 0) produce(ST);
    // Q tile (scoring rows mt*128.. of group g; row m -> head g*G + m / L_q, position m % L_q); the previous
    // segment's MMAs are complete (its softmax consumed every S tile before the barrier below was passed)
    for (int i = tid; i < kTileM * kChunksPerRow; i += kScoreThreads) {
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

    if (warp == kTmaWarp) {
        // =============================== TMA producer ===============================
        if (lane == 0) produce(INT_MAX);
        __syncwarp();
    } else if (warp == kMmaWarp) {
        // =============================== MMA issuer ===============================
        if (lane == 0) {
            for (int n = n0; n < n1; ++n) {
                const bool leader = tail_groups && (n - n0) % kTailGroup == 0;
                for (int tt = 0; tt < main_tiles + (leader ? 1 : 0); ++tt, ++q) {
                    const int stage = q % ST, buf = q & 1;
                    const int valid = min(kTileN, p.Cp - tt * kTileN);
                    const uint32_t n_mma = tt < main_tiles ? (uint32_t)(valid + 15) & ~15u : 16u * (uint32_t)min(kTailGroup, n1 - n);
                    mbar_wait(k_full(stage), (q / ST) & 1);
                    mbar_wait(s_free(buf), ((q >> 1) & 1) ^ 1);
                    tc_fence_after();
                    const uint32_t idesc = umma_idesc_bf16(kTileM, n_mma, 0, 0);
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t off = (uint32_t)(ks >> 2) * Cfg::kPanelBytes + (uint32_t)(ks & 3) * 32u;
                        umma_ss(tmem + 128u * buf, umma_desc_sw128(sQ + off, 16, 1024),
                                umma_desc_sw128(sK(stage) + off, 16, 1024), idesc, ks > 0);
                    }
                    umma_commit(s_ready(buf));
                    umma_commit(k_free(stage));
                }
            }
        }
        __syncwarp();
    } else {
        // =============================== softmax (thread = row) ===============================
        // Per chunk a running (reference max m_ref, sum l) in log2 units.  The chunk's first tile fixes m_ref with a max
        // pass; later tiles take one exp pass against it.  A 32-column block whose row sum exceeds kSumLimit (some
        // logit outgrew the reference by > 13 octaves; rare) raises m_ref by whole octaves and is recomputed.
        // Two threads per row: warps 0-3 take columns 0-63 of every tile, warps 4-7 columns 64-127 (both may read
        // the row's TMEM lanes), each with its own (m_ref, l); the halves are merged once per chunk.
        const int half = warp >> 2, row = tid & (kTileM - 1);
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32) << 16) + 64u * (uint32_t)half;
        const bool row_ok = mt * kTileM + row < p.rows;
        constexpr float kSumLimit = 8192.f;
        for (int n = n0; n < n1; ++n) {
            float m_ref = -INFINITY, l = 0.f;
            const int in_group = tail_groups ? (n - n0) % kTailGroup : 0;
            const bool leader = tail_groups && in_group == 0;
            if (in_group > 0 && half == 0) {          // the chunk starts from its tail row, taken in the group's tail step
                m_ref = s_tail[in_group - 1][row];    // (written by this very thread)
                l = 1.f;
            }
            // sum over 32 columns of 2^(c2*x - m_ref): packed f32x2 arithmetic, exponentials on the MUFU pipe
            auto block_sum = [&](const uint32_t(&v)[32]) {
                const uint64_t c2v = pack_f32x2(p.c2, p.c2), mv = pack_f32x2(-m_ref, -m_ref);
                uint64_t acc0 = 0ull, acc1 = 0ull;
#pragma unroll
                for (int e = 0; e < 32; e += 4) {
                    float x0, x1, x2, x3, p0, p1;
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e], v[e + 1]), c2v, mv), x0, x1);
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e + 2], v[e + 3]), c2v, mv), x2, x3);
                    if ((e & 4) == 0 && kPolyShare) {     // a share of the exponentials runs on the FMA pipe
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
                const int valid = min(kTileN, p.Cp - tt * kTileN);
                const uint32_t tS = tmem + 128u * buf + lane_base;
                mbar_wait(s_ready(buf), (q >> 1) & 1);
                tc_fence_after();
                if (valid == kTileN) {
                    uint32_t va[32], vb[32];
                    bool max_pass = tt == 0;
                    float tsum;
                    for (;;) {
                        if (max_pass) {
                            float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
                            tmem_ld32(tS, va);
                            tmem_ld32(tS + 32u, vb);
                            tmem_wait_ld();
#pragma unroll
                            for (int e = 0; e < 32; ++e)
                                mx[e & 3] = fmaxf(mx[e & 3], fmaxf(__uint_as_float(va[e]), __uint_as_float(vb[e])));
                            const float tm2 = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * p.c2;
                            if (tt == 0 && !(l > 0.f)) {
                                m_ref = tm2;
                            } else {                      // raise the reference by whole octaves (exact rescale of l)
                                const float up = fmaxf(ceilf(tm2 - m_ref), 0.f);
                                l *= ex2_approx(-up);
                                m_ref += up;
                            }
                        }
                        // this thread's 64 columns; the second TMEM load flies under the first block's arithmetic
                        tmem_ld32(tS, va);
                        tmem_wait_ld();
                        tmem_ld32(tS + 32u, vb);
                        tsum = block_sum(va);
                        tmem_wait_ld();
                        tsum += block_sum(vb);
                        // some logit outgrew the reference by > 13 octaves (rare): redo the tile behind a max pass
                        if (!__any_sync(0xffffffffu, !(tsum <= 2.f * kSumLimit))) break;
                        max_pass = true;
                    }
                    tc_fence_before();
                    mbar_arrive(s_free(buf));
                    l += tsum;
                } else if (valid == 1) {
                    // the one-row tail of a C = 2^k chunk (Cp = C + 1 with the BOS row): a single column, taken by the
                    // threads of column half 0 alone
                    if (half == 0) {
                        const uint32_t xv = tmem_ld1(tS);
                        uint32_t xg[kTailGroup - 1];
                        if (leader) {                     // the tails of the group's other chunks sit 16 columns apart
#pragma unroll
                            for (int k = 0; k < kTailGroup - 1; ++k) xg[k] = tmem_ld1(tS + 16u * (k + 1));
                        }
                        tmem_wait_ld();
                        if (leader) {
#pragma unroll
                            for (int k = 0; k < kTailGroup - 1; ++k) s_tail[k][row] = __uint_as_float(xg[k]) * p.c2;
                        }
                        const float x2 = __uint_as_float(xv) * p.c2;
                        tc_fence_before();
                        mbar_arrive(s_free(buf));
                        const float m_new = fmaxf(m_ref, x2);
                        l = l * ex2_approx(m_ref - m_new) + ex2_approx(x2 - m_new);
                        m_ref = m_new;
                    } else {
                        tc_fence_before();
                        mbar_arrive(s_free(buf));
                    }
                } else {
                    // ragged tail tile of the chunk: online update per 32-column block with column masks
                    const int mine = max(0, min(64, valid - 64 * half));       // valid columns of this thread's half
                    const int nchunks = (mine + 31) >> 5;
                    if (nchunks == 0) {
                        tc_fence_before();
                        mbar_arrive(s_free(buf));
                    }
                    for (int ch = 0; ch < nchunks; ++ch) {
                        uint32_t v[32];
                        tmem_ld32(tS + 32u * ch, v);
                        tmem_wait_ld();
                        if (ch == nchunks - 1) {
                            tc_fence_before();
                            mbar_arrive(s_free(buf));
                        }
                        const int nv = mine - ch * 32;
                        float cmax = -INFINITY;
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (e < nv) cmax = fmaxf(cmax, __uint_as_float(v[e]));
                        const float m_new = fmaxf(m_ref, cmax * p.c2);
                        float sum = 0.f;
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (e < nv) sum += ex2_approx(fmaf(__uint_as_float(v[e]), p.c2, -m_new));
                        l = l * ex2_approx(m_ref - m_new) + sum;
                        m_ref = m_new;
                    }
                }
            }
            // chunk n finished: merge the two column halves, then the log-mass of this row, summed over the tile's rows
            float(*ml)[2] = s_ml[(n - n0) & 1];
            if (half == 1) {
                ml[row][0] = m_ref;
                ml[row][1] = l;
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");
            if (half == 0) {
                const float m1 = ml[row][0], l1 = ml[row][1];
                const float m = fmaxf(m_ref, m1);
                const float lt = l * ex2_approx(m_ref - m) + (l1 > 0.f ? l1 * ex2_approx(m1 - m) : 0.f);
                float ell = row_ok ? (m + lg2_approx(lt)) * 0.6931471805599453f : 0.f;
                if (p.row_lse && row_ok) p.row_lse[((int64_t)bg * p.N + n) * p.rows + mt * kTileM + row] = ell;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) ell += __shfl_xor_sync(0xffffffffu, ell, o);
                if (lane == 0) s_acc[(n - n0) * 4 + warp] = ell;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (tid < n1 - n0) {
        const float tot = ((s_acc[tid * 4 + 0] + s_acc[tid * 4 + 1]) + (s_acc[tid * 4 + 2] + s_acc[tid * 4 + 3])) * p.inv_rows;
        float *dst = p.scores + (int64_t)bg * p.N + n0 + tid;
        if (p.partials) p.partials[(int64_t)mt * p.part_stride + (int64_t)bg * p.N + n0 + tid] = tot;
        else if (p.use_atomic) atomicAdd(dst, tot);
        else *dst = tot;
    }
    u += n1 - n0;
    }   // segments
    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp) tmem_dealloc(tmem, 256);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess)
            f = nullptr;
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}

}  // namespace

// bf16 [rows, d] row-major, box = [box_rows, 64 columns], 128-byte swizzle, OOB rows read as zero.
bool make_rows_tmap(CUtensorMap *tm, const void *base, uint64_t rows, int d, int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)d, rows};
    cuuint64_t strides[1] = {(cuuint64_t)d * 2};
    cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    cuuint32_t es[2] = {1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool make_rows_tmap3d(CUtensorMap *tm, const void *base, uint64_t groups, uint64_t rows, int d, int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)d, rows, groups};
    cuuint64_t strides[2] = {(cuuint64_t)d * 2, (cuuint64_t)d * 2 * rows};
    cuuint32_t box[3] = {64, (cuuint32_t)box_rows, 1};
    cuuint32_t es[3] = {1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

namespace {

template <int D>
cudaError_t launch_score_d(const ScoreParams &p, const CUtensorMap &t128, const CUtensorMap &t16, int BG, cudaStream_t st) {
    using Cfg = ScoreCfg<D>;
    cudaError_t e = cudaFuncSetAttribute(score_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmem);
    if (e != cudaSuccess) return e;
    const int64_t slots = 2ll * device_num_sms();          // two CTAs per SM
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p.units < slots ? p.units : slots), 1, 1);
    cfg.blockDim = dim3(kScoreThreads, 1, 1);
    cfg.dynamicSmemBytes = Cfg::kSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, score_kernel<D>, p, t128, t16);
}

}  // namespace

cudaError_t launch_score(const Dims &s, const void *Q, int64_t q_batch_stride, int64_t q_head_stride, const void *Kcache,
                         float *scores, float *row_lse, float *partials, cudaStream_t st, int32_t *zero_counter) {
    ScoreParams p;
    p.zero_counter = zero_counter;
    p.Q = static_cast<const uint16_t *>(Q);
    p.q_batch_stride = q_batch_stride;
    p.q_head_stride = q_head_stride;
    p.scores = scores;
    p.row_lse = row_lse;
    p.H_kv = s.H_kv; p.G = s.G; p.N = s.N; p.Cp = s.Cp; p.L_q = s.L_q;
    p.rows = s.G * s.L_q;
    p.m_tiles = (p.rows + kTileM - 1) / kTileM;
    const int BG = s.B * s.H_kv;
    p.units = (int64_t)BG * s.N * p.m_tiles;
    p.c2 = s.scale * 1.4426950408889634f;
    p.inv_rows = 1.0f / (float)p.rows;
    p.partials = p.m_tiles > 1 ? partials : nullptr;
    p.part_stride = (int64_t)BG * s.N;
    p.use_atomic = p.m_tiles > 1 && !p.partials;
    p.evict_first = p.m_tiles == 1;

    CUtensorMap t128, t16;
    const uint64_t rows = (uint64_t)BG * s.N * s.Cp;
    if (!make_rows_tmap(&t128, Kcache, rows, s.d, 128) || !make_rows_tmap(&t16, Kcache, rows, s.d, 16))
        return cudaErrorInvalidValue;
    if (p.use_atomic) {
        cudaError_t e = cudaMemsetAsync(scores, 0, sizeof(float) * (size_t)BG * s.N, st);
        if (e != cudaSuccess) return e;
    }
    return s.d == 128 ? launch_score_d<128>(p, t128, t16, BG, st) : launch_score_d<64>(p, t128, t16, BG, st);
}

}  // namespace pdllm
