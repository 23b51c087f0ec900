// attn.cu -- a3 + a4: index-driven gather of the selected BOS+chunk KV rows and the Split-S partial
// attention kernel (R7-R11), tcgen05 / TMEM, sm_100a.
//
// One CTA = one 128-row tile of the G*L query rows that share a KV head (GQA groups are packed into
// the MMA M dimension, so K/V are read once per group) x one split of the virtual KV sequence
//     [ K*Bk gathered cache rows  ||  L_s decode-block rows ].
// Per 128-row KV tile:  producers (4 warps) gather K and V rows with 16-byte cp.async into
// 128B-swizzled shared-memory panels;  one thread issues  S = Q K^T  (tcgen05.mma, SS) into TMEM;
// the 128 softmax threads (thread = row) read S with tcgen05.ld, keep the running reference max / sum,
// write P = exp2(.) as packed bf16 back into TMEM (aliasing S);  the MMA thread issues  O += P V
// (tcgen05.mma, A from TMEM, V as MN-major B).  Two CTAs are resident per SM (<=113 KB smem,
// 256 TMEM columns each) so one CTA's softmax overlaps the other's MMAs.
#include "pdllm_internal.h"
#include "ptx.cuh"

namespace pdllm {

namespace {

constexpr int kSoftmaxThreads = 128;
constexpr int kProducerThreads = 128;
constexpr int kAttnThreads = kSoftmaxThreads + kProducerThreads + 32;   // + the MMA warp
constexpr int kInvalidRow = INT32_MIN;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 between reference-max updates

struct AttnParams {
    const uint16_t *Q, *Kc, *Vc, *Kd, *Vd;
    const int32_t *ids, *keep;
    uint16_t *O;
    float *LSE, *O_part, *lse_part;
    int H_kv, N, Cp, K, Bk, L_s, S_pre, S_kv, rows_g;
    int n_splits, n_tiles;
    int64_t total_rows;    // B*H*L
    float c2;              // scale * log2(e)
};

enum { BAR_QFULL = 0, BAR_KFULL, BAR_VFULL, BAR_SREADY, BAR_PREADY, BAR_PVDONE, BAR_COUNT };

template <int D>
__global__ void __launch_bounds__(kAttnThreads, 2) attn_kernel(const AttnParams p) {
    constexpr int kPanels = D / 64;                 // 64-column (128-byte) panels per row
    constexpr int kChunksPerRow = D / 8;            // 16-byte chunks per row
    constexpr int kRowsPerInstr = 32 / kChunksPerRow;
    constexpr uint32_t kPanelBytes = 128 * 128;     // [128 rows][128 B]
    constexpr uint32_t kTileBytes = kPanels * kPanelBytes;
    constexpr uint32_t kTmemCols = 256;             // S/P: 128 columns, O: D columns
    constexpr uint32_t kOCol = 128;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base, sK = smem_base + kTileBytes, sV = smem_base + 2 * kTileBytes;

    __shared__ uint64_t bars[BAR_COUNT];
    __shared__ uint32_t tmem_slot;
    __shared__ int32_t s_ids[64];
    __shared__ int32_t s_table[128];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int mt = blockIdx.x, bg = blockIdx.y, split = blockIdx.z;
    const int t0 = (int)((int64_t)split * p.n_tiles / p.n_splits);
    const int t1 = (int)((int64_t)(split + 1) * p.n_tiles / p.n_splits);
    const int nt = t1 - t0;

    const uint32_t bar0 = smem_u32(&bars[0]);
    auto bar = [&](int i) { return bar0 + 8u * i; };

    if (tid == 0) {
        mbar_init(bar(BAR_QFULL), kProducerThreads);
        mbar_init(bar(BAR_KFULL), kProducerThreads);
        mbar_init(bar(BAR_VFULL), kProducerThreads);
        mbar_init(bar(BAR_SREADY), 1);
        mbar_init(bar(BAR_PREADY), kSoftmaxThreads);
        mbar_init(bar(BAR_PVDONE), 1);
        fence_mbar_init();
    }
    if (tid < p.K) s_ids[tid] = p.ids[(int64_t)bg * p.K + tid];
    if (warp == 8) {
        tmem_alloc(smem_u32(&tmem_slot), kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_slot;
    const uint32_t tS = tmem, tO = tmem + kOCol;

    if (warp >= 4 && warp < 8) {
        // =============================== producers: gather ===============================
        const int pt = tid - kSoftmaxThreads, pw = pt >> 5;
        const int rsub = lane / kChunksPerRow, c = lane % kChunksPerRow;
        const uint32_t dst_pc = (uint32_t)(c >> 3) * kPanelBytes;
        const uint16_t *Kc = p.Kc + (int64_t)bg * p.N * p.Cp * D, *Vc = p.Vc + (int64_t)bg * p.N * p.Cp * D;
        const uint16_t *Kd = p.Kd + (int64_t)bg * p.L_s * D, *Vd = p.Vd + (int64_t)bg * p.L_s * D;
        {   // Q tile: rows mt*128 .. +127 of the rows_g contiguous rows of this KV group
            const uint16_t *Qg = p.Q + (int64_t)bg * p.rows_g * D;
#pragma unroll 4
            for (int i = 0; i < kChunksPerRow; ++i) {
                const int r = pw * 32 + i * kRowsPerInstr + rsub;
                const int qr = mt * kTileM + r;
                const bool ok = qr < p.rows_g;
                cp_async16_zfill(sQ + dst_pc + sw128_off(r, c & 7), ok ? Qg + (int64_t)qr * D + c * 8 : Qg, ok ? 16u : 0u);
            }
            cp_async_commit();
            cp_async_wait<0>();
            fence_proxy_async_smem();
            mbar_arrive(bar(BAR_QFULL));
        }
        const int kv_end = min(p.S_kv, t1 * kTileN);
        for (int jj = 0; jj < nt; ++jj) {
            const int j = t0 + jj;
            // row table of this tile (a3): virtual row -> cache row (>= 0) / decode row (< 0)
            {
                const int vr = j * kTileN + pt;
                int idx = kInvalidRow;
                if (vr < kv_end) {
                    if (vr < p.S_pre) {
                        const int k = vr / p.Bk, t = vr - k * p.Bk;
                        const int n = s_ids[k];
                        const int slot = p.keep ? __ldg(p.keep + ((int64_t)bg * p.N + n) * p.Bk + t) : t;
                        idx = n * p.Cp + slot;
                    } else {
                        idx = -(vr - p.S_pre) - 1;
                    }
                }
                s_table[pt] = idx;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            const int n_valid = min(kTileN, kv_end - j * kTileN);
            const int n_mma = (n_valid + 15) & ~15;
            if (jj > 0) mbar_wait(bar(BAR_SREADY), (jj - 1) & 1);      // QK(j-1) done: K buffer free
#pragma unroll 4
            for (int i = 0; i < kChunksPerRow; ++i) {
                const int r = pw * 32 + i * kRowsPerInstr + rsub;
                if (r < n_mma) {
                    const int idx = s_table[r];
                    const bool ok = idx != kInvalidRow;
                    const uint16_t *src = idx >= 0 ? Kc + (int64_t)idx * D : Kd + (int64_t)(-idx - 1) * D;
                    cp_async16_zfill(sK + dst_pc + sw128_off(r, c & 7), ok ? src + c * 8 : Kc, ok ? 16u : 0u);
                }
            }
            cp_async_commit();
            if (jj > 0) mbar_wait(bar(BAR_PVDONE), (jj - 1) & 1);      // PV(j-1) done: V buffer free
#pragma unroll 4
            for (int i = 0; i < kChunksPerRow; ++i) {
                const int r = pw * 32 + i * kRowsPerInstr + rsub;
                if (r < n_mma) {
                    const int idx = s_table[r];
                    const bool ok = idx != kInvalidRow;
                    const uint16_t *src = idx >= 0 ? Vc + (int64_t)idx * D : Vd + (int64_t)(-idx - 1) * D;
                    cp_async16_zfill(sV + dst_pc + sw128_off(r, c & 7), ok ? src + c * 8 : Vc, ok ? 16u : 0u);
                }
            }
            cp_async_commit();
            cp_async_wait<1>();
            fence_proxy_async_smem();
            mbar_arrive(bar(BAR_KFULL));
            cp_async_wait<0>();
            fence_proxy_async_smem();
            mbar_arrive(bar(BAR_VFULL));
            asm volatile("bar.sync 1, 128;" ::: "memory");              // table may be rewritten
        }
    } else if (warp == 8) {
        // =============================== MMA issuer ===============================
        if (lane == 0) {
            const int kv_end = min(p.S_kv, t1 * kTileN);
            mbar_wait(bar(BAR_QFULL), 0);
            for (int jj = 0; jj < nt; ++jj) {
                const int j = t0 + jj;
                const int n_valid = min(kTileN, kv_end - j * kTileN);
                const uint32_t n_mma = (uint32_t)(n_valid + 15) & ~15u;
                mbar_wait(bar(BAR_KFULL), jj & 1);
                if (jj > 0) mbar_wait(bar(BAR_PVDONE), (jj - 1) & 1);  // S aliases P(j-1)
                tc_fence_after();
                const uint32_t idesc_qk = umma_idesc_bf16(kTileM, n_mma, 0, 0);
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t off = (uint32_t)(ks >> 2) * kPanelBytes + (uint32_t)(ks & 3) * 32u;
                    umma_ss(tS, umma_desc_sw128(sQ + off, 16, 1024), umma_desc_sw128(sK + off, 16, 1024), idesc_qk, ks > 0);
                }
                umma_commit(bar(BAR_SREADY));
                mbar_wait(bar(BAR_PREADY), jj & 1);
                mbar_wait(bar(BAR_VFULL), jj & 1);
                tc_fence_after();
                const uint32_t idesc_pv = umma_idesc_bf16(kTileM, D, 0, 1);
                const int ksteps = (int)(n_mma >> 4);
                for (int ks = 0; ks < ksteps; ++ks) {
                    // 16 kv rows per step: A = 8 TMEM columns of packed bf16 P, B = V rows (MN-major)
                    umma_ts(tO, tS + 8u * ks, umma_desc_sw128(sV + 2048u * ks, kPanelBytes, 1024), idesc_pv,
                            (jj > 0 || ks > 0) ? 1u : 0u);
                }
                umma_commit(bar(BAR_PVDONE));
            }
        }
        __syncwarp();
    } else {
        // =============================== softmax (thread = row) ===============================
        const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
        const int kv_end = min(p.S_kv, t1 * kTileN);
        float m_ref = -INFINITY, l = 0.f;
        for (int jj = 0; jj < nt; ++jj) {
            const int j = t0 + jj;
            const int n_valid = min(kTileN, kv_end - j * kTileN);
            const int n_mma = (n_valid + 15) & ~15;
            const int nchunks = (n_mma + 31) >> 5;
            mbar_wait(bar(BAR_SREADY), jj & 1);
            tc_fence_after();
            // pass 1: row max of the raw logits
            float tmax = -INFINITY;
            for (int ch = 0; ch < nchunks; ++ch) {
                uint32_t v[32];
                tmem_ld32(tS + lane_base + 32u * ch, v);
                tmem_wait_ld();
                if (n_valid == kTileN) {
#pragma unroll
                    for (int e = 0; e < 32; ++e) tmax = fmaxf(tmax, __uint_as_float(v[e]));
                } else {
#pragma unroll
                    for (int e = 0; e < 32; ++e)
                        if (ch * 32 + e < n_valid) tmax = fmaxf(tmax, __uint_as_float(v[e]));
                }
            }
            const float tm2 = tmax * p.c2;
            const bool need = tm2 > m_ref + kRescaleThreshold;          // always true on the first tile
            if (__any_sync(0xffffffffu, need)) {
                const float m_new = need ? tm2 : m_ref;
                const float f = need ? ex2_approx(m_ref - m_new) : 1.f;  // m_ref = -inf -> 0
                l *= f;
                if (jj > 0) {
#pragma unroll 1
                    for (int ch = 0; ch < D / 32; ++ch) {
                        uint32_t o[32];
                        tmem_ld32(tO + lane_base + 32u * ch, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
                        tmem_st32(tO + lane_base + 32u * ch, o);
                    }
                }
                m_ref = m_new;
            }
            // pass 2: P = 2^(c2*S - m_ref), packed bf16 into the first 64 columns of S
            for (int ch = 0; ch < nchunks; ++ch) {
                uint32_t v[32];
                tmem_ld32(tS + lane_base + 32u * ch, v);
                tmem_wait_ld();
                uint32_t w[16];
                float lsum = 0.f;
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    float p0 = ex2_approx(fmaf(__uint_as_float(v[e]), p.c2, -m_ref));
                    float p1 = ex2_approx(fmaf(__uint_as_float(v[e + 1]), p.c2, -m_ref));
                    if (n_valid != kTileN) {
                        if (ch * 32 + e >= n_valid) p0 = 0.f;
                        if (ch * 32 + e + 1 >= n_valid) p1 = 0.f;
                    }
                    lsum += p0 + p1;
                    w[e >> 1] = pack_bf16x2(p0, p1);
                }
                l += lsum;
                tmem_st16(tS + lane_base + 16u * ch, w);
            }
            tmem_wait_st();
            tc_fence_before();
            mbar_arrive(bar(BAR_PREADY));
        }
        // ------------------------------- epilogue -------------------------------
        mbar_wait(bar(BAR_PVDONE), (nt - 1) & 1);
        tc_fence_after();
        const int qr = mt * kTileM + tid;
        const bool row_ok = qr < p.rows_g;
        const int64_t grow = (int64_t)bg * p.rows_g + qr;
        const float inv = 1.f / l;
        const float lse = (m_ref + lg2_approx(l)) * 0.6931471805599453f;
        if (p.n_splits == 1) {
            if (row_ok) p.LSE[grow] = lse;
#pragma unroll 1
            for (int ch = 0; ch < D / 32; ++ch) {
                uint32_t o[32];
                tmem_ld32(tO + lane_base + 32u * ch, o);
                tmem_wait_ld();
                if (row_ok) {
                    uint4 *dst = reinterpret_cast<uint4 *>(p.O + grow * D + ch * 32);
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        uint4 u;
                        u.x = pack_bf16x2(__uint_as_float(o[q4 * 8 + 0]) * inv, __uint_as_float(o[q4 * 8 + 1]) * inv);
                        u.y = pack_bf16x2(__uint_as_float(o[q4 * 8 + 2]) * inv, __uint_as_float(o[q4 * 8 + 3]) * inv);
                        u.z = pack_bf16x2(__uint_as_float(o[q4 * 8 + 4]) * inv, __uint_as_float(o[q4 * 8 + 5]) * inv);
                        u.w = pack_bf16x2(__uint_as_float(o[q4 * 8 + 6]) * inv, __uint_as_float(o[q4 * 8 + 7]) * inv);
                        dst[q4] = u;
                    }
                }
            }
        } else {
            if (row_ok) p.lse_part[(int64_t)split * p.total_rows + grow] = lse;
#pragma unroll 1
            for (int ch = 0; ch < D / 32; ++ch) {
                uint32_t o[32];
                tmem_ld32(tO + lane_base + 32u * ch, o);
                tmem_wait_ld();
                if (row_ok) {
                    float4 *dst = reinterpret_cast<float4 *>(p.O_part + ((int64_t)split * p.total_rows + grow) * D + ch * 32);
#pragma unroll
                    for (int q4 = 0; q4 < 8; ++q4)
                        dst[q4] = make_float4(__uint_as_float(o[q4 * 4 + 0]) * inv, __uint_as_float(o[q4 * 4 + 1]) * inv,
                                              __uint_as_float(o[q4 * 4 + 2]) * inv, __uint_as_float(o[q4 * 4 + 3]) * inv);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, kTmemCols);
}

template <int D>
cudaError_t launch_attn_d(const AttnParams &p, int m_tiles, int BG, cudaStream_t st) {
    constexpr size_t smem = 1024 + 3 * (size_t)(D / 64) * 128 * 128;
    cudaError_t e = cudaFuncSetAttribute(attn_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)m_tiles, (unsigned)BG, (unsigned)p.n_splits);
    attn_kernel<D><<<grid, kAttnThreads, smem, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_attn(const Dims &s, const void *Q_dec, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                        const int32_t *keep, const void *K_dec, const void *V_dec, int n_splits, void *O, float *LSE,
                        float *O_part, float *lse_part, cudaStream_t st) {
    AttnParams p;
    p.Q = static_cast<const uint16_t *>(Q_dec);
    p.Kc = static_cast<const uint16_t *>(Kcache);
    p.Vc = static_cast<const uint16_t *>(Vcache);
    p.Kd = static_cast<const uint16_t *>(K_dec);
    p.Vd = static_cast<const uint16_t *>(V_dec);
    p.ids = chunk_ids;
    p.keep = keep;
    p.O = static_cast<uint16_t *>(O);
    p.LSE = LSE;
    p.O_part = O_part;
    p.lse_part = lse_part;
    p.H_kv = s.H_kv; p.N = s.N; p.Cp = s.Cp; p.K = s.K; p.Bk = s.Bk; p.L_s = s.L_s;
    p.S_pre = s.S_pre; p.S_kv = s.S_kv; p.rows_g = s.rows_g;
    p.n_tiles = (s.S_kv + kTileN - 1) / kTileN;
    p.n_splits = n_splits;
    p.total_rows = (int64_t)s.B * s.H * s.L;
    p.c2 = s.scale * 1.4426950408889634f;
    const int m_tiles = (s.rows_g + kTileM - 1) / kTileM;
    const int BG = s.B * s.H_kv;
    return s.d == 128 ? launch_attn_d<128>(p, m_tiles, BG, st) : launch_attn_d<64>(p, m_tiles, BG, st);
}

}  // namespace pdllm
