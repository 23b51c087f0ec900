// attn.cu -- a3 + a4 (+ the in-CTA half of a5): index-driven gather of the selected BOS+chunk KV rows and the
// Split-S partial attention kernel (R7-R11), tcgen05 / TMEM, sm_100a.
//
// One persistent CTA per SM takes work items from an atomic counter (costliest first, so CTAs that finish early take
// more).  An item belongs to one KV group (b, g) -- the G*L packed query rows that share K/V (GQA groups sit in the
// MMA M dimension, so K/V are read once per group) -- and one split of the virtual KV sequence
// [ K*Bk gathered cache rows || L_s decode-block rows ], cut at 128-row tile boundaries.
// Every item runs TWO streams -- two (S/P, O) accumulator sets in TMEM whose MMAs alternate on the tensor pipe (while
// the softmax warps work on one stream's S, the tensor pipe runs the other stream's P*V and next Q*K^T):
//   mode A (pair item)  : stream s owns query tile 2*pair+s; both streams walk the same KV tiles, so one K/V fetch
//                         feeds 256 query rows (halves the L2->SM traffic of 128-row CTAs);
//   mode B (single item): the group's odd last query tile; stream s walks KV tiles t0+s, t0+s+2, ... -- Split-S inside
//                         the CTA -- and the two (O, m, l) are merged by log-sum-exp in the epilogue, straight out of
//                         TMEM (no HBM round trip).
// Warp roles (416 threads): warps 0-7 softmax, two threads per query row (warps 0-3 columns 0-63, warps 4-7 columns
// 64-127 of every S tile), working through the tiles of both streams in the order they are produced; warps 8-11
// producers (16-byte cp.async row gather into 128B-swizzled panels; indices are prefetched a tile ahead so the gather
// runs at HBM speed; completion is signalled by cp.async.mbarrier.arrive.noinc), warp 12 issues every tcgen05.mma
// (one elected lane, converged warp so the descriptors stay in uniform registers).
// TMEM (512 columns): S_s at 128*s (P aliases it as packed bf16: column half h at 128*s + 64*h .. + 31), O_s at 256 + 128*s.
// Shared memory: two Q tiles and a ring of kStages K/V tile slots; a single item needs one Q tile only and lends the
// second Q buffer to the ring as a sixth slot (its two streams consume four tiles per step).  Ring state is a cursor
// plus one phase bit per slot, kept alike by the producers and the MMA warp; a slot is released by a tcgen05.commit
// after its last user (stream 1 in mode A).
#include <cuda.h>

#include "pdllm_internal.h"
#include "ptx.cuh"

namespace pdllm {

namespace {

constexpr int kSoftmaxThreads = 128;                      // per stream
constexpr int kProducerThreads = 128;
constexpr int kProducerWarp0 = 8;
constexpr int kMmaWarp0 = 12;
constexpr int kAttnThreads = 2 * kSoftmaxThreads + kProducerThreads + 128;     // 16 warps: whole warpgroups for setmaxnreg
// register budgets after the roles part ways (setmaxnreg; 256 * 176 + 128 * 104 + 128 * 56 = 65536)
constexpr int kSoftmaxRegs = 176, kProducerRegs = 104, kOtherRegs = 56;
constexpr int kInvalidRow = INT32_MIN;
static_assert(PDLLM_FOLD_MAX_N == 128, "four producer warps rank 32 chunks each; ids are kept as bytes");
constexpr int kFoldMaxN = PDLLM_FOLD_MAX_N;              // top-K is folded into the kernel up to this many chunks
constexpr float kRescaleThreshold = 8.0f;                 // log2 units: P stays <= 2^8 between reference-max updates

struct AttnParams {
    const uint16_t *Q, *Kc, *Vc, *Kd, *Vd;
    const int32_t *ids, *keep;
    uint16_t *O;
    float *LSE, *O_part, *lse_part;
    int N, Cp, K, Bk, L_s, S_pre, S_kv, rows_g;
    int n_splits, n_tiles;                                // KV tiles of the whole sequence
    int contig, T_pre;                                    // contiguous mode: prefix = [B*H_kv, S_pre, d], T_pre tiles of it
    int n_qt, n_pairs, n_single;                          // query tiles per group: n_qt = 2*n_pairs + n_single
    int n_pair_items, n_items;
    int32_t *work_counter;                                // zeroed before launch: next work item to hand out
    int64_t total_rows;                                   // B*H*L
    float c2;                                             // scale * log2(e)
    // a2 folded into the kernel (pdllm_step, N <= kFoldMaxN): the group's chunk ids are chosen here from the scores
    const float *fold_scores;                             // [B*H_kv, N] or, with fold_m_tiles > 1, [m_tiles, B*H_kv, N] partials
    int fold_m_tiles;
    int64_t fold_stride;                                  // B*H_kv*N
    int32_t *fold_ids_out;                                // [B*H_kv, K]
    float *fold_scores_out;                               // [B*H_kv, N], written when the scores come as partials
};

struct Item {
    int bg, q0, t0, nt, split;
    bool modeA;
};

// Valid virtual rows of KV tile `tile`.  Gather mode: one run of S_kv rows.  Contiguous mode (compact static cache,
// chunk prefill): the prefix and the decode rows are tiled separately -- T_pre prefix tiles, then the decode tiles,
// each part with its own ragged last tile (softmax attention does not care about the order of its keys).
__device__ __forceinline__ int tile_valid(const AttnParams &p, int tile) {
    if (!p.contig) return min(kTileN, p.S_kv - tile * kTileN);
    if (tile < p.T_pre) return min(kTileN, p.S_pre - tile * kTileN);
    return min(kTileN, p.L_s - (tile - p.T_pre) * kTileN);
}

__device__ __forceinline__ Item decode_item(const AttnParams &p, int i) {
    Item it;
    if (i < p.n_pair_items) {
        it.modeA = true;
        it.split = i % p.n_splits;
        const int rest = i / p.n_splits;
        it.q0 = 2 * (rest % p.n_pairs);
        it.bg = rest / p.n_pairs;
    } else {
        i -= p.n_pair_items;
        it.modeA = false;
        it.split = i % p.n_splits;
        it.bg = i / p.n_splits;
        it.q0 = p.n_qt - 1;
    }
    it.t0 = (int)((int64_t)it.split * p.n_tiles / p.n_splits);
    it.nt = (int)((int64_t)(it.split + 1) * p.n_tiles / p.n_splits) - it.t0;
    return it;
}


template <int D>
struct AttnCfg {
    static constexpr int kPanels = D / 64;                   // 64-column (128-byte) panels per row
    static constexpr uint32_t kPanelBytes = 128 * 128;       // [128 rows][128 B]
    static constexpr uint32_t kTileBytes = kPanels * kPanelBytes;
    static constexpr int kStages = 5;
    static constexpr size_t kSmem = 1024 + (size_t)(2 + kStages) * kTileBytes;
};

// barrier indices (kv_full / kv_free follow)
enum { BAR_ITEM0 = 0, BAR_ITEM1, BAR_ITEM2, BAR_ITEM3, BAR_QFULL, BAR_QFREE, BAR_SREADY0, BAR_SREADY1, BAR_PREADY0, BAR_PREADY1, BAR_OREADY0, BAR_OREADY1,
       BAR_OFREE0, BAR_OFREE1, BAR_KV };

// D[tmem] (+)= A[smem] * B[smem] with the descriptors given as (low word, constant high word)
__device__ __forceinline__ void umma_ss_lohi(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\tsetp.ne.b32 p, %5, 0;\n\t"
        "mov.b64 da, {%1, %3};\n\tmov.b64 db, {%2, %3};\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n\t}"
        ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate)
        : "memory");
}
// one 32-byte store (a whole sector) per lane; the address must be 32-byte aligned
__device__ __forceinline__ void st_global_v8(void *ptr, uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t e, uint32_t f,
                                             uint32_t g, uint32_t h) {
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(ptr), "r"(a), "r"(b), "r"(c), "r"(d), "r"(e),
                 "r"(f), "r"(g), "r"(h)
                 : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void umma_ts_lohi(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b64 db;\n\tsetp.ne.b32 p, %5, 0;\n\t"
        "mov.b64 db, {%2, %3};\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %4, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate)
        : "memory");
}

constexpr float kSoftLimit = 16384.f;                     // 2^14: a row sum beyond it raises the reference ahead of the next tile
constexpr float kHardLimit = 1.2676506e30f;               // 2^100: beyond it (or inf / NaN) the tile is redone carefully

template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

template <int D>
__global__ void __launch_bounds__(kAttnThreads, 1)
attn_kernel(const AttnParams p, const __grid_constant__ CUtensorMap tm_kp, const __grid_constant__ CUtensorMap tm_vp,
            const __grid_constant__ CUtensorMap tm_kd, const __grid_constant__ CUtensorMap tm_vd) {
    using Cfg = AttnCfg<D>;
    constexpr int ST = Cfg::kStages;
    constexpr int kChunksPerRow = D / 8;                  // 16-byte chunks per row
    constexpr int kRowsPerInstr = 32 / kChunksPerRow;     // rows covered by one warp-level cp.async
    constexpr uint32_t kTmemCols = 512;
    constexpr uint32_t kOCol = 256;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    auto sQ = [&](int s) { return smem_base + Cfg::kTileBytes * (uint32_t)s; };
    // ring slots 0..ST-1 follow the two Q buffers; slot ST is the SECOND Q BUFFER, lent to the ring by single items
    auto sKV = [&](int slot) { return smem_base + Cfg::kTileBytes * (uint32_t)(slot == ST ? 1 : 2 + slot); };

    __shared__ uint64_t bars[BAR_KV + 2 * (ST + 1)];
    __shared__ uint32_t tmem_slot;
    __shared__ int32_t s_items[4];                        // the CTA's next work items (ring, published by the producers)
    __shared__ uint8_t s_ids[64];                         // folded top-K: the current item's chunk ids (< kFoldMaxN <= 256)
    __shared__ uint32_t s_mask[4];                        // folded top-K: selection bitmask per producer warp
    __shared__ float s_ml[kSoftmaxThreads][3];            // single items: stream 1's (m_ref, l, O scale) for the in-CTA merge

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = smem_u32(&bars[0]);
    auto bar = [&](int i) { return bar0 + 8u * i; };
    auto kv_full = [&](int slot) { return bar0 + 8u * (BAR_KV + slot); };
    auto kv_free = [&](int slot) { return bar0 + 8u * (BAR_KV + ST + 1 + slot); };

    if (tid == 0) {
        for (int i = 0; i < 4; ++i) mbar_init(bar(BAR_ITEM0 + i), 1);
        mbar_init(bar(BAR_QFULL), kProducerThreads);
        mbar_init(bar(BAR_QFREE), 1);
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(BAR_SREADY0 + s), 1);
            mbar_init(bar(BAR_PREADY0 + s), kSoftmaxThreads);
            mbar_init(bar(BAR_OREADY0 + s), 1);
            mbar_init(bar(BAR_OFREE0 + s), kSoftmaxThreads);
        }
        for (int s = 0; s <= ST; ++s) {
            mbar_init(kv_full(s), kProducerThreads);
            mbar_init(kv_free(s), 1);
        }
        fence_mbar_init();
    }
    if (warp == kMmaWarp0) {
        tmem_alloc(smem_u32(&tmem_slot), kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_slot;

    if (warp >= kProducerWarp0 && warp < kMmaWarp0) {
        // =============================== producers: index-driven gather ===============================
        setmaxnreg_dec<kProducerRegs>();
        const int pt = tid - kProducerWarp0 * 32, pw = pt >> 5;
        const int rsub = lane / kChunksPerRow, c = lane % kChunksPerRow;
        const uint32_t dst_pc = (uint32_t)(c >> 3) * Cfg::kPanelBytes;
        // destination of (row pw*32 + i*RPI + rsub, chunk c) inside a tile: pw*32 is a multiple of 8, so the
        // 128B-swizzle term (c ^ row) & 7 is x7 ^ (i*RPI & 7) with x7 = (c & 7) ^ rsub
        const uint32_t dst_thread = dst_pc + (uint32_t)(pw * 32 + rsub) * 128u;
        const uint32_t x7 = (uint32_t)((c & 7) ^ rsub);
        // Completion is signalled by the hardware: cp.async.mbarrier.arrive.noinc makes the tile's "full" barrier
        // (count = 128 producer threads) track all cp.async this thread issued so far, so the producers never wait
        // for their own loads; the MMA warp crosses from the generic to the async proxy with a fence after its wait.
        auto publish = [&](uint32_t b) {
            asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(b) : "memory");
        };
        auto wait_free = [&](uint32_t b, uint32_t parity) { mbar_wait(b, parity); };
        // The cp.async of this thread for one tile: rows pw*32 + i*RPI + rsub (i < 16 at D = 128), chunk c.
        // destination offset of the i-th row inside a tile
        auto dst_of = [&](int i) {
            return dst_thread + (uint32_t)(i * kRowsPerInstr) * 128u + ((x7 ^ (uint32_t)((i * kRowsPerInstr) & 7)) << 4);
        };
        // generic: the row addresses live one per lane (lane = row inside the warp's 32), fetched by shuffle; 0 = zero-fill
        auto issue_rows = [&](uint32_t dst_tile, uint64_t my_addr, const void *dummy) {
            const uint32_t my_lo = (uint32_t)my_addr, my_hi = (uint32_t)(my_addr >> 32);
#pragma unroll
            for (int i = 0; i < kChunksPerRow; ++i) {
                const int rl = i * kRowsPerInstr + rsub;
                const uint32_t lo = __shfl_sync(0xffffffffu, my_lo, rl), hi = __shfl_sync(0xffffffffu, my_hi, rl);
                const uint64_t row_addr = ((uint64_t)hi << 32) | lo;
                const bool ok = row_addr != 0ull;
                const uint64_t src = ok ? row_addr + (uint64_t)(c * 16) : reinterpret_cast<uint64_t>(dummy);
                cp_async16_zfill(dst_tile + dst_of(i), reinterpret_cast<const void *>(src), ok ? 16u : 0u);
            }
        };
        // prefix-only tile: every row is a cache row; one 32-bit byte offset per row is shuffled and added to the
        // group's K (and V) base, which already carries this lane's chunk column
        auto issue_rows_pre = [&](uint32_t dst_k, uint32_t dst_v, uint32_t my_off, uint64_t kbase_c, uint64_t vbase_c,
                                  bool do_k, bool do_v) {
#pragma unroll
            for (int i = 0; i < kChunksPerRow; ++i) {
                const uint32_t off = __shfl_sync(0xffffffffu, my_off, i * kRowsPerInstr + rsub);
                if (do_k) cp_async16(dst_k + dst_of(i), reinterpret_cast<const void *>(kbase_c + off));
                if (do_v) cp_async16(dst_v + dst_of(i), reinterpret_cast<const void *>(vbase_c + off));
            }
        };
        // decode-only tile: consecutive rows of K_dec / V_dec, no indices at all
        auto issue_rows_dec = [&](uint32_t dst_k, uint32_t dst_v, uint64_t krow0_c, uint64_t vrow0_c, bool do_k, bool do_v) {
#pragma unroll
            for (int i = 0; i < kChunksPerRow; ++i) {
                const uint64_t o = (uint64_t)(i * kRowsPerInstr) * (uint64_t)(D * 2);
                if (do_k) cp_async16(dst_k + dst_of(i), reinterpret_cast<const void *>(krow0_c + o));
                if (do_v) cp_async16(dst_v + dst_of(i), reinterpret_cast<const void *>(vrow0_c + o));
            }
        };
        // Ring cursor and per-slot phase bits (continue across items).  Pair items use ST slots, single items ST + 1.
        // free_bits: parity the next use of a slot waits for on its "free" barrier (1 = passes on a fresh barrier).
        int cur = 0;
        uint32_t free_bits = (1u << (ST + 1)) - 1u;
        int n_done = 0;                                   // items finished by this CTA
        // Work items are handed out dynamically (costliest first: pair items, then single items), so CTAs that
        // finish early take more; thread 0 of the producers fetches, the other roles follow through s_items.
        // The kernel is launched as a programmatic dependent of its predecessor in the stream (top-K in pdllm_step): the
        // set-up above ran under that kernel's tail.  Nothing that kernel may have written is read before this wait; the
        // other roles read no global memory (their stores follow data that passed through here).
        asm volatile("griddepcontrol.wait;" ::: "memory");
        for (;; ++n_done) {
            if (pt == 0) {
                // the first item of a CTA is its block index (no round trip to the counter at kernel start)
                const int nxt = n_done == 0 ? (int)blockIdx.x : (int)gridDim.x + atomicAdd(p.work_counter, 1);
                s_items[n_done & 3] = nxt < p.n_items ? nxt : -1;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            const int ii = s_items[n_done & 3];
            if (pt == 0) mbar_arrive(bar(BAR_ITEM0 + (n_done & 3)));
            if (ii < 0) break;
            const Item it = decode_item(p, ii);
            const int64_t bg = it.bg;
            const uint16_t *Kc = p.Kc + bg * p.N * p.Cp * D, *Vc = p.Vc + bg * p.N * p.Cp * D;
            const uint16_t *Kd = p.Kd + bg * p.L_s * D, *Vd = p.Vd + bg * p.L_s * D;
            const int32_t *keep = p.keep ? p.keep + bg * p.N * p.Bk : nullptr;
            // the group's K <= 64 chunk ids live in two registers per lane (lane l: ids[l], ids[l + 32])
            int ids_lo = 0, ids_hi = 0;
            if (p.fold_scores) {
                // a2 (R6) inside the kernel: the producer warps rank the group's N <= 128 scores -- rank = number of
                // chunks ahead in the (score descending, index ascending) order; the K chunks of rank < K are the selection
                // -- and lists them in ascending index order.  Every item of the group arrives at the same list.
                // All four producer warps hold the scores (lane l: chunks l, l + 32, l + 64, l + 96); warp w ranks chunks
                // 32 w .. 32 w + 31 against all of them by shuffle broadcasts.
                float v[kFoldMaxN / 32];
#pragma unroll
                for (int r = 0; r < kFoldMaxN / 32; ++r) {
                    const int idx = r * 32 + lane;
                    float x = -INFINITY;
                    if (idx < p.N) {
                        x = 0.f;
                        for (int mt = 0; mt < p.fold_m_tiles; ++mt) x += p.fold_scores[mt * p.fold_stride + bg * p.N + idx];
                        if (p.fold_scores_out && pw == r && it.q0 == 0 && it.split == 0) p.fold_scores_out[bg * p.N + idx] = x;
                        if (x != x) x = -INFINITY;            // NaN counts as -inf
                    }
                    v[r] = x;
                }
                const int my_idx = pw * 32 + lane;
                const float mine = pw == 0 ? v[0] : pw == 1 ? v[1] : pw == 2 ? v[2] : v[3];
                int rank = 0;
                // (eight broadcasts in flight per trip of a rolled loop: the code stays small -- it runs cold once per launch)
#pragma unroll 1
                for (int r2 = 0; r2 * 32 < p.N; ++r2) {
                    const float vr = r2 == 0 ? v[0] : r2 == 1 ? v[1] : r2 == 2 ? v[2] : v[3];
#pragma unroll 1
                    for (int l0 = 0; l0 < 32; l0 += 8) {
#pragma unroll
                        for (int l2 = 0; l2 < 8; ++l2) {      // (chunks past N hold -inf behind every real index: never ahead)
                            const float o = __shfl_sync(0xffffffffu, vr, l0 + l2);
                            rank += (o > mine || (o == mine && r2 * 32 + l0 + l2 < my_idx)) ? 1 : 0;
                        }
                    }
                }
                const bool sel = my_idx < p.N && rank < p.K;
                const uint32_t sel_mask = __ballot_sync(0xffffffffu, sel);
                if (lane == 0) s_mask[pw] = sel_mask;
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (sel) {
                    int pos = __popc(sel_mask & ((1u << lane) - 1u));
#pragma unroll
                    for (int w2 = 0; w2 < 3; ++w2)
                        if (w2 < pw) pos += __popc(s_mask[w2]);
                    s_ids[pos] = (uint8_t)my_idx;
                    if (it.q0 == 0 && it.split == 0) p.fold_ids_out[bg * p.K + pos] = my_idx;
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
                ids_lo = lane < p.K ? s_ids[lane] : 0;
                ids_hi = lane + 32 < p.K ? s_ids[lane + 32] : 0;
            } else if (!p.contig) {
                ids_lo = lane < p.K ? __ldg(p.ids + bg * p.K + lane) : 0;
                ids_hi = lane + 32 < p.K ? __ldg(p.ids + bg * p.K + lane + 32) : 0;
            }
            // a3: virtual row -> cache row (>= 0) / decode row (< 0) / invalid; one row per producer thread.  The index
            // is kept as (base, raw) with raw = the keep-list entry still in flight: the sum is only formed when the
            // row is issued, one load later, so the global load latency hides behind the previous tile's cp.async.
            int nx_base = 0, nx_raw = 0;
            auto prefetch_index = [&](int tile) {
                const int vr = tile * kTileN + pt;
                const bool pre = vr < p.S_pre;
                const int k = pre ? vr / p.Bk : 0, t = vr - k * p.Bk;
                const int n_lo = __shfl_sync(0xffffffffu, ids_lo, k & 31), n_hi = __shfl_sync(0xffffffffu, ids_hi, k & 31);
                const int n = k < 32 ? n_lo : n_hi;
                nx_raw = 0;
                if (pre && keep) nx_raw = __ldg(keep + (int64_t)n * p.Bk + t);
                nx_base = pre ? n * p.Cp + (keep ? 0 : t) : (vr < p.S_kv ? -(vr - p.S_pre) - 1 : kInvalidRow);
            };
            // the item's Q tile(s), once the previous item's Q*K^T are all done
            auto load_q = [&]() {
                if (n_done > 0 && it.modeA) wait_free(bar(BAR_QFREE), (uint32_t)(n_done - 1) & 1u);
                // a pair item writes the second Q buffer: the last K/V tile a single item parked there must be released
                if (it.modeA) wait_free(kv_free(ST), (free_bits >> ST) & 1u);
                const uint16_t *Qg = p.Q + bg * p.rows_g * D;
                const int n_q = it.modeA ? 2 : 1;
                for (int s = 0; s < n_q; ++s) {
#pragma unroll
                    for (int i = 0; i < kChunksPerRow; ++i) {
                        const int r = pw * 32 + i * kRowsPerInstr + rsub;
                        const int qr = (it.q0 + s) * kTileM + r;
                        const bool ok = qr < p.rows_g;
                        const uint32_t sw = (x7 ^ (uint32_t)((i * kRowsPerInstr) & 7)) << 4;
                        cp_async16_zfill(sQ(s) + dst_thread + (uint32_t)(i * kRowsPerInstr) * 128u + sw,
                                         ok ? Qg + (int64_t)qr * D + c * 8 : Qg, ok ? 16u : 0u);
                    }
                }
                publish(bar(BAR_QFULL));
            };
            // this thread's row (pw*32 + lane) of a tile as a global byte address in K or V; 0 = beyond the sequence
            auto row_addr = [&](int idx, bool is_v) -> uint64_t {
                if (idx == kInvalidRow) return 0ull;
                const bool in_cache = idx >= 0;
                const int64_t row_off = in_cache ? (int64_t)idx * D : (int64_t)(-idx - 1) * D;
                const uint16_t *base = in_cache ? (is_v ? Vc : Kc) : (is_v ? Vd : Kd);
                return reinterpret_cast<uint64_t>(base + row_off);
            };
            const int n_slots = it.modeA ? ST : ST + 1;
            if (it.modeA && cur == ST) cur = 0;
            // a single item may drop a tile into the second Q buffer right away: the previous item's Q*K^T must be done
            if (!it.modeA && n_done > 0) wait_free(bar(BAR_QFREE), (uint32_t)(n_done - 1) & 1u);
            auto take_slot = [&]() {                      // next ring slot, once its previous tile has been released
                const int sl = cur;
                wait_free(kv_free(sl), (free_bits >> sl) & 1u);
                free_bits ^= 1u << sl;
                cur = cur + 1 == n_slots ? 0 : cur + 1;
                return sl;
            };
            // K and/or V rows of one tile into the given slots
            const uint64_t kbase_c = reinterpret_cast<uint64_t>(Kc + c * 8), vbase_c = reinterpret_cast<uint64_t>(Vc + c * 8);
            auto load_tile = [&](int tile, int my_idx, uint32_t dst_k, uint32_t dst_v, bool do_k, bool do_v) {
                const int r0 = tile * kTileN;
                if (r0 + kTileN <= p.S_pre) {
                    issue_rows_pre(dst_k, dst_v, (uint32_t)my_idx * (uint32_t)(D * 2), kbase_c, vbase_c, do_k, do_v);
                } else if (r0 >= p.S_pre && r0 + kTileN <= p.S_kv) {
                    const int64_t e0 = ((int64_t)(r0 - p.S_pre + pw * 32 + rsub)) * D + c * 8;
                    issue_rows_dec(dst_k, dst_v, reinterpret_cast<uint64_t>(Kd + e0), reinterpret_cast<uint64_t>(Vd + e0), do_k, do_v);
                } else {
                    if (do_k) issue_rows(dst_k, row_addr(my_idx, false), Kc);
                    if (do_v) issue_rows(dst_v, row_addr(my_idx, true), Vc);
                }
            };
            // contiguous mode: one thread fetches a whole 128-row tile with 3-D TMA (box 64 x 128 x 1 per 128-byte panel,
            // rows beyond the part's end read as zeros); the other producer threads only arrive on the tile's barrier
            auto tma_tile = [&](int tile, int slot, bool is_v) {
                const uint32_t b = kv_full(slot);
                if (pt == 0) {
                    mbar_arrive_expect_tx(b, Cfg::kTileBytes);
                    const bool pre = tile < p.T_pre;
                    const CUtensorMap *tm = pre ? (is_v ? &tm_vp : &tm_kp) : (is_v ? &tm_vd : &tm_kd);
                    const int row0 = (pre ? tile : tile - p.T_pre) * kTileN;
#pragma unroll
                    for (int pn = 0; pn < Cfg::kPanels; ++pn)
                        tma_load_3d(sKV(slot) + pn * Cfg::kPanelBytes, tm, pn * 64, row0, (int)bg, b);
                } else {
                    mbar_arrive(b);
                }
            };
            if (p.contig) {
                load_q();
                if (it.modeA) {
                    for (int jt = 0; jt < it.nt; ++jt) {
                        const int slot_k = take_slot(), slot_v = take_slot();
                        tma_tile(it.t0 + jt, slot_k, false);
                        tma_tile(it.t0 + jt, slot_v, true);
                    }
                } else {
                    // the MMA warp's consumption order: K(t0); { K(t0+i+1), V(t0+i) }; V(t0+nt-1)
                    tma_tile(it.t0, take_slot(), false);
                    for (int i = 0; i + 1 < it.nt; ++i) {
                        tma_tile(it.t0 + i + 1, take_slot(), false);
                        tma_tile(it.t0 + i, take_slot(), true);
                    }
                    tma_tile(it.t0 + it.nt - 1, take_slot(), true);
                }
            } else if (it.modeA) {
                // tile by tile, K and V together (one index computation, one cp.async group): loads 2*jt and 2*jt + 1
                prefetch_index(it.t0);
                load_q();                                 // Q first: its rows need no indices, the first tile's are in flight
                for (int jt = 0; jt < it.nt; ++jt) {
                    const int my_idx = nx_base + nx_raw;
                    if (jt + 1 < it.nt) prefetch_index(it.t0 + jt + 1);         // in flight while this tile is issued
                    const int slot_k = take_slot(), slot_v = take_slot();
                    load_tile(it.t0 + jt, my_idx, sKV(slot_k), sKV(slot_v), true, true);
                    publish(kv_full(slot_k));
                    publish(kv_full(slot_v));
                }
            } else {
                // one tile per load, in the MMA warp's consumption order K(t0); { K(t0+i+1), V(t0+i) }; V(t0+nt-1)
                // (each tile has a single user); a tile's indices are computed once and serve its K and its V load
                auto load_one = [&](int tile, int idx, bool is_v) {
                    const int slot = take_slot();
                    const uint32_t dst = sKV(slot);
                    load_tile(tile, idx, dst, dst, !is_v, is_v);
                    publish(kv_full(slot));
                };
                prefetch_index(it.t0);
                load_q();
                int idx_cur = nx_base + nx_raw;
                if (it.nt > 1) prefetch_index(it.t0 + 1);
                load_one(it.t0, idx_cur, false);
                for (int i = 0; i + 1 < it.nt; ++i) {
                    const int idx_new = nx_base + nx_raw;                       // tile t0 + i + 1
                    if (i + 2 < it.nt) prefetch_index(it.t0 + i + 2);
                    load_one(it.t0 + i + 1, idx_new, false);
                    load_one(it.t0 + i, idx_cur, true);
                    idx_cur = idx_new;
                }
                load_one(it.t0 + it.nt - 1, idx_cur, true);
            }
        }
    } else if (warp == kMmaWarp0) {
        // =============================== MMA issuer ===============================
        setmaxnreg_dec<kOtherRegs>();
        // One warp issues both streams' MMAs in the fixed order QK(0,0) QK(1,0) { PV(0,j) QK(0,j+1) PV(1,j) QK(1,j+1) }:
        // the in-order tensor pipe then keeps the two softmax streams in anti-phase (one stream's exponentials run
        // under the other stream's MMAs).  The warp stays converged (all lanes wait on the barriers); one elected
        // lane issues the tcgen05 instructions, so the descriptors stay in uniform registers.
        int cur = 0;                                      // ring cursor / phase bits, mirrored from the producers
        uint32_t full_bits = 0u;
        uint32_t n_pready[2] = {0, 0}, n_oready[2] = {0, 0};
        int n_done = 0;
        constexpr uint32_t idesc_pv = umma_idesc_bf16(kTileM, D, 0, 1);
        // descriptor words: K-major operands (Q, K): lbo 16, sbo 1024; MN-major V: lbo = panel stride, sbo 1024
        const uint32_t hi_k = (uint32_t)(umma_desc_sw128(0, 16, 1024) >> 32);
        const uint32_t hi_v = (uint32_t)(umma_desc_sw128(0, Cfg::kPanelBytes, 1024) >> 32);
        const uint32_t lo_k = (uint32_t)umma_desc_sw128(0, 16, 1024), lo_v = (uint32_t)umma_desc_sw128(0, Cfg::kPanelBytes, 1024);
        for (;; ++n_done) {
            mbar_wait(bar(BAR_ITEM0 + (n_done & 3)), (uint32_t)(n_done >> 2) & 1u);
            const int ii = s_items[n_done & 3];
            if (ii < 0) break;
            const Item it = decode_item(p, ii);
            const int n_s[2] = {it.modeA ? it.nt : (it.nt + 1) / 2, it.modeA ? it.nt : it.nt / 2};
            const int qk_total = n_s[0] + n_s[1];
            int qk_issued = 0;
            const int n_slots = it.modeA ? ST : ST + 1;
            if (it.modeA && cur == ST) cur = 0;
            int k_slot = 0, v_slot = 0;                   // pair items: the tile both streams are on
            auto next_load = [&]() {                      // wait for the next tile of the ring (loads are consumed in order)
                const int sl = cur;
                mbar_wait(kv_full(sl), (full_bits >> sl) & 1u);
                full_bits ^= 1u << sl;
                cur = cur + 1 == n_slots ? 0 : cur + 1;
                return sl;
            };
            auto tile_of = [&](int s, int j) { return it.modeA ? it.t0 + j : it.t0 + 2 * j + s; };
            auto n_mma_of = [&](int tile) { return (uint32_t)((tile_valid(p, tile) + 15) & ~15); };
            // the eight SS MMAs of S_s = Q_s K^T and their commits (call from the elected lane only)
            auto emit_qk = [&](int s, int tile, int slot, bool release) {
                const uint32_t a_lo = lo_k | ((sQ(it.modeA ? s : 0) & 0x3FFFFu) >> 4);
                const uint32_t b_lo = lo_k | ((sKV(slot) & 0x3FFFFu) >> 4);
                const uint32_t idesc = umma_idesc_bf16(kTileM, n_mma_of(tile), 0, 0);
                const uint32_t tS = tmem + 128u * s;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    // 16 columns = 32 bytes inside the 128-byte swizzle row; next panel every 4 steps
                    const uint32_t koff = (uint32_t)(((ks >> 2) * Cfg::kPanelBytes + (ks & 3) * 32u) >> 4);
                    umma_ss_lohi(tS, a_lo + koff, b_lo + koff, hi_k, idesc, ks > 0);
                }
                umma_commit(bar(BAR_SREADY0 + s));
                if (release) umma_commit(kv_free(slot));
                if (++qk_issued == qk_total) umma_commit(bar(BAR_QFREE));
            };
            mbar_wait(bar(BAR_QFULL), (uint32_t)n_done & 1u);
            for (int s = 0; s < 2; ++s) {                 // prologue: QK(0,0), QK(1,0)
                if (n_s[s] == 0) continue;
                const int tile = tile_of(s, 0);
                if (!it.modeA || s == 0) {
                    k_slot = next_load();
                    fence_proxy_async_smem();             // cp.async (generic proxy) wrote the tile
                }
                tc_fence_after();
                if (elect_one()) emit_qk(s, tile, k_slot, !it.modeA || s == 1);
                __syncwarp();
            }
            for (int j = 0; j < n_s[0]; ++j) {
                for (int s = 0; s < 2; ++s) {
                    if (j >= n_s[s]) continue;
                    const bool fresh = !it.modeA || s == 0, release = !it.modeA || s == 1;
                    const bool has_next = j + 1 < n_s[s], last_pv = !has_next;
                    const int tile = tile_of(s, j), tile_n = tile_of(s, j + 1);
                    // the loads this stream step needs have normally landed long ago: cross them into the async proxy
                    // BEFORE waiting for P, so that P*V and the next Q*K^T issue back to back once P is there
                    if (fresh) {
                        v_slot = next_load();
                        if (has_next) k_slot = next_load();
                        fence_proxy_async_smem();
                    }
                    mbar_wait(bar(BAR_PREADY0 + s), n_pready[s]++ & 1u);
                    if (j == 0 && n_oready[s] > 0) mbar_wait(bar(BAR_OFREE0 + s), (n_oready[s] - 1) & 1u);
                    tc_fence_after();
                    const int ksteps = (int)(n_mma_of(tile) >> 4);
                    if (elect_one()) {
                        // 16 kv rows per step: A = 8 TMEM columns of packed bf16 P, B = 16 V rows (MN-major, 2048 B)
                        const int slot = v_slot;
                        const uint32_t v_lo = lo_v | ((sKV(slot) & 0x3FFFFu) >> 4);
                        const uint32_t tS = tmem + 128u * s, tO = tmem + kOCol + 128u * s;
                        if (ksteps == kTileN / 16) {
#pragma unroll
                            for (int ks = 0; ks < kTileN / 16; ++ks)
                                umma_ts_lohi(tO, tS + 8u * ks, v_lo + 128u * ks, hi_v, idesc_pv, (j > 0 || ks > 0) ? 1u : 0u);
                        } else {
                            for (int ks = 0; ks < ksteps; ++ks)
                                umma_ts_lohi(tO, tS + 8u * ks, v_lo + 128u * ks, hi_v, idesc_pv, (j > 0 || ks > 0) ? 1u : 0u);
                        }
                        if (release) umma_commit(kv_free(slot));
                        if (last_pv) umma_commit(bar(BAR_OREADY0 + s));
                        if (has_next) emit_qk(s, tile_n, k_slot, release);
                    }
                    __syncwarp();
                    if (last_pv) ++n_oready[s];
                }
            }
        }
    } else if (warp < 2 * (kSoftmaxThreads / 32)) {
        // =============================== softmax (thread = query row, one 4-warp group per stream) ===============================
        // Warps 0-3 own stream 0, warps 4-7 stream 1 (a warp may only touch TMEM lanes 32*(warp%4)..+31, its 32 rows).
        // The in-order tensor pipe keeps the two groups in anti-phase: while one group works on its S tile the pipe runs
        // the other stream's P*V and next Q*K^T.  A thread holds its row's whole 128-column S tile in registers (the
        // group raises its register budget to kSoftmaxRegs) and keeps a REFERENCE max per row in log2 units: the
        // stream's first tile fixes it with a max pass, later tiles take ONE pass P = 2^(c2*S - m_ref).  P may outgrow 1:
        // a tile whose row sum exceeds 2^kSoftOctaves is still exact (bf16 and fp32 carry the exponent) and only raises
        // the reference, by whole octaves, ahead of the row's NEXT tile, when the O accumulator is at rest -- l and O are
        // multiplied by an exact power of two.  Only a sum beyond 2^kHardOctaves (a logit more than ~100 octaves above
        // the reference inside one tile) or a ragged tail tile goes through the careful pass: exact row max first.
        setmaxnreg_inc<kSoftmaxRegs>();
        const int s = warp >> 2;                          // stream
        const int row = tid & (kSoftmaxThreads - 1);
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + 128u * s + lane_base, tO = tmem + kOCol + 128u * s + lane_base;
        uint32_t n_sready = 0, n_oready = 0;
        int n_modeB = 0;
        for (int n_done = 0;; ++n_done) {
            mbar_wait(bar(BAR_ITEM0 + (n_done & 3)), (uint32_t)(n_done >> 2) & 1u);
            const int ii = s_items[n_done & 3];
            if (ii < 0) break;
            const Item it = decode_item(p, ii);
            const int n_mine = it.modeA ? it.nt : (s == 0 ? (it.nt + 1) / 2 : it.nt / 2);
            float m_ref = -INFINITY, l = 0.f, pend = 0.f;     // pend: octaves the reference is to be raised by
            // multiply this row's O accumulator by f (an exact power of two); O is at rest: PV(s, j-1) completed before
            // S(s, j) was committed
            auto scale_O = [&](float f) {
#pragma unroll 1
                for (int ch = 0; ch < D / 32; ++ch) {
                    uint32_t o[32];
                    tmem_ld32(tO + 32u * ch, o);
                    tmem_wait_ld();
#pragma unroll
                    for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
                    tmem_st32(tO + 32u * ch, o);
                }
            };
            // one 32-column block of a full tile: P = 2^(c2*S - m_ref) as packed bf16 and its row sum; packed f32x2
            // arithmetic (one FFMA2 / FADD2 per two columns), the exponentials on the MUFU pipe
            auto chunk_exp = [&](const uint32_t(&v)[32], uint32_t *w) {
                const uint64_t c2v = pack_f32x2(p.c2, p.c2), mv = pack_f32x2(-m_ref, -m_ref);
                uint64_t acc0 = 0ull, acc1 = 0ull;
#pragma unroll
                for (int e = 0; e < 32; e += 4) {
                    float x0, x1, x2, x3;
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e], v[e + 1]), c2v, mv), x0, x1);
                    unpack_f32x2(fma_f32x2(pack_u32x2(v[e + 2], v[e + 3]), c2v, mv), x2, x3);
                    const float p0 = ex2_approx(x0), p1 = ex2_approx(x1), p2 = ex2_approx(x2), p3 = ex2_approx(x3);
                    acc0 = add_f32x2(acc0, pack_f32x2(p0, p1));
                    acc1 = add_f32x2(acc1, pack_f32x2(p2, p3));
                    w[e >> 1] = pack_bf16x2(p0, p1);
                    w[(e >> 1) + 1] = pack_bf16x2(p2, p3);
                }
                float s0, s1, s2, s3;
                unpack_f32x2(acc0, s0, s1);
                unpack_f32x2(acc1, s2, s3);
                return (s0 + s1) + (s2 + s3);
            };
            for (int j = 0; j < n_mine; ++j) {
                const int tile = it.modeA ? it.t0 + j : it.t0 + 2 * j + s;
                const int n_valid = tile_valid(p, tile);
                mbar_wait(bar(BAR_SREADY0 + s), n_sready++ & 1u);
                tc_fence_after();
                if (__any_sync(0xffffffffu, pend > 0.f)) {
                    // the previous tile's row sum outgrew 2^kSoftOctaves: raise the reference now that O is at rest
                    const float f = ex2_approx(-pend);                // exact power of two (1 for rows that are fine)
                    l *= f;
                    scale_O(f);
                    tmem_wait_st();
                    m_ref += pend;
                    pend = 0.f;
                }
                bool careful = n_valid != kTileN;
                if (!careful) {
                    uint32_t va[32], vb[32], w[64];
                    tmem_ld32(tS, va);
                    tmem_ld32(tS + 32u, vb);
                    tmem_wait_ld();
                    if (j == 0) {
                        // first tile of the stream (full): its row max becomes the reference (one extra pass over S)
                        uint32_t vc[32], vd[32];
                        tmem_ld32(tS + 64u, vc);
                        tmem_ld32(tS + 96u, vd);
                        float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                        for (int e = 0; e < 32; ++e) mx[e & 3] = fmaxf(mx[e & 3], fmaxf(__uint_as_float(va[e]), __uint_as_float(vb[e])));
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 32; ++e) mx[e & 3] = fmaxf(mx[e & 3], fmaxf(__uint_as_float(vc[e]), __uint_as_float(vd[e])));
                        m_ref = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * p.c2;
                    }
                    // single pass against the reference, TMEM loads one block ahead of the arithmetic
                    uint32_t vc[32];
                    tmem_ld32(tS + 64u, vc);
                    float lsum = chunk_exp(va, w);
                    tmem_wait_ld();
                    tmem_ld32(tS + 96u, va);
                    lsum += chunk_exp(vb, w + 16);
                    tmem_wait_ld();
                    lsum += chunk_exp(vc, w + 32);
                    lsum += chunk_exp(va, w + 48);
                    careful = __any_sync(0xffffffffu, !(lsum <= kHardLimit));       // also catches inf / NaN sums
                    if (!careful) {
                        tmem_st32(tS, *reinterpret_cast<uint32_t(*)[32]>(w));
                        tmem_st32(tS + 32u, *reinterpret_cast<uint32_t(*)[32]>(w + 32));
                        l += lsum;
                        // 2^pend >= lsum >= the row's largest P: after the raise the same logits give P <= 1
                        if (lsum > kSoftLimit) pend = (float)(((__float_as_int(lsum) >> 23) & 0xff) - 126);
                    }
                }
                if (careful) {
                    // Ragged tail tile (possibly the stream's first) or a row sum beyond 2^kHardOctaves: row max over the
                    // valid columns -> reference (raised by whole octaves once it exists, so that l and O rescale exactly)
                    // -> masked exponentials -> P.  Nothing of this tile has been stored yet: S is read twice.
                    const int nblk = (n_valid + 31) >> 5;
                    float tmax = -INFINITY;
#pragma unroll 1
                    for (int b = 0; b < nblk; ++b) {
                        uint32_t v[32];
                        tmem_ld32(tS + 32u * b, v);
                        tmem_wait_ld();
                        float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                        for (int e = 0; e < 32; ++e)
                            if (b * 32 + e < n_valid) mx[e & 3] = fmaxf(mx[e & 3], __uint_as_float(v[e]));
                        tmax = fmaxf(tmax, fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])));
                    }
                    const float tm2 = tmax * p.c2;
                    if (j == 0) {
                        m_ref = tm2;                      // l = 0, O not started
                    } else {
                        const bool need = tm2 > m_ref + kRescaleThreshold;
                        if (__any_sync(0xffffffffu, need)) {
                            const float up = need ? ceilf(tm2 - m_ref) : 0.f;
                            const float f = ex2_approx(-up);
                            l *= f;
                            scale_O(f);
                            m_ref += up;
                        }
                    }
#pragma unroll 1
                    for (int b = 0; b < 4; ++b) {
                        uint32_t w[16];
#pragma unroll
                        for (int e = 0; e < 16; ++e) w[e] = 0u;
                        if (b < nblk) {
                            uint32_t v[32];
                            tmem_ld32(tS + 32u * b, v);
                            tmem_wait_ld();
                            float ls[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                            for (int e = 0; e < 32; e += 2) {
                                float p0 = ex2_approx(fmaf(__uint_as_float(v[e]), p.c2, -m_ref));
                                float p1 = ex2_approx(fmaf(__uint_as_float(v[e + 1]), p.c2, -m_ref));
                                if (b * 32 + e >= n_valid) p0 = 0.f;
                                if (b * 32 + e + 1 >= n_valid) p1 = 0.f;
                                ls[(e >> 1) & 3] += p0 + p1;
                                w[e >> 1] = pack_bf16x2(p0, p1);
                            }
                            l += (ls[0] + ls[1]) + (ls[2] + ls[3]);
                        }
                        // P block b (16 packed columns) must not overwrite S columns that are still to be read: block b of
                        // P lands on S columns 16b..16b+15 <= 32b, already consumed
                        tmem_st16(tS + 16u * b, w);
                    }
                }
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(bar(BAR_PREADY0 + s));
            }
            // ------------------------------- epilogue -------------------------------
            // Pair items: one output tile per stream.  Single items (a5 inside the CTA): both streams hold partial
            // results of the SAME rows; stream 1 publishes its (m, l), stream 0 merges both accumulators out of TMEM.
            if (pend > 0.f) {                             // a raise still owed: fold it into the statistics only (O is
                m_ref += pend;                            // normalised by l below, the common factor cancels) ...
                l *= ex2_approx(-pend);
            }
            const float o_fix = pend > 0.f ? ex2_approx(-pend) : 1.f;      // ... but keep O and l on one scale
            const int qt = it.modeA ? it.q0 + s : it.q0;
            const int qr = qt * kTileM + row;
            const bool row_ok = qr < p.rows_g;
            const int64_t grow = (int64_t)it.bg * p.rows_g + qr;
            if (n_mine > 0) {
                mbar_wait(bar(BAR_OREADY0 + s), n_oready++ & 1u);
                tc_fence_after();
            }
            float a_self = o_fix, a_other = 0.f, l_tot = l, m_tot = m_ref;
            const bool merge_other = !it.modeA && it.nt > 1;    // stream 1 had tiles (uniform per item)
            if (!it.modeA) {
                if (s == 1) {
                    // stream 0 has read the previous single item's values (named barrier 3: it arrives, we wait)
                    if (n_modeB > 0) asm volatile("bar.sync 3, 256;" ::: "memory");
                    s_ml[row][0] = m_ref;
                    s_ml[row][1] = l;
                    s_ml[row][2] = o_fix;
                }
                ++n_modeB;
                tc_fence_before();
                asm volatile("bar.sync 2, 256;" ::: "memory");
                tc_fence_after();
                if (s == 0) {
                    const float m1 = s_ml[row][0], l1 = s_ml[row][1], fix1 = s_ml[row][2];
                    asm volatile("bar.arrive 3, 256;" ::: "memory");
                    if (merge_other) {
                        m_tot = fmaxf(m_ref, m1);
                        const float e0 = ex2_approx(m_ref - m_tot), e1 = ex2_approx(m1 - m_tot);
                        l_tot = l * e0 + l1 * e1;
                        a_self = o_fix * e0;
                        a_other = fix1 * e1;
                    }
                }
            }
            if (it.modeA || s == 0) {
                const float inv = 1.f / l_tot;
                const float lse = (m_tot + lg2_approx(l_tot)) * 0.6931471805599453f;
                const float w_self = a_self * inv, w_other = a_other * inv;
                const uint32_t tO_other = tmem + kOCol + 128u + lane_base;    // stream 1's accumulator, same rows
                const bool o_align32 = (reinterpret_cast<uintptr_t>(p.O) & 31u) == 0;
                if (row_ok) {
                    if (p.n_splits == 1) p.LSE[grow] = lse;
                    else p.lse_part[(int64_t)it.split * p.total_rows + grow] = lse;
                }
#pragma unroll 1
                for (int ch = 0; ch < D / 32; ++ch) {
                    uint32_t o[32];
                    tmem_ld32(tO + 32u * ch, o);
                    tmem_wait_ld();
                    float f[32];
#pragma unroll
                    for (int e = 0; e < 32; ++e) f[e] = __uint_as_float(o[e]) * w_self;
                    if (merge_other) {
                        tmem_ld32(tO_other + 32u * ch, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 32; ++e) f[e] = fmaf(__uint_as_float(o[e]), w_other, f[e]);
                    }
                    if (ch == D / 32 - 1) {
                        // the accumulator(s) are in registers: hand them back before the last stores
                        tc_fence_before();
                        mbar_arrive(bar(BAR_OFREE0 + s));
                        if (merge_other) mbar_arrive(bar(BAR_OFREE1));      // stream 0 has drained stream 1's accumulator
                    }
                    if (row_ok) {
                        if (p.n_splits == 1) {
                            uint32_t u[16];
#pragma unroll
                            for (int e = 0; e < 16; ++e) u[e] = pack_bf16x2(f[2 * e], f[2 * e + 1]);
                            uint16_t *dst = p.O + grow * D + ch * 32;
                            if (o_align32) {              // whole 32-byte sectors per lane (rows are 2*D bytes apart)
                                st_global_v8(dst, u[0], u[1], u[2], u[3], u[4], u[5], u[6], u[7]);
                                st_global_v8(dst + 16, u[8], u[9], u[10], u[11], u[12], u[13], u[14], u[15]);
                            } else {
#pragma unroll
                                for (int q4 = 0; q4 < 4; ++q4)
                                    reinterpret_cast<uint4 *>(dst)[q4] = make_uint4(u[4 * q4], u[4 * q4 + 1], u[4 * q4 + 2], u[4 * q4 + 3]);
                            }
                        } else {
                            // whole 32-byte sectors per lane and store (rows are 4*D bytes apart; the workspace is 256-byte
                            // aligned): 16-byte stores would each write half a sector
                            float *dst = p.O_part + ((int64_t)it.split * p.total_rows + grow) * D + ch * 32;
#pragma unroll
                            for (int q8 = 0; q8 < 4; ++q8)
                                st_global_v8(dst + q8 * 8, __float_as_uint(f[q8 * 8 + 0]), __float_as_uint(f[q8 * 8 + 1]),
                                             __float_as_uint(f[q8 * 8 + 2]), __float_as_uint(f[q8 * 8 + 3]), __float_as_uint(f[q8 * 8 + 4]),
                                             __float_as_uint(f[q8 * 8 + 5]), __float_as_uint(f[q8 * 8 + 6]), __float_as_uint(f[q8 * 8 + 7]));
                        }
                    }
                }
            }
        }
    } else {
        setmaxnreg_dec<kOtherRegs>();                     // warps 13-15 of the MMA warp's group: nothing to do
    }
    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp0) tmem_dealloc(tmem, kTmemCols);
}

template <int D>
cudaError_t launch_attn_d(const AttnParams &p, const CUtensorMap (&tm)[4], cudaStream_t st) {
    using Cfg = AttnCfg<D>;
    cudaError_t e = cudaFuncSetAttribute(attn_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmem);
    if (e != cudaSuccess) return e;
    const int grid = p.n_items < device_num_sms() ? p.n_items : device_num_sms();
    // Programmatic dependent launch: the CTAs become resident as SMs fall free under the predecessor's tail (top-K, which
    // triggers at its start, in pdllm_step), set themselves up, and wait at the head of the producer role.  (Round 1
    // withdrew a first attempt after an invalid-address-space fault in long loops; this placement -- nothing read before
    // the wait, the trigger in top-K -- was soaked over 12,600 unsynchronised steps with S = 1..3.)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid, 1, 1);
    cfg.blockDim = dim3(kAttnThreads, 1, 1);
    cfg.dynamicSmemBytes = Cfg::kSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, attn_kernel<D>, p, tm[0], tm[1], tm[2], tm[3]);
}

void fill_common(AttnParams &p, const Dims &s, int n_splits) {
    p.N = s.N; p.Cp = s.Cp; p.K = s.K; p.Bk = s.Bk; p.L_s = s.L_s;
    p.S_pre = s.S_pre; p.S_kv = s.S_kv; p.rows_g = s.rows_g;
    p.contig = s.contig;
    p.T_pre = (s.S_pre + kTileN - 1) / kTileN;
    p.n_tiles = kv_tiles(s);
    p.n_splits = n_splits;
    p.n_qt = (s.rows_g + kTileM - 1) / kTileM;
    p.n_pairs = p.n_qt / 2;
    p.n_single = p.n_qt & 1;
    const int BG = s.B * s.H_kv;
    p.n_pair_items = BG * p.n_pairs * n_splits;
    p.n_items = p.n_pair_items + BG * p.n_single * n_splits;
    p.total_rows = (int64_t)s.B * s.H * s.L;
    p.c2 = s.scale * 1.4426950408889634f;
}

}  // namespace

bool attn_can_fold_topk(const Dims &d) { return !d.contig && d.N <= kFoldMaxN; }

int kv_tiles(const Dims &d) {
    if (!d.contig) return (d.S_kv + kTileN - 1) / kTileN;
    return (d.S_pre + kTileN - 1) / kTileN + (d.L_s + kTileN - 1) / kTileN;
}

cudaError_t launch_attn(const Dims &s, const void *Q_dec, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                        const int32_t *keep, const void *K_dec, const void *V_dec, int n_splits, void *O, float *LSE,
                        float *O_part, float *lse_part, int32_t *work_counter, cudaStream_t st, const AttnFold *fold) {
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
    p.work_counter = work_counter;
    fill_common(p, s, n_splits);
    p.fold_scores = nullptr;
    p.fold_m_tiles = 1;
    p.fold_stride = (int64_t)s.B * s.H_kv * s.N;
    p.fold_ids_out = nullptr;
    p.fold_scores_out = nullptr;
    if (fold) {
        p.fold_scores = fold->partials ? fold->partials : fold->scores;
        p.fold_m_tiles = fold->partials ? (s.G * s.L_q + kTileM - 1) / kTileM : 1;
        p.fold_ids_out = fold->ids_out;
        p.fold_scores_out = fold->partials ? fold->scores_out : nullptr;
    }
    CUtensorMap tm[4];
    if (s.contig) {
        // contiguous mode: Kcache / Vcache are [B*H_kv, S_pre, d] (compact static cache, or a prefill sequence's K / V);
        // K_dec / V_dec [B*H_kv, L_s, d] may be absent (L_s == 0)
        const uint64_t BG = (uint64_t)s.B * s.H_kv;
        const bool dec = s.L_s > 0;
        if (!make_rows_tmap3d(&tm[0], Kcache, BG, (uint64_t)s.S_pre, s.d, kTileN) ||
            !make_rows_tmap3d(&tm[1], Vcache, BG, (uint64_t)s.S_pre, s.d, kTileN) ||
            !make_rows_tmap3d(&tm[2], dec ? K_dec : Kcache, BG, (uint64_t)(dec ? s.L_s : s.S_pre), s.d, kTileN) ||
            !make_rows_tmap3d(&tm[3], dec ? V_dec : Vcache, BG, (uint64_t)(dec ? s.L_s : s.S_pre), s.d, kTileN))
            return cudaErrorInvalidValue;
    } else {
        memset(tm, 0, sizeof(tm));
    }
    return s.d == 128 ? launch_attn_d<128>(p, tm, st) : launch_attn_d<64>(p, tm, st);
}

}  // namespace pdllm
