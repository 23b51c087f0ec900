// pdllm_api.cu -- the C-ABI entry points of include/pdllm.h: host-side validation, shape
// resolution, split-count choice, workspace carving and the enqueue sequences.  No arithmetic
// of the method happens on the host.
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>

#include "pdllm_internal.h"

namespace pdllm {

// SM count of the CURRENT device (an immutable hardware fact, remembered per device index after the first query).
int device_num_sms() {
    constexpr int kMaxDev = 64;
    static std::atomic<int> cache[kMaxDev];
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (dev >= 0 && dev < kMaxDev && (n = cache[dev].load(std::memory_order_relaxed)) > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
    if (dev >= 0 && dev < kMaxDev) cache[dev].store(n, std::memory_order_relaxed);
    return n;
}

namespace {

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int resolve(const pdllm_shape *sh, bool has_keep, Dims *out) {
    if (!sh) return PDLLM_ERR_NULL;
    if (sh->B < 1 || sh->H < 1 || sh->H_kv < 1 || sh->H % sh->H_kv != 0) return PDLLM_ERR_SHAPE;
    if (sh->d != 64 && sh->d != 128) return PDLLM_ERR_SHAPE;
    if (sh->N < 1 || sh->N > 4096 || sh->C < 1) return PDLLM_ERR_SHAPE;
    if (sh->K < 1 || sh->K > sh->N || sh->K > 64) return PDLLM_ERR_SHAPE;
    if (sh->Bk < 1 || sh->Bk > sh->C + 1) return PDLLM_ERR_SHAPE;
    if (!has_keep && sh->Bk != sh->C + 1) return PDLLM_ERR_SHAPE;
    if (sh->L_q < 1 || sh->L < 1 || sh->L_s < 1) return PDLLM_ERR_SHAPE;
    const int64_t cache_rows = (int64_t)sh->B * sh->H_kv * sh->N * (sh->C + 1);
    if (cache_rows >= (1ll << 31)) return PDLLM_ERR_SHAPE;
    if ((int64_t)sh->K * sh->Bk + sh->L_s >= (1ll << 30)) return PDLLM_ERR_SHAPE;
    // one KV group's cache is addressed with 32-bit byte offsets by the gather (attn.cu)
    if ((int64_t)sh->N * (sh->C + 1) * sh->d * 2 >= (1ll << 32)) return PDLLM_ERR_SHAPE;
    if ((int64_t)sh->B * sh->H_kv > 65535) return PDLLM_ERR_SHAPE;
    Dims d;
    d.B = sh->B; d.H = sh->H; d.H_kv = sh->H_kv; d.G = sh->H / sh->H_kv; d.d = sh->d;
    d.N = sh->N; d.C = sh->C; d.Cp = sh->C + 1; d.K = sh->K; d.Bk = sh->Bk;
    d.L_q = sh->L_q; d.L = sh->L; d.L_s = sh->L_s;
    d.S_pre = sh->K * sh->Bk; d.S_kv = d.S_pre + sh->L_s;
    d.rows_g = d.G * sh->L;
    d.scale = sh->scale > 0.f ? sh->scale : 1.0f / std::sqrt((float)sh->d);
    d.contig = 0;
    *out = d;
    return PDLLM_OK;
}

// a6: the attention kernel runs one persistent CTA per SM over work items (attn.cu): per KV group and split,
// floor(n_qt/2) pair items (both streams walk the split's tiles: ceil(T/S) steps) and n_qt%2 single items (the two
// streams share the tiles: half the steps); item i goes to CTA i mod num_sms, pair items first.  The model below
// scores a split count by the busiest CTA's steps (+ a fixed per-item cost) and, when S > 1, the combine kernel's
// launch and its 2*S*rows*d*4 bytes of partial traffic; the cheapest S wins (ties -> smaller S).
double split_cost_us(const Dims &d, int S, int sms) {
    const int T = kv_tiles(d), BG = d.B * d.H_kv;
    const int n_qt = (d.rows_g + kTileM - 1) / kTileM, n_pairs = n_qt / 2, n_single = n_qt & 1;
    // constants fitted to the measured split sweeps (profiles/r2_splitsweep_dream16k.md, C2-C4, the Fig. 5(b) shapes) and checked
    // on the configs[4] sweep: partials that stay in L2 (write + read <= 64 MB) move at ~8 TB/s, larger ones through HBM
    // against the attention's own traffic at ~3 TB/s
    const double kStepUs = 1.3, kItemSteps = 0.5, kLaunchUs = 1.0, kL2BytesPerUs = 8.0e6, kHbmBytesPerUs = 3.0e6, kL2Traffic = 64.0e6;
    const int64_t na = (int64_t)BG * n_pairs * S, nb = (int64_t)BG * n_single * S;
    const double ca = (T + S - 1) / S + kItemSteps, cb = ((T + S - 1) / S + 1) / 2 + kItemSteps;
    // CTA c receives items c, c + sms, ...: those below na cost ca, the rest cb
    double worst = 0.0;
    for (int c = 0; c < sms; ++c) {
        const int64_t total = (na + nb > c) ? (na + nb - c - 1) / sms + 1 : 0;
        const int64_t a = (na > c) ? (na - c - 1) / sms + 1 : 0;
        const double load = a * ca + (total - a) * cb;
        if (load > worst) worst = load;
    }
    double us = worst * kStepUs;
    if (S > 1) {
        const double traffic = 2.0 * S * (double)d.B * d.H * d.L * d.d * 4.0;
        us += kLaunchUs + traffic / (traffic <= kL2Traffic ? kL2BytesPerUs : kHbmBytesPerUs);
    }
    return us;
}

int auto_splits(const Dims &d, int num_sms) {
    const int sms = num_sms > 0 ? num_sms : device_num_sms();
    const int T = kv_tiles(d);
    const int Smax = T < 64 ? T : 64;
    int best = 1;
    double best_us = split_cost_us(d, 1, sms);
    for (int S = 2; S <= Smax; ++S) {
        const double us = split_cost_us(d, S, sms);
        if (us < best_us * 0.97) {      // a split must pay for itself by a clear margin
            best_us = us;
            best = S;
        }
    }
    return best;
}

int effective_splits(const Dims &d, int n_splits, int num_sms) {
    int S = n_splits == 0 ? auto_splits(d, num_sms) : n_splits;
    const int T = kv_tiles(d);
    return S > T ? T : S;       // no empty split (R10)
}

// scratch of the attention: 256 bytes for the work-item counter of the persistent kernel (always), then, for S > 1,
// the fp32 partials O_part [S, rows, d] and lse_part [S, rows]
constexpr size_t kCounterBytes = 256;
// (pdllm_step only) per-M-tile chunk-score partials when G*L_q > 128: summed in a fixed order by the top-K kernel
size_t score_partial_bytes(const Dims &d) {
    const size_t m_tiles = ((size_t)d.G * d.L_q + kTileM - 1) / kTileM;
    return m_tiles > 1 ? align_up(m_tiles * d.B * d.H_kv * d.N * sizeof(float), 256) : 0;
}
size_t partials_bytes(const Dims &d, int S) {
    if (S <= 1) return 0;
    const size_t rows = (size_t)d.B * d.H * d.L;
    return align_up((size_t)S * rows * d.d * sizeof(float), 256) + align_up((size_t)S * rows * sizeof(float), 256);
}
size_t workspace_for(const Dims &d, int S) { return kCounterBytes + partials_bytes(d, S) + score_partial_bytes(d); }

struct HostScratch {
    size_t q, kd, vd, scores, ids, o, lse, ws, total;
};
HostScratch host_scratch(const Dims &d, int S) {
    HostScratch h;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes, 256); return o; };
    h.q = take((size_t)d.B * d.H * d.L * d.d * 2);
    h.kd = take((size_t)d.B * d.H_kv * d.L_s * d.d * 2);
    h.vd = take((size_t)d.B * d.H_kv * d.L_s * d.d * 2);
    h.scores = take((size_t)d.B * d.H_kv * d.N * 4);
    h.ids = take((size_t)d.B * d.H_kv * d.K * 4);
    h.o = take((size_t)d.B * d.H * d.L * d.d * 2);
    h.lse = take((size_t)d.B * d.H * d.L * 4);
    h.ws = off;
    off += workspace_for(d, S);
    h.total = off;
    return h;
}

int cuda_rc(cudaError_t e) { return e == cudaSuccess ? PDLLM_OK : PDLLM_ERR_CUDA; }

// PDLLM_DEBUG_VALIDATE=1 (include/pdllm.h, "DEBUG SWITCH"): check the index lists on the device, synchronise, report.
bool debug_validate_on() {
    const char *e = std::getenv("PDLLM_DEBUG_VALIDATE");
    return e && e[0] != '\0' && std::strcmp(e, "0") != 0;
}
int debug_validate(const Dims &d, const int32_t *chunk_ids, const int32_t *keep, cudaStream_t st) {
    if (!debug_validate_on() || (!chunk_ids && !keep)) return PDLLM_OK;
    int32_t *flag = nullptr, h = 0;
    if (cudaMalloc(&flag, sizeof(int32_t)) != cudaSuccess) return PDLLM_ERR_CUDA;
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int32_t), st);
    if (e == cudaSuccess) e = launch_validate(d, chunk_ids, keep, flag, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, flag, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(flag);
    if (e != cudaSuccess) return PDLLM_ERR_CUDA;
    return h ? PDLLM_ERR_DATA : PDLLM_OK;
}

}  // namespace
}  // namespace pdllm

using namespace pdllm;

extern "C" {

int pdllm_version(void) { return 200; }

const char *pdllm_strerror(int status) {
    switch (status) {
        case PDLLM_OK: return "ok";
        case PDLLM_ERR_NULL: return "a required pointer is NULL";
        case PDLLM_ERR_ALIGN: return "a device pointer or stride is not 16-byte aligned";
        case PDLLM_ERR_SHAPE: return "a shape field is out of range";
        case PDLLM_ERR_WORKSPACE: return "workspace too small";
        case PDLLM_ERR_UNSUPPORTED: return "unsupported request";
        case PDLLM_ERR_CUDA: return "CUDA call or launch failed";
        case PDLLM_ERR_DATA: return "PDLLM_DEBUG_VALIDATE: a chunk id or token-keep list on the device is malformed";
        case PDLLM_ERR_SCRATCH_LIMIT: return "pdllm_sparse_attn_noalloc: the request needs more scratch than PDLLM_NOALLOC_SCRATCH_BYTES";
        default: return "unknown pdllm status";
    }
}

int32_t pdllm_auto_splits(const pdllm_shape *shape, int32_t num_sms) {
    Dims d;
    if (resolve(shape, shape && shape->Bk != shape->C + 1, &d) != PDLLM_OK) return 1;
    return effective_splits(d, 0, num_sms);
}

size_t pdllm_workspace_bytes(const pdllm_shape *shape, int32_t n_splits, int32_t num_sms) {
    Dims d;
    if (n_splits < 0 || resolve(shape, shape && shape->Bk != shape->C + 1, &d) != PDLLM_OK) return 0;
    return workspace_for(d, effective_splits(d, n_splits, num_sms));
}

size_t pdllm_step_host_scratch_bytes(const pdllm_shape *shape, int32_t n_splits, int32_t num_sms) {
    Dims d;
    if (n_splits < 0 || resolve(shape, shape && shape->Bk != shape->C + 1, &d) != PDLLM_OK) return 0;
    return host_scratch(d, effective_splits(d, n_splits, num_sms)).total;
}

int pdllm_score_chunks(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                       const void *Kcache, float *scores, pdllm_stream_t stream) {
    if (!shape || !Q || !Kcache || !scores) return PDLLM_ERR_NULL;
    Dims d;
    // scoring never reads the keep list (R3): Bk is not constrained here
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (int rc = resolve(&sh, false, &d)) return rc;
    if (!aligned16(Q) || !aligned16(Kcache) || !aligned16(scores)) return PDLLM_ERR_ALIGN;
    if ((q_batch_stride & 7) || (q_head_stride & 7) || q_head_stride < (int64_t)d.L_q * d.d) return PDLLM_ERR_ALIGN;
    return cuda_rc(launch_score(d, Q, q_batch_stride, q_head_stride, Kcache, scores, nullptr, nullptr, static_cast<cudaStream_t>(stream)));
}

int pdllm_select_topk(const pdllm_shape *shape, const float *scores, int32_t *chunk_ids, pdllm_stream_t stream) {
    if (!shape || !scores || !chunk_ids) return PDLLM_ERR_NULL;
    Dims d;
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (int rc = resolve(&sh, false, &d)) return rc;
    return cuda_rc(launch_topk(d, scores, chunk_ids, static_cast<cudaStream_t>(stream)));
}

int pdllm_gather_idx(const pdllm_shape *shape, const int32_t *chunk_ids, const int32_t *token_keep_idx,
                     int32_t *gather_idx, pdllm_stream_t stream) {
    if (!shape || !chunk_ids || !gather_idx) return PDLLM_ERR_NULL;
    Dims d;
    if (int rc = resolve(shape, token_keep_idx != nullptr, &d)) return rc;
    if (int rc = debug_validate(d, chunk_ids, token_keep_idx, static_cast<cudaStream_t>(stream))) return rc;
    return cuda_rc(launch_gather_idx(d, chunk_ids, token_keep_idx, gather_idx, static_cast<cudaStream_t>(stream)));
}

int pdllm_lse_combine(const float *O_part, const float *lse_part, int32_t S, int64_t rows, int32_t d, void *O, float *LSE,
                      pdllm_stream_t stream) {
    if (!O_part || !lse_part || !O || !LSE) return PDLLM_ERR_NULL;
    if (S < 1 || rows < 1 || (d != 64 && d != 128)) return PDLLM_ERR_SHAPE;
    if (!aligned16(O_part) || !aligned16(O)) return PDLLM_ERR_ALIGN;
    return cuda_rc(launch_combine(O_part, lse_part, S, rows, d, O, LSE, static_cast<cudaStream_t>(stream)));
}

namespace {

// PDLLM_NO_FOLD=1 keeps a2 a kernel of its own in pdllm_step (A/B switch; read once)
bool no_fold() {
    static const bool v = [] { const char *e = getenv("PDLLM_NO_FOLD"); return e && e[0] == '1'; }();
    return v;
}

int record(void *ev, cudaStream_t st) {
    if (!ev) return PDLLM_OK;
    return cuda_rc(cudaEventRecord(static_cast<cudaEvent_t>(ev), st));
}

// a3 + a4 + a5 on validated arguments; ev_mid / ev_end (may be NULL) are recorded after a4 / a5.
int attn_impl(const Dims &d, const void *Q_dec, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
              const int32_t *token_keep_idx, const void *K_dec, const void *V_dec, int S, void *O, float *LSE,
              int32_t *gather_idx_out, void *workspace, bool counter_zeroed, void *ev_mid, void *ev_end, cudaStream_t st,
              const AttnFold *fold = nullptr) {
    int32_t *counter = static_cast<int32_t *>(workspace);
    if (!counter_zeroed)
        if (int rc = cuda_rc(cudaMemsetAsync(counter, 0, sizeof(int32_t), st))) return rc;
    if (gather_idx_out)
        if (int rc = cuda_rc(launch_gather_idx(d, chunk_ids, token_keep_idx, gather_idx_out, st))) return rc;
    const size_t rows = (size_t)d.B * d.H * d.L;
    float *O_part = nullptr, *lse_part = nullptr;
    if (S > 1) {
        O_part = reinterpret_cast<float *>(static_cast<char *>(workspace) + kCounterBytes);
        lse_part = reinterpret_cast<float *>(static_cast<char *>(workspace) + kCounterBytes +
                                             align_up((size_t)S * rows * d.d * sizeof(float), 256));
    }
    if (int rc = cuda_rc(launch_attn(d, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, S, O, LSE, O_part,
                                     lse_part, counter, st, fold)))
        return rc;
    if (int rc = record(ev_mid, st)) return rc;
    if (S > 1)
        if (int rc = cuda_rc(launch_combine(O_part, lse_part, S, (int64_t)rows, d.d, O, LSE, st))) return rc;
    return record(ev_end, st);
}

int attn_validate(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
                  const int32_t *chunk_ids, const int32_t *token_keep_idx, const void *K_dec, const void *V_dec,
                  int32_t n_splits, void *O, float *LSE, void *workspace, size_t workspace_bytes, Dims *d, int *S) {
    if (!shape || !Q_dec || !Kcache || !Vcache || !chunk_ids || !K_dec || !V_dec || !O || !LSE) return PDLLM_ERR_NULL;
    if (n_splits < 0) return PDLLM_ERR_SHAPE;
    if (int rc = resolve(shape, token_keep_idx != nullptr, d)) return rc;
    if (!aligned16(Q_dec) || !aligned16(Kcache) || !aligned16(Vcache) || !aligned16(K_dec) || !aligned16(V_dec) ||
        !aligned16(O) || !aligned16(workspace))
        return PDLLM_ERR_ALIGN;
    *S = effective_splits(*d, n_splits, device_num_sms());
    if (!workspace) return PDLLM_ERR_WORKSPACE;
    // n_splits == 0 leaves the count to the library: should the caller have sized the workspace for another SM count
    // (pdllm_workspace_bytes with a num_sms that is not this device's), the largest count that fits is taken
    if (n_splits == 0)
        while (*S > 1 && workspace_bytes < workspace_for(*d, *S)) --*S;
    if (workspace_bytes < workspace_for(*d, *S)) return PDLLM_ERR_WORKSPACE;
    return PDLLM_OK;
}

}  // namespace

int pdllm_sparse_attn(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
                      const int32_t *chunk_ids, const int32_t *token_keep_idx, const void *K_dec, const void *V_dec,
                      int32_t n_splits, void *O, float *LSE, int32_t *gather_idx_out, void *workspace,
                      size_t workspace_bytes, pdllm_stream_t stream) {
    Dims d;
    int S = 1;
    if (int rc = attn_validate(shape, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, n_splits, O, LSE,
                               workspace, workspace_bytes, &d, &S))
        return rc;
    if (int rc = debug_validate(d, chunk_ids, token_keep_idx, static_cast<cudaStream_t>(stream))) return rc;
    return attn_impl(d, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, S, O, LSE, gather_idx_out,
                     workspace, false, nullptr, nullptr, static_cast<cudaStream_t>(stream));
}

// ---- the static-selection fast path and the chunk prefill: attention over contiguous K/V (TMA tiles)
namespace {

int resolve_dense(const pdllm_dense_shape *sh, Dims *out) {
    if (!sh) return PDLLM_ERR_NULL;
    if (sh->B < 1 || sh->H < 1 || sh->H_kv < 1 || sh->H % sh->H_kv != 0) return PDLLM_ERR_SHAPE;
    if (sh->d != 64 && sh->d != 128) return PDLLM_ERR_SHAPE;
    if (sh->S_pre < 1 || sh->L < 1 || sh->L_s < 0) return PDLLM_ERR_SHAPE;
    if ((int64_t)sh->S_pre + sh->L_s >= (1ll << 30) || (int64_t)sh->B * sh->H_kv > 65535) return PDLLM_ERR_SHAPE;
    Dims d;
    memset(&d, 0, sizeof d);
    d.B = sh->B; d.H = sh->H; d.H_kv = sh->H_kv; d.G = sh->H / sh->H_kv; d.d = sh->d;
    d.N = 1; d.C = sh->S_pre - 1; d.Cp = sh->S_pre; d.K = 1; d.Bk = sh->S_pre;
    d.L_q = 1; d.L = sh->L; d.L_s = sh->L_s;
    d.S_pre = sh->S_pre; d.S_kv = sh->S_pre + sh->L_s;
    d.rows_g = d.G * sh->L;
    d.scale = sh->scale > 0.f ? sh->scale : 1.0f / std::sqrt((float)sh->d);
    d.contig = 1;
    *out = d;
    return PDLLM_OK;
}

int dense_attn(const pdllm_dense_shape *shape, const void *Q, const void *Kpre, const void *Vpre, const void *K_dec,
               const void *V_dec, int32_t n_splits, void *O, float *LSE, void *workspace, size_t workspace_bytes,
               pdllm_stream_t stream) {
    if (!shape || !Q || !Kpre || !Vpre || !O || !LSE) return PDLLM_ERR_NULL;
    if (n_splits < 0) return PDLLM_ERR_SHAPE;
    Dims d;
    if (int rc = resolve_dense(shape, &d)) return rc;
    if (d.L_s > 0 && (!K_dec || !V_dec)) return PDLLM_ERR_NULL;
    if (!aligned16(Q) || !aligned16(Kpre) || !aligned16(Vpre) || !aligned16(O) || !aligned16(workspace) ||
        (d.L_s > 0 && (!aligned16(K_dec) || !aligned16(V_dec))))
        return PDLLM_ERR_ALIGN;
    int S = effective_splits(d, n_splits, device_num_sms());
    if (!workspace) return PDLLM_ERR_WORKSPACE;
    if (n_splits == 0)
        while (S > 1 && workspace_bytes < workspace_for(d, S)) --S;
    if (workspace_bytes < workspace_for(d, S)) return PDLLM_ERR_WORKSPACE;
    return attn_impl(d, Q, Kpre, Vpre, nullptr, nullptr, K_dec, V_dec, S, O, LSE, nullptr, workspace, false, nullptr,
                     nullptr, static_cast<cudaStream_t>(stream));
}

}  // namespace

size_t pdllm_dense_workspace_bytes(const pdllm_dense_shape *shape, int32_t n_splits, int32_t num_sms) {
    Dims d;
    if (n_splits < 0 || resolve_dense(shape, &d) != PDLLM_OK) return 0;
    return workspace_for(d, effective_splits(d, n_splits, num_sms));
}

int32_t pdllm_dense_auto_splits(const pdllm_dense_shape *shape, int32_t num_sms) {
    Dims d;
    if (resolve_dense(shape, &d) != PDLLM_OK) return 1;
    return effective_splits(d, 0, num_sms);
}

int pdllm_compact_kv(const pdllm_shape *shape, const void *Kcache, const void *Vcache, const int32_t *chunk_ids,
                     const int32_t *token_keep_idx, void *Kcompact, void *Vcompact, pdllm_stream_t stream) {
    if (!shape || !Kcache || !Vcache || !chunk_ids || !Kcompact || !Vcompact) return PDLLM_ERR_NULL;
    Dims d;
    if (int rc = resolve(shape, token_keep_idx != nullptr, &d)) return rc;
    if (!aligned16(Kcache) || !aligned16(Vcache) || !aligned16(Kcompact) || !aligned16(Vcompact)) return PDLLM_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (int rc = debug_validate(d, chunk_ids, token_keep_idx, st)) return rc;
    return cuda_rc(launch_compact_kv(d, Kcache, Vcache, chunk_ids, token_keep_idx, Kcompact, Vcompact, st));
}

int pdllm_static_attn(const pdllm_dense_shape *shape, const void *Q_dec, const void *Kcompact, const void *Vcompact,
                      const void *K_dec, const void *V_dec, int32_t n_splits, void *O, float *LSE, void *workspace,
                      size_t workspace_bytes, pdllm_stream_t stream) {
    return dense_attn(shape, Q_dec, Kcompact, Vcompact, K_dec, V_dec, n_splits, O, LSE, workspace, workspace_bytes, stream);
}

int pdllm_prefill_attn(const pdllm_dense_shape *shape, const void *Q, const void *K, const void *V, int32_t n_splits,
                       void *O, float *LSE, void *workspace, size_t workspace_bytes, pdllm_stream_t stream) {
    if (shape && (shape->L_s != 0 || shape->L != shape->S_pre)) return PDLLM_ERR_SHAPE;
    return dense_attn(shape, Q, K, V, nullptr, nullptr, n_splits, O, LSE, workspace, workspace_bytes, stream);
}

// ---- NEXT-1: token eviction scores and top-B retention
namespace {
struct TokScratch { size_t scores, row_lse, part, total; };
TokScratch tok_scratch(const Dims &d) {
    TokScratch t;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes, 256); return o; };
    const size_t BG = (size_t)d.B * d.H_kv, rows = (size_t)d.G * d.L_q, m_tiles = (rows + kTileM - 1) / kTileM;
    t.scores = take(BG * d.N * sizeof(float));
    t.row_lse = take(BG * d.N * rows * sizeof(float));
    t.part = off;
    if (m_tiles > 1) take(m_tiles * BG * d.N * d.Cp * sizeof(float));
    t.total = off;
    return t;
}
}  // namespace

size_t pdllm_score_tokens_workspace_bytes(const pdllm_shape *shape) {
    if (!shape) return 0;
    Dims d;
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (resolve(&sh, false, &d) != PDLLM_OK) return 0;
    return tok_scratch(d).total;
}

int pdllm_score_tokens(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                       const void *Kcache, float *token_scores, void *workspace, size_t workspace_bytes,
                       pdllm_stream_t stream) {
    if (!shape || !Q || !Kcache || !token_scores || !workspace) return PDLLM_ERR_NULL;
    Dims d;
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (int rc = resolve(&sh, false, &d)) return rc;
    if (!aligned16(Q) || !aligned16(Kcache) || !aligned16(token_scores) || !aligned16(workspace)) return PDLLM_ERR_ALIGN;
    if ((q_batch_stride & 7) || (q_head_stride & 7) || q_head_stride < (int64_t)d.L_q * d.d) return PDLLM_ERR_ALIGN;
    const TokScratch t = tok_scratch(d);
    if (workspace_bytes < t.total) return PDLLM_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char *base = static_cast<char *>(workspace);
    float *row_lse = reinterpret_cast<float *>(base + t.row_lse);
    // pass 1: the chunk-score kernel exports every scoring row's log-mass per chunk; pass 2: the token kernel
    if (int rc = cuda_rc(launch_score(d, Q, q_batch_stride, q_head_stride, Kcache, reinterpret_cast<float *>(base + t.scores),
                                      row_lse, nullptr, st)))
        return rc;
    return cuda_rc(launch_token_scores(d, Q, q_batch_stride, q_head_stride, Kcache, row_lse, token_scores,
                                       reinterpret_cast<float *>(base + t.part), st));
}

int pdllm_select_topb(const pdllm_shape *shape, const float *token_scores, int32_t *token_keep_idx, pdllm_stream_t stream) {
    if (!shape || !token_scores || !token_keep_idx) return PDLLM_ERR_NULL;
    Dims d;
    if (int rc = resolve(shape, true, &d)) return rc;
    if (d.Cp > topb_max_cp()) return PDLLM_ERR_UNSUPPORTED;
    return cuda_rc(launch_topb(d, token_scores, token_keep_idx, static_cast<cudaStream_t>(stream)));
}

int pdllm_pool_keys(const pdllm_shape *shape, const void *Kcache, float *kbar, pdllm_stream_t stream) {
    if (!shape || !Kcache || !kbar) return PDLLM_ERR_NULL;
    Dims d;
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (int rc = resolve(&sh, false, &d)) return rc;
    if (!aligned16(Kcache) || !aligned16(kbar)) return PDLLM_ERR_ALIGN;
    return cuda_rc(launch_pool_keys(d, Kcache, kbar, static_cast<cudaStream_t>(stream)));
}

int pdllm_score_chunks_pooled(const pdllm_shape *shape, const void *Q, int64_t q_batch_stride, int64_t q_head_stride,
                              const float *kbar, float *scores, pdllm_stream_t stream) {
    if (!shape || !Q || !kbar || !scores) return PDLLM_ERR_NULL;
    Dims d;
    pdllm_shape sh = *shape;
    sh.Bk = sh.C + 1;
    if (int rc = resolve(&sh, false, &d)) return rc;
    if (q_head_stride < (int64_t)d.L_q * d.d) return PDLLM_ERR_ALIGN;
    return cuda_rc(launch_pooled_scores(d, Q, q_batch_stride, q_head_stride, kbar, scores, static_cast<cudaStream_t>(stream)));
}

int pdllm_step_profiled(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
                        const int32_t *token_keep_idx, const void *K_dec, const void *V_dec, int32_t n_splits,
                        float *scores_out, int32_t *chunk_ids_out, void *O, float *LSE, int32_t *gather_idx_out,
                        void *workspace, size_t workspace_bytes, const pdllm_stage_events *ev, pdllm_stream_t stream) {
    if (!shape || !scores_out || !chunk_ids_out) return PDLLM_ERR_NULL;
    if (shape->L_q > shape->L) return PDLLM_ERR_SHAPE;
    // validate the attention arguments before anything is enqueued
    Dims d;
    int S = 1;
    if (int rc = attn_validate(shape, Q_dec, Kcache, Vcache, chunk_ids_out, token_keep_idx, K_dec, V_dec, n_splits, O,
                               LSE, workspace, workspace_bytes, &d, &S))
        return rc;
    if (!aligned16(scores_out)) return PDLLM_ERR_ALIGN;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (int rc = debug_validate(d, nullptr, token_keep_idx, st)) return rc;
    // the attention's work-item counter is cleared by the score kernel (no memset node between the step's kernels)
    if (int rc = record(ev ? ev->begin : nullptr, st)) return rc;
    // with several M tiles of scoring rows (G*L_q > 128) the score kernel leaves per-M-tile partials in the workspace
    // and the top-K kernel sums them in M-tile order: no float atomics, bit-reproducible scores
    float *sp = score_partial_bytes(d) ? reinterpret_cast<float *>(static_cast<char *>(workspace) + kCounterBytes + partials_bytes(d, S))
                                       : nullptr;
    if (int rc = cuda_rc(launch_score(d, Q_dec, (int64_t)d.H * d.L * d.d, (int64_t)d.L * d.d, Kcache, scores_out, nullptr, sp, st, static_cast<int32_t *>(workspace))))
        return rc;
    // a2 inside the attention kernel (one launch fewer; the attention becomes the score kernel's programmatic
    // dependent) when the chunk count allows it, no gather-index export wants the ids ahead of a4 and no stage
    // events are asked for; the ids and scores written are those the top-K kernel would write
    if (!ev && !gather_idx_out && attn_can_fold_topk(d) && !no_fold()) {
        AttnFold fold{scores_out, sp, chunk_ids_out, scores_out};
        return attn_impl(d, Q_dec, Kcache, Vcache, chunk_ids_out, token_keep_idx, K_dec, V_dec, S, O, LSE, nullptr,
                         workspace, true, nullptr, nullptr, st, &fold);
    }
    if (int rc = record(ev ? ev->after_score : nullptr, st)) return rc;
    if (int rc = cuda_rc(launch_topk(d, scores_out, chunk_ids_out, st, sp, scores_out))) return rc;
    if (int rc = record(ev ? ev->after_topk : nullptr, st)) return rc;
    return attn_impl(d, Q_dec, Kcache, Vcache, chunk_ids_out, token_keep_idx, K_dec, V_dec, S, O, LSE, gather_idx_out,
                     workspace, true, ev ? ev->after_attn : nullptr, ev ? ev->end : nullptr, st);
}

int pdllm_step(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
               const int32_t *token_keep_idx, const void *K_dec, const void *V_dec, int32_t n_splits, float *scores_out,
               int32_t *chunk_ids_out, void *O, float *LSE, int32_t *gather_idx_out, void *workspace,
               size_t workspace_bytes, pdllm_stream_t stream) {
    return pdllm_step_profiled(shape, Q_dec, Kcache, Vcache, token_keep_idx, K_dec, V_dec, n_splits, scores_out,
                               chunk_ids_out, O, LSE, gather_idx_out, workspace, workspace_bytes, nullptr, stream);
}

int pdllm_step_host(const pdllm_shape *shape, const void *h_Q_dec, const void *h_K_dec, const void *h_V_dec,
                    const void *d_Kcache, const void *d_Vcache, const int32_t *d_token_keep_idx, int32_t n_splits,
                    void *h_O, float *h_LSE, int32_t *h_chunk_ids, void *d_scratch, size_t scratch_bytes,
                    const pdllm_side_stream *side, pdllm_stream_t stream) {
    if (!shape || !h_Q_dec || !h_K_dec || !h_V_dec || !d_Kcache || !d_Vcache || !h_O || !h_LSE || !h_chunk_ids || !d_scratch)
        return PDLLM_ERR_NULL;
    if (n_splits < 0) return PDLLM_ERR_SHAPE;
    Dims d;
    if (int rc = resolve(shape, d_token_keep_idx != nullptr, &d)) return rc;
    if (!aligned16(d_scratch)) return PDLLM_ERR_ALIGN;
    const int S = effective_splits(d, n_splits, device_num_sms());
    const HostScratch h = host_scratch(d, S);
    if (scratch_bytes < h.total) return PDLLM_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char *base = static_cast<char *>(d_scratch);
    const size_t qb = (size_t)d.B * d.H * d.L * d.d * 2, kb = (size_t)d.B * d.H_kv * d.L_s * d.d * 2;
    int32_t *ids = reinterpret_cast<int32_t *>(base + h.ids);
    float *scores = reinterpret_cast<float *>(base + h.scores);
    Dims dv;
    int Sv = 1;
    if (int rc = attn_validate(shape, base + h.q, d_Kcache, d_Vcache, ids, d_token_keep_idx, base + h.kd, base + h.vd,
                               n_splits, base + h.o, reinterpret_cast<float *>(base + h.lse), base + h.ws, h.total - h.ws,
                               &dv, &Sv))
        return rc;
    if (shape->L_q > shape->L) return PDLLM_ERR_SHAPE;
    if (int rc = debug_validate(dv, nullptr, d_token_keep_idx, st)) return rc;
    // Scoring and top-K need only Q: with a caller-supplied side stream K_dec / V_dec travel underneath them and join
    // before the attention (fork after everything queued on `stream`, so an earlier step's kernels have let go of
    // the scratch buffers).  Without one, all copies go on `stream` in order.
    if (side && (!side->stream || !side->ev_fork || !side->ev_join)) return PDLLM_ERR_NULL;
    cudaStream_t st2 = side ? static_cast<cudaStream_t>(side->stream) : st;
    cudaEvent_t ev_fork = side ? static_cast<cudaEvent_t>(side->ev_fork) : nullptr;
    cudaEvent_t ev_join = side ? static_cast<cudaEvent_t>(side->ev_join) : nullptr;
    if (side) {
        if (cudaEventRecord(ev_fork, st) != cudaSuccess) return PDLLM_ERR_CUDA;
        if (cudaStreamWaitEvent(st2, ev_fork, 0) != cudaSuccess) return PDLLM_ERR_CUDA;
    }
    if (cudaMemcpyAsync(base + h.q, h_Q_dec, qb, cudaMemcpyHostToDevice, st) != cudaSuccess) return PDLLM_ERR_CUDA;
    if (cudaMemcpyAsync(base + h.kd, h_K_dec, kb, cudaMemcpyHostToDevice, st2) != cudaSuccess) return PDLLM_ERR_CUDA;
    if (cudaMemcpyAsync(base + h.vd, h_V_dec, kb, cudaMemcpyHostToDevice, st2) != cudaSuccess) return PDLLM_ERR_CUDA;
    if (side && cudaEventRecord(ev_join, st2) != cudaSuccess) return PDLLM_ERR_CUDA;
    float *sp = score_partial_bytes(dv) ? reinterpret_cast<float *>(base + h.ws + kCounterBytes + partials_bytes(dv, Sv)) : nullptr;
    if (int rc = cuda_rc(launch_score(dv, base + h.q, (int64_t)dv.H * dv.L * dv.d, (int64_t)dv.L * dv.d, d_Kcache, scores, nullptr, sp, st, reinterpret_cast<int32_t *>(base + h.ws))))
        return rc;
    const bool fold_topk = attn_can_fold_topk(dv) && !no_fold();
    if (!fold_topk)
        if (int rc = cuda_rc(launch_topk(dv, scores, ids, st, sp, scores))) return rc;
    if (side && cudaStreamWaitEvent(st, ev_join, 0) != cudaSuccess) return PDLLM_ERR_CUDA;
    AttnFold fold{scores, sp, ids, scores};
    if (int rc = attn_impl(dv, base + h.q, d_Kcache, d_Vcache, ids, d_token_keep_idx, base + h.kd, base + h.vd, Sv,
                           base + h.o, reinterpret_cast<float *>(base + h.lse), nullptr, base + h.ws, true, nullptr, nullptr,
                           st, fold_topk ? &fold : nullptr))
        return rc;
    if (cudaMemcpyAsync(h_O, base + h.o, qb, cudaMemcpyDeviceToHost, st) != cudaSuccess) return PDLLM_ERR_CUDA;
    if (cudaMemcpyAsync(h_LSE, base + h.lse, (size_t)d.B * d.H * d.L * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return PDLLM_ERR_CUDA;
    if (cudaMemcpyAsync(h_chunk_ids, base + h.ids, (size_t)d.B * d.H_kv * d.K * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return PDLLM_ERR_CUDA;
    return PDLLM_OK;
}

}  // extern "C"
