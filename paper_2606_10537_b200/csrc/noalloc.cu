// noalloc.cu -- pdllm_sparse_attn_noalloc: a3 + a4 + a5 for callers that cannot allocate device memory
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// pdllm_sparse_attn wants a caller-allocated workspace (the persistent kernel's work-item counter and, for n_splits > 1,
// the fp32 Split-S partials the combine kernel merges).  Here that scratch is a file-scope device array of
// PDLLM_NOALLOC_SCRATCH_BYTES: every GPU that loads the library holds it until the process exits, and no call allocates
// or frees anything.  The rest of the path is pdllm_sparse_attn itself (same kernels, same split choice, same results).
//
// In host code the array's NAME is a host-side stand-in, not a device address: handing it to a kernel faults or, where the
// GPU can reach host memory, silently uses the wrong memory.  The device address comes from cudaGetSymbolAddress, asked
// once per device with that device current, and is what the kernels get.
#include <atomic>
#include <cstdlib>
#include <cstring>

#include "pdllm_internal.h"

namespace {

// the one scratch array: shared by every call on the device, never cleared as a whole, keeps the last call's contents
static __device__ __align__(256) unsigned char g_noalloc_scratch[PDLLM_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;

// device address of g_noalloc_scratch on the CURRENT device (looked up once per device); nullptr + *rc on failure
void *scratch_on_current_device(int *rc) {
    static std::atomic<void *> cache[kMaxDevices];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        *rc = PDLLM_ERR_CUDA;
        return nullptr;
    }
    if (dev < 0 || dev >= kMaxDevices) {
        *rc = PDLLM_ERR_UNSUPPORTED;
        return nullptr;
    }
    void *ptr = cache[dev].load(std::memory_order_acquire);
    if (ptr) return ptr;
    // two threads may both get here: both read the same address, the second store is harmless
    if (cudaGetSymbolAddress(&ptr, g_noalloc_scratch) != cudaSuccess || !ptr) {
        (void)cudaGetLastError();
        *rc = PDLLM_ERR_CUDA;
        return nullptr;
    }
    cache[dev].store(ptr, std::memory_order_release);
    return ptr;
}

}  // namespace

extern "C" int pdllm_sparse_attn_noalloc(const pdllm_shape *shape, const void *Q_dec, const void *Kcache, const void *Vcache,
                                         const int32_t *chunk_ids, const int32_t *token_keep_idx, const void *K_dec,
                                         const void *V_dec, int32_t n_splits, void *O, float *LSE, int32_t *gather_idx_out,
                                         pdllm_stream_t stream) {
    if (!shape) return PDLLM_ERR_NULL;
    if (n_splits < 0) return PDLLM_ERR_SHAPE;
    // the debug switch (include/pdllm.h, "DEBUG SWITCH") makes pdllm_sparse_attn allocate a 4-byte flag and synchronise
    // the stream: not something this entry point may do, so it refuses to run under it rather than skip the check
    if (const char *e = std::getenv("PDLLM_DEBUG_VALIDATE"))
        if (e[0] != '\0' && std::strcmp(e, "0") != 0) return PDLLM_ERR_UNSUPPORTED;
    // an explicit split count whose partials do not fit the fixed array is refused before anything touches the device;
    // n_splits == 0 cannot overflow it: pdllm_sparse_attn then takes the largest split count the scratch holds
    if (n_splits > 0) {
        const size_t need = pdllm_workspace_bytes(shape, n_splits, 0);
        if (need == 0) return PDLLM_ERR_SHAPE;
        if (need > (size_t)PDLLM_NOALLOC_SCRATCH_BYTES) return PDLLM_ERR_SCRATCH_LIMIT;
    }
    int rc = PDLLM_OK;
    void *scratch = scratch_on_current_device(&rc);
    if (!scratch) return rc;
    // what must start at zero -- the work-item counter at the head of the scratch -- is cleared on the stream by
    // pdllm_sparse_attn itself; the partials are written in full before the combine kernel reads them
    return pdllm_sparse_attn(shape, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, n_splits, O, LSE,
                             gather_idx_out, scratch, (size_t)PDLLM_NOALLOC_SCRATCH_BYTES, stream);
}
