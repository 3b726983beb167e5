// skv_noalloc.cu -- skv_importance_kvnorm_noalloc (include/skv.h): the KV-norm fallback score of Alg. 1 step 2
// for callers that cannot hand the library a workspace.
//
// Who that is: code that sits inside somebody else's serving engine -- a C / C++ plug-in on the prefill worker, say --
// and receives only the tensors of the call (the key cache in, the scores out).  By the time it runs, the engine's own
// memory pool has reserved the device's HBM, so a cudaMalloc of its own fails with out-of-memory (and on a latency-
// critical loop it would be unwelcome anyway: cudaMalloc / cudaFree stall every stream of the device), and the engine
// gives the plug-in no handle to its pool.  Every other entry point of this library asks such a caller for a
// `workspace_dev` it has no means to produce.
//
// What it does instead: the two kernels of skv_kvnorm.cu need scratch in global memory between them (the un-normalised
// score of every token and one partial sum per 64 tokens).  Here that scratch is a fixed array that is part of the
// library image, SKV_NOALLOC_SCRATCH_BYTES large.  The driver places it on a GPU when the library's code is loaded
// there and it stays until the process exits -- that is the price: 4.25 MiB of HBM per GPU that uses the library,
// whether this entry point is ever called or not.
//
// The entry point itself calls no cudaMalloc, no cudaFree and no library routine that allocates; its only CUDA calls
// are cudaGetDevice, cudaGetSymbolAddress (first call per device only) and the two kernel launches of the existing
// path (launch_importance_kvnorm through skv_importance_kvnorm, unchanged).
#include <mutex>

#include "skv_common.cuh"

namespace {

// The scratch.  In HOST code this name is only a handle for the runtime's symbol table -- taking its address here
// gives a host pointer that a kernel must never see.  The device address comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_noalloc_scratch[SKV_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void *g_scratch_dev[kMaxDevices];        // per CUDA device ordinal: device address of g_noalloc_scratch, nullptr = not looked up yet

// Device address of the scratch on the CURRENT device; looked up once per device and cached.
int scratch_on_current_device(void **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return SKV_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return SKV_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_dev[dev]) {
        void *p = nullptr;
        // every GPU holds its own copy of the array at its own address: the answer is the current device's
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return SKV_ERR_CUDA;
        g_scratch_dev[dev] = p;
    }
    *out = g_scratch_dev[dev];
    return SKV_OK;
}

}  // namespace

extern "C" int skv_importance_kvnorm_noalloc(const skv_shape *shape, const void *K_dev, float lambda,
                                             float *importance_dev, void *cuda_stream)
{
    if (!shape || shape->n_layers <= 0 || shape->n_tokens <= 0 || shape->n_requests <= 0) return SKV_ERR_INVALID_ARG;
    // size first: a problem that does not fit is refused before anything touches the device
    skv::Geom g = {};
    g.R = shape->n_requests; g.L = shape->n_layers; g.n = shape->n_tokens;      // all that kvnorm_ws_bytes reads
    const int64_t max_scores = (int64_t)SKV_NOALLOC_SCRATCH_BYTES / 4;          // one f32 per (request, layer, token)
    const int64_t rl = (int64_t)g.R * g.L;                                      // < 2^62: no overflow
    if (rl > max_scores || rl * g.n > max_scores ||                             // (also keeps the next line from overflowing)
        skv::kvnorm_ws_bytes(g) > (size_t)SKV_NOALLOC_SCRATCH_BYTES)
        return SKV_ERR_NOALLOC_LIMIT;
    void *scratch = nullptr;
    const int rc = scratch_on_current_device(&scratch);
    if (rc) return rc;
    // Nothing in the scratch has to start at zero: the first kernel writes every score and every partial sum that the
    // second one reads, so whatever the previous call (of any shape) left behind is never looked at.
    return skv_importance_kvnorm(shape, K_dev, lambda, importance_dev, scratch, (size_t)SKV_NOALLOC_SCRATCH_BYTES, cuda_stream);
}
