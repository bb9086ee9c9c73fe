// mttkrp_get_perm_noalloc: mttkrp_get_perm for callers that have no device memory to lend.
//
// mttkrp_get_perm carries the original-position array from layout 0 to layout d by ping-ponging between the
// caller's output and a second nnz-word buffer that the caller must bring along.  Bringing it along means
// allocating it at the moment of the call, and some callers cannot: code that runs inside an application whose
// memory pool already owns the whole GPU (a raw cudaMalloc then fails, or goes behind the pool's back), and code on a
// multi-stream pipeline that must not take the device-wide stall cudaMalloc / cudaFree cause.  For them the second
// buffer lives here, in a fixed array that is part of the loaded library image, and the entry point calls nothing
// that allocates.
//
// The price: the array has a fixed size (kNoAllocMaxNnz words = 16 MiB), every GPU that loads the library carries it
// until the process exits whether or not the entry point is ever called, and every call on a device shares it.
#include <mutex>
#include "common.cuh"

namespace mk {

constexpr int64_t kNoAllocMaxNnz = MTTKRP_NOALLOC_MAX_NNZ;
constexpr int kNoAllocMaxDevices = 64;

// The ping-pong partner of perm_dev.  A call leaves behind whichever intermediate original-position array it wrote
// there last (d == 0 does not touch it).  No call reads a word it has not written first, so nothing is cleared.
static __device__ __align__(256) uint32_t g_perm_scratch[kNoAllocMaxNnz];

// In host code `g_perm_scratch` is only the host compiler's shadow of the device array; its address means nothing
// to a kernel.  The device address is asked for once per device (with that device current) and kept here.
static std::mutex g_scratch_mu;
static uint32_t* g_scratch_dev[kNoAllocMaxDevices];      // zero-initialised: not resolved yet

static mttkrp_status_t perm_scratch_for_current_device(int expect_device, uint32_t** out) {
    int dev = -1;
    MK_CUDA(cudaGetDevice(&dev));
    if (dev != expect_device) {
        set_error("mttkrp_get_perm_noalloc: current device %d is not the handle's device %d", dev, expect_device);
        return MTTKRP_EINVAL;
    }
    if (dev < 0 || dev >= kNoAllocMaxDevices) {
        set_error("mttkrp_get_perm_noalloc: device ordinal %d outside [0,%d)", dev, kNoAllocMaxDevices);
        return MTTKRP_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_dev[dev]) {
        void* p = nullptr;
        MK_CUDA(cudaGetSymbolAddress(&p, g_perm_scratch));   // loads this module on `dev` if it is not loaded yet
        if (!p) { set_error("mttkrp_get_perm_noalloc: cudaGetSymbolAddress returned NULL"); return MTTKRP_ECUDA; }
        g_scratch_dev[dev] = static_cast<uint32_t*>(p);
    }
    *out = g_scratch_dev[dev];
    return MTTKRP_OK;
}

}  // namespace mk

using namespace mk;

extern "C" mttkrp_status_t mttkrp_get_perm_noalloc(mttkrp_handle_t h, int d, uint32_t* perm_dev, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (d < 0 || d >= h->N) { set_error("mode %d outside [0,%d)", d, h->N); return MTTKRP_EINVAL; }
    if (h->nnz > kNoAllocMaxNnz) {
        set_error("mttkrp_get_perm_noalloc: nnz %lld exceeds the built-in scratch of %lld entries (MTTKRP_NOALLOC_MAX_NNZ); "
                  "use mttkrp_get_perm with a caller-provided scratch buffer",
                  (long long)h->nnz, (long long)kNoAllocMaxNnz);
        return MTTKRP_EUNSUPPORTED;
    }
    if (h->nnz == 0) return MTTKRP_OK;
    if (!perm_dev) { set_error("perm_dev is NULL"); return MTTKRP_EINVAL; }
    uint32_t* scratch = nullptr;
    MK_TRY(perm_scratch_for_current_device(h->device, &scratch));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // Same ordering rule as every call on a handle (api.cu order_begin / order_end): wait for the handle's previous
    // work if it went to another stream, leave an event behind for the next call.  The event exists since create.
    if (h->launched && st != h->last_stream) MK_CUDA(cudaStreamWaitEvent(st, h->ev_order, 0));
    // perm_{j+1}[k] = perm_j[next_j[k]] (Observation 1: every step is a bijection); the start
    // buffer is chosen so that step d lands in perm_dev.
    uint32_t* a = (d % 2 == 0) ? perm_dev : scratch;
    uint32_t* b = (d % 2 == 0) ? scratch : perm_dev;
    MK_CUDA(cudaMemcpyAsync(a, h->perm0, (size_t)h->nnz * 4, cudaMemcpyDeviceToDevice, st));
    for (int j = 0; j < d; ++j) {
        MK_TRY(launch_perm_step(h->mode[j].next, a, b, h->nnz, st));
        uint32_t* t = a; a = b; b = t;
    }
    MK_CUDA(cudaEventRecord(h->ev_order, st));
    h->last_stream = st;
    h->launched = 1;
    return MTTKRP_OK;
}
