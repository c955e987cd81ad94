// hlc2_static.cu -- hlc2_crossmatch_static: the match of hlc2_crossmatch with its scratch memory (the planner's job
// lists of the two-grid kernel, the general-row list of the same-grid kernel) in a file-scope device array instead of a
// caller buffer, for callers that cannot allocate device memory (include/hlc2.h).
//
// The array costs HLC2_STATIC_SCRATCH_BYTES on every GPU that loads the library, until the process exits.  Every call on
// a device shares it: calls that overlap on the GPU race on it.  It keeps the last call's contents; the match launchers
// zero the counters they keep in their scratch on every call (they never assumed a cleared caller buffer), nothing else
// in it is read before it is written.
//
// In host code the array's NAME is a host-side stand-in, not a device address: the address is taken once per device, with
// that device current, by cudaGetSymbolAddress below, and that address is what the kernels get.
#include <mutex>

#include "hlc2_internal.cuh"

namespace hlc2 {

static __device__ __align__(256) unsigned char g_static_scratch[HLC2_STATIC_SCRATCH_BYTES];

// device address of g_static_scratch on the CURRENT device (resolved on first use, cached per device)
static cudaError_t static_scratch_ptr(void** out) {
    static std::mutex mu;
    static void* cache[kMaxDevices] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!cache[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        cache[dev] = p;
    }
    *out = cache[dev];
    return cudaSuccess;
}

}  // namespace hlc2

extern "C" int hlc2_crossmatch_static(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                                      int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                                      int64_t capacity, unsigned long long* d_count, void* cuda_stream) {
    size_t need = 0;
    int rc = hlc2_crossmatch_sizes(A, B, &need);          // also checks the handles
    if (rc != HLC2_OK) return rc;
    if (need > (size_t)HLC2_STATIC_SCRATCH_BYTES) return HLC2_ERR_STATIC_LIMIT;
    void* scratch = nullptr;
    cudaError_t e = hlc2::static_scratch_ptr(&scratch);
    if (e != cudaSuccess) { hlc2::note_cuda_error(e); return HLC2_ERR_CUDA; }
    // the existing path from here on, with the static array as its scratch: no cudaMalloc / cudaFree anywhere in it
    return hlc2_crossmatch(A, B, radius_arcsec, mode, d_out_idA, d_out_idB, d_out_sep_arcsec, capacity, d_count,
                           scratch, (size_t)HLC2_STATIC_SCRATCH_BYTES, cuda_stream);
}
