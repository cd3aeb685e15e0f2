// sm_trace_dk_static: the band-structure energy tr(D K) (Eq.(10)) for callers that must not allocate
// (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same quantity as sm_trace_dk's
// tr_DK, but no plan and no allocation of any kind: the reduction scratch is a file-scope __device__ array of a
// fixed maximum size, held by every GPU that loads the library until the process exits.
//
// Reduction (deterministic, independent of the grid size): the value arrays are cut into chunks of NA_CHUNK
// elements; a CTA reduces a chunk in a fixed order and writes partial[chunk] into the scratch; the CTA that takes
// the last ticket sums the partials in a fixed order and writes the result.  The ticket counter lives in the same
// array and must be zero when a call starts: it is cleared on the caller's stream at the start of every call
// (the array keeps the previous call's contents).
//
// The scratch is shared by all calls: two calls whose kernels overlap on the GPU (different streams, or different
// host threads on different streams) race on it; calls on one stream are ordered and safe.
#include <algorithm>
#include <cstdio>
#include <mutex>

#include "common.cuh"

namespace smb {

constexpr int NA_CHUNK = 4096;           // values per partial
constexpr int NA_MAX_CHUNKS = 65536;     // => SM_STATIC_MAX_NNZ = 268,435,456 values; 512 KB + 256 B of scratch
constexpr int NA_THREADS = 256;
static_assert((int64_t)NA_CHUNK * NA_MAX_CHUNKS == SM_STATIC_MAX_NNZ, "header constant out of step with the scratch size");

// [0, NA_MAX_CHUNKS): partials; [NA_MAX_CHUNKS]: ticket counter (first 4 bytes)
static __device__ __align__(256) double g_na_scratch[NA_MAX_CHUNKS + 32];

// `scratch` is the DEVICE address of g_na_scratch (cudaGetSymbolAddress; in host code the symbol's name is only a
// host-side stand-in and must not be passed to a kernel).
__global__ void __launch_bounds__(NA_THREADS)
k_trace_dk_static(int64_t nnz, int n_chunks, const double* __restrict__ D, const double* __restrict__ K,
                  double* __restrict__ scratch, double* __restrict__ out) {
    __shared__ double s[NA_THREADS];
    __shared__ unsigned s_ticket;
    for (int c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const int64_t b = (int64_t)c * NA_CHUNK, e = min(b + NA_CHUNK, nnz);
        double a = 0.0;
        for (int64_t i = b + threadIdx.x; i < e; i += NA_THREADS) a = fma(D[i], K[i], a);
        s[threadIdx.x] = a;
        __syncthreads();
        for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) scratch[c] = s[0];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        __threadfence();  // this CTA's partials before its ticket
        s_ticket = atomicAdd(reinterpret_cast<unsigned*>(scratch + NA_MAX_CHUNKS), 1u);
    }
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    __threadfence();      // last CTA: every other CTA's partials are visible
    double a = 0.0;
    for (int c = threadIdx.x; c < n_chunks; c += NA_THREADS) a += __ldcg(scratch + c);
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = s[0];
}

// Device address of the scratch array on the current device: resolved once per device, with that device current.
static std::mutex g_na_mu;
static double* g_na_ptr[64] = {nullptr};

static sm_status_t na_scratch(double** ptr) {
    int dev = -1;
    SM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) {
        set_error_text("sm_trace_dk_static: device ordinal outside the supported range 0..63");
        return SM_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_na_mu);
    if (!g_na_ptr[dev]) {
        double* p = nullptr;
        SM_CUDA(cudaGetSymbolAddress((void**)&p, g_na_scratch));
        if (!p) {
            set_error_text("sm_trace_dk_static: cudaGetSymbolAddress returned a null address");
            return SM_ERR_CUDA;
        }
        g_na_ptr[dev] = p;
    }
    *ptr = g_na_ptr[dev];
    return SM_OK;
}

}  // namespace smb

using namespace smb;

extern "C" sm_status_t sm_trace_dk_static(int64_t nnz, const double* d_D, const double* d_K, double* d_tr_DK,
                                          void* cuda_stream) {
    // argument checks first: host logic only, no CUDA call
    if (nnz < 0 || !d_tr_DK || (nnz > 0 && (!d_D || !d_K))) {
        set_error_text("sm_trace_dk_static: negative size or null pointer");
        return SM_ERR_INVALID_ARG;
    }
    if (nnz > (int64_t)SM_STATIC_MAX_NNZ) {
        char msg[200];
        snprintf(msg, sizeof(msg), "sm_trace_dk_static: nnz = %lld exceeds SM_STATIC_MAX_NNZ = %lld (fixed scratch; use sm_trace_dk)",
                 (long long)nnz, (long long)SM_STATIC_MAX_NNZ);
        set_error_text(msg);
        return SM_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* scratch = nullptr;
    sm_status_t s = na_scratch(&scratch);
    if (s) return s;
    const int n_chunks = (int)((nnz + NA_CHUNK - 1) / NA_CHUNK);
    int sms = 0, dev = 0;
    SM_CUDA(cudaGetDevice(&dev));
    SM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = std::max(1, std::min(n_chunks, std::max(sms, 1) * 8));
    // the ticket counter must start at zero; the array keeps whatever the previous call left
    SM_CUDA(cudaMemsetAsync(scratch + NA_MAX_CHUNKS, 0, 8, st));
    k_trace_dk_static<<<grid, NA_THREADS, 0, st>>>(nnz, n_chunks, d_D, d_K, scratch, d_tr_DK);
    SM_CUDA(cudaGetLastError());
    return SM_OK;
}
