// no_alloc.cu -- fredopt_volume_histogram_no_alloc: the cumulative volume histogram (DVH / LVH / cDLVH)
// of the caller's own voxel arrays for callers that cannot allocate device memory (code under CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc).  A variant of k_value_hist (kernels_eval.cuh), whose bin counters are plan-owned
// scratch: here the counters live in a file-scope __device__ array of a fixed maximum size, so the call needs no plan and
// allocates nothing.  The file shares no code path with the rest of the library.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include <string>

#include "../../include/fredopt.h"

extern thread_local std::string g_last_cuda_error;      // passes.cu; read through fredopt_last_cuda_error()

namespace fredopt {

// The scratch: FREDOPT_NO_ALLOC_MAX_BINS bin counters + the structure's voxel count.  32 776 bytes of device memory on every GPU
// that loads the library, until the process exits.  Shared by every call on that GPU and never cleared between calls: each
// call clears the counters it uses first, in stream order; calls that overlap on one GPU (two streams) race.
static __device__ __align__(256) unsigned long long g_hist_scratch[FREDOPT_NO_ALLOC_MAX_BINS + 1];

constexpr int NA_MAX_DEVICES = 64;
static unsigned long long* g_scratch_ptr[NA_MAX_DEVICES];      // device address of g_hist_scratch per device (host-side table)
static std::mutex g_scratch_mutex;

constexpr int NA_THREADS = 256;

__global__ void __launch_bounds__(NA_THREADS) k_na_clear(unsigned long long* __restrict__ cnt, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) cnt[i] = 0ULL;
}

// cnt[b] += 1 for the largest b with b * vmax / n_bins <= value over the voxels of the structure (labels[i] == label, or every
// voxel when labels == NULL); cnt[n_bins] += the structure's voxel count.  The bin of a value is decided as k_value_hist
// decides it (fp64, edges b * vmax / n_bins; values below edge 0 and NaN are in the volume but in no bin).  Counts are
// gathered per CTA in shared memory and flushed once.
__global__ void __launch_bounds__(NA_THREADS)
k_na_count(long long n, const float* __restrict__ values, const int32_t* __restrict__ labels, int label, int n_bins, double vmax,
           unsigned long long* __restrict__ cnt) {
    __shared__ unsigned int sm[FREDOPT_NO_ALLOC_MAX_BINS + 1];
    for (int b = threadIdx.x; b <= n_bins; b += blockDim.x) sm[b] = 0u;
    __syncthreads();
    // a CTA handles at most 2^31 voxels (grid sizing in the launcher), so the 32-bit shared counters cannot wrap
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        if (labels && labels[i] != label) continue;
        atomicAdd(sm + n_bins, 1u);
        const double t = (double)values[i];
        if (!(t >= 0.0)) continue;                       // edge 0 is 0
        const double g = floor(t / vmax * (double)n_bins);
        int b = g >= (double)(n_bins - 1) ? n_bins - 1 : (int)g;
        while (b + 1 < n_bins && (double)(b + 1) * vmax / (double)n_bins <= t) ++b;
        while (b > 0 && (double)b * vmax / (double)n_bins > t) --b;
        atomicAdd(sm + b, 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b <= n_bins; b += blockDim.x)
        if (sm[b]) atomicAdd(cnt + b, (unsigned long long)sm[b]);
}

// hist[b] = (number of voxels in bins >= b) / (voxels of the structure), 0 for an empty structure.  One CTA of 1024 threads,
// each owning 4 neighbouring bins; integer sums, so the order of the additions does not matter.
__global__ void __launch_bounds__(1024)
k_na_finish(const unsigned long long* __restrict__ cnt, int n_bins, float* __restrict__ hist, long long* __restrict__ n_voxels) {
    __shared__ unsigned long long suf[1024];
    const int t = threadIdx.x, b0 = 4 * t;
    unsigned long long c[4];
    unsigned long long own = 0ULL;
#pragma unroll
    for (int k = 0; k < 4; ++k) { c[k] = b0 + k < n_bins ? cnt[b0 + k] : 0ULL; own += c[k]; }
    suf[t] = own;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {                 // inclusive suffix sums over the threads
        const unsigned long long add = t + o < 1024 ? suf[t + o] : 0ULL;
        __syncthreads();
        suf[t] += add;
        __syncthreads();
    }
    const unsigned long long nr = cnt[n_bins];
    unsigned long long cum = suf[t] - own;               // voxels in the bins of the threads above
#pragma unroll
    for (int k = 3; k >= 0; --k) {
        cum += c[k];
        if (b0 + k < n_bins) hist[b0 + k] = nr ? (float)((double)cum / (double)nr) : 0.f;
    }
    if (t == 0 && n_voxels) *n_voxels = (long long)nr;
}

static int na_fail(const char* what) {
    g_last_cuda_error = what;
    return FREDOPT_INVALID_ARG;
}

// device address of the scratch on the current device, looked up once per device with that device current
static int na_scratch(unsigned long long** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { g_last_cuda_error = std::string("cudaGetDevice: ") + cudaGetErrorString(e); cudaGetLastError(); return FREDOPT_CUDA_ERROR; }
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail("fredopt_no_alloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        int major = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) { g_last_cuda_error = std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e); cudaGetLastError(); return FREDOPT_CUDA_ERROR; }
        if (major != 10) return FREDOPT_UNSUPPORTED_ARCH;
        unsigned long long* p = nullptr;
        // in host code `g_hist_scratch` names a host-side stand-in of the symbol, not device memory: ask the runtime
        e = cudaGetSymbolAddress((void**)&p, g_hist_scratch);
        if (e != cudaSuccess || !p) {
            g_last_cuda_error = std::string("cudaGetSymbolAddress(g_hist_scratch): ") + cudaGetErrorString(e);
            cudaGetLastError();
            return FREDOPT_CUDA_ERROR;
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return FREDOPT_OK;
}

}  // namespace fredopt

using namespace fredopt;

extern "C" {

int fredopt_no_alloc_setup(void) {
    unsigned long long* p;
    return na_scratch(&p);
}

int fredopt_volume_histogram_no_alloc(const float* values, const int32_t* labels, int64_t n_voxels, int32_t label, int32_t n_bins,
                                      double vmax, float* hist, int64_t* n_in_structure, void* cuda_stream) {
    if (!values || !hist || n_voxels < 0) return na_fail("fredopt_volume_histogram_no_alloc: null values / hist or negative n_voxels");
    if (!(vmax > 0.0) || !std::isfinite(vmax)) return na_fail("fredopt_volume_histogram_no_alloc: vmax must be positive and finite");
    if (n_bins < 1) return na_fail("fredopt_volume_histogram_no_alloc: n_bins < 1");
    if (n_bins > FREDOPT_NO_ALLOC_MAX_BINS) {
        char msg[160];
        snprintf(msg, sizeof msg, "fredopt_volume_histogram_no_alloc: n_bins = %d exceeds FREDOPT_NO_ALLOC_MAX_BINS = %d (the fixed scratch)",
                 (int)n_bins, (int)FREDOPT_NO_ALLOC_MAX_BINS);
        return na_fail(msg);
    }
    unsigned long long* cnt = nullptr;
    const int rc = na_scratch(&cnt);
    if (rc != FREDOPT_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_na_clear<<<(n_bins + 1 + NA_THREADS - 1) / NA_THREADS, NA_THREADS, 0, st>>>(cnt, n_bins + 1);
    if (n_voxels > 0) {
        long long g = (n_voxels + NA_THREADS - 1) / NA_THREADS;
        if (g > 148 * 8) g = 148 * 8;                              // 8 CTAs per SM; each CTA strides over n / grid <= 2^31 voxels
        const long long gmin = (n_voxels >> 31) + 1;               // ... for any n_voxels the C-ABI can express on one GPU
        if (g < gmin) g = gmin;
        k_na_count<<<(unsigned)g, NA_THREADS, 0, st>>>((long long)n_voxels, values, labels, (int)label, (int)n_bins, vmax, cnt);
    }
    k_na_finish<<<1, 1024, 0, st>>>(cnt, (int)n_bins, hist, (long long*)n_in_structure);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { g_last_cuda_error = std::string("fredopt_volume_histogram_no_alloc launch: ") + cudaGetErrorString(e); return FREDOPT_CUDA_ERROR; }
    return FREDOPT_OK;
}

}  // extern "C"
