// pa_static.cu -- pa_weighted_average_static: the weighted average of M independent runs (Sec. 2.2, Eq. 6-7,
// PAPER.md L99-L109; reading O13) for callers that must not allocate.
//
// Who that is.  pa_weighted_average stages its host arguments through a cudaMalloc'd buffer and frees it again.  That
// is the wrong tool (a) for a program that has already handed the GPU's memory out -- populations sized to fill the
// 180 GB, or a host framework whose caching pool owns whatever is left -- where an allocation at temperature step
// 300 of 500 can simply fail; (b) for a program that combines its runs at every temperature while other handles are
// sweeping on other streams: cudaMalloc and cudaFree are device-wide synchronisation points, so each call would
// stall every one of those streams; and (c) for code that runs where blocking on the driver's allocator is not
// allowed at all (a host callback on a stream, a latency-bounded service loop).  For them this file gives ONE entry
// point that calls no cudaMalloc, no cudaFree and no library routine that allocates: inputs and outputs are the
// caller's device buffers, and the one piece of scratch the kernel needs -- the normalised weights omega_m, which it
// writes and reads back -- lives in the file-scope array below.
//
// The price.  The array has a fixed size, PA_WAVG_STATIC_MAX_RUNS doubles = 32 KiB, which every GPU that loads this
// library holds until the process exits.  All calls on one GPU share it, and it keeps what the last call left there.
// Nothing in it has to start at zero (a call writes omega_0 .. omega_{M-1} before it reads them and touches nothing
// beyond), so there is no clearing step; but two calls that overlap on the same GPU (different streams, or different
// host threads on different streams) race on it and both results are then garbage.  Serialise them: one stream, or
// an event between them.
#include "../../include/pa.h"
#include <cuda_runtime.h>
#include <math.h>
#include <mutex>

static_assert(PA_WAVG_STATIC_MAX_RUNS == 4096, "pa.h states 4096 runs = 32 KiB; keep the two in step");

// The scratch itself.  NOTE for whoever edits the host code below: in host code this name is only the host-side
// shadow of the symbol, not a device address -- a kernel handed `pa_wavg_static_omega` directly would fault (or, on a
// GPU that can reach host memory, quietly use the wrong bytes).  The address comes from cudaGetSymbolAddress.
static __device__ __align__(256) double pa_wavg_static_omega[PA_WAVG_STATIC_MAX_RUNS];

// Block-wide reduction in a fixed order (shuffle tree inside a warp, then over the warp leaders): the same order on
// every call, so the result does not depend on scheduling.  256 threads.
template <bool IS_MAX>
static __device__ __forceinline__ double block_reduce_256(double v, double* sh) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const double o = __shfl_down_sync(0xffffffffu, v, off);
        v = IS_MAX ? fmax(v, o) : v + o;
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < 8 ? sh[threadIdx.x] : (IS_MAX ? -INFINITY : 0.0);
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const double o = __shfl_down_sync(0xffffffffu, v, off);
            v = IS_MAX ? fmax(v, o) : v + o;
        }
        if (threadIdx.x == 0) sh[32] = v;
    }
    __syncthreads();
    return sh[32];
}

// Eq. 6-7: omega_m = exp(lnZ_m - max) / sum_m exp(lnZ_m - max),  A~_k = sum_m omega_m A[m][k].  One CTA of 256 threads.
// `omega` is the scratch: M doubles, written in the first phase, read in the second.
__global__ void __launch_bounds__(256)
pa_wavg_static_kernel(int M, const double* __restrict__ lnZ, const double* __restrict__ A, int nobs,
                      double* __restrict__ A_out, double* __restrict__ omega) {
    __shared__ double sh[33];
    double zmax = -INFINITY;
    for (int m = threadIdx.x; m < M; m += 256) zmax = fmax(zmax, lnZ[m]);
    zmax = block_reduce_256<true>(zmax, sh);
    double s = 0.0;
    for (int m = threadIdx.x; m < M; m += 256) s += exp(lnZ[m] - zmax);
    s = block_reduce_256<false>(s, sh);
    for (int m = threadIdx.x; m < M; m += 256) omega[m] = exp(lnZ[m] - zmax) / s;
    __syncthreads();                                   // the weights of all threads are visible to the CTA from here on
    for (int k = 0; k < nobs; ++k) {
        double acc = 0.0;
        for (int m = threadIdx.x; m < M; m += 256) acc += omega[m] * A[(size_t)m * nobs + k];
        acc = block_reduce_256<false>(acc, sh);
        if (threadIdx.x == 0) A_out[k] = acc;
    }
}

namespace {

constexpr int PA_STATIC_MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_omega_of_device[PA_STATIC_MAX_DEVICES];      // device address of the array on each GPU, nullptr = not looked up yet

// The device address of the scratch array on the CURRENT device; looked up once per device and remembered.
cudaError_t scratch_of_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < PA_STATIC_MAX_DEVICES;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (cached && g_omega_of_device[dev]) { *out = g_omega_of_device[dev]; return cudaSuccess; }
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, pa_wavg_static_omega);      // loads this file's device code on `dev` if need be
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (cached) g_omega_of_device[dev] = p;
    *out = p;
    return cudaSuccess;
}

// True if the CUDA runtime knows `p` as memory a kernel on the current device may touch (device or managed memory).
bool is_device_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int pa_weighted_average_static_max_runs(void) { return PA_WAVG_STATIC_MAX_RUNS; }

extern "C" int pa_weighted_average_static(int M, const double* d_lnZ, const double* d_A, int nobs, double* d_A_out,
                                          void* cuda_stream) {
    if (M < 1 || nobs < 0 || !d_lnZ || (nobs > 0 && (!d_A || !d_A_out))) return PA_ERR_INVALID_ARG;
    if (M > PA_WAVG_STATIC_MAX_RUNS) return PA_ERR_STATIC_LIMIT;     // more runs than the fixed array holds: use pa_weighted_average
    if (!is_device_pointer(d_lnZ) || (nobs > 0 && (!is_device_pointer(d_A) || !is_device_pointer(d_A_out))))
        return PA_ERR_INVALID_ARG;                                   // a host pointer would fault inside the kernel
    double* omega = nullptr;
    if (scratch_of_current_device(&omega) != cudaSuccess) { cudaGetLastError(); return PA_ERR_CUDA; }
    pa_wavg_static_kernel<<<1, 256, 0, (cudaStream_t)cuda_stream>>>(M, d_lnZ, d_A, nobs, d_A_out, omega);
    if (cudaGetLastError() != cudaSuccess) return PA_ERR_CUDA;
    return PA_OK;
}
