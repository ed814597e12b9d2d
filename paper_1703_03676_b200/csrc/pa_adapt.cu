// pa_adapt.cu -- the adaptive temperature step (Sec. 2.3, Eq. 8) without 41 host
// round trips.
//
// O10 fixes WHAT is computed: alpha(dbeta) = TREE1024_j(min(1, R w_j / W)) / R_cur with host-libm weight tables, and 40
// bisection steps on alpha(mid) >= alpha*.  Every such decision must be the oracle's, bit for bit, or the beta sequence
// differs.  It does not fix how the decisions are reached.  alpha depends on the energies only through their histogram
// H[d] = #{j : (E_j - E_min)/4 = d}, so   alpha'(x) = sum_d H[d] min(1, R w'_d / W') / R_cur,  W' = sum_d H[d] w'_d,
// w'_d = exp(-(x (double)(4d))) -- dmax + 1 terms instead of R_cur -- equals the TREE1024 value up to rounding, and the
// rounding is bounded:  |alpha' - alpha| <= (2 R_cur + 2 dmax + 32) 2^-53  to first order.  The kernel
// below runs the whole bisection on the histogram in ONE launch and decides an iteration only when alpha'(mid) is further
// than B = 4 x that bound from alpha*; otherwise it stops and hands the iteration back to the host, which evaluates
// alpha(mid) exactly (weight table from libm, pa_tree_kernel<0>, pa_tree_kernel<1>) and relaunches from the next iteration.
// alpha' - alpha* shrinks by 2 per iteration while B ~ 1e-10, so about the last three of the 40 iterations are handed back:
// the result is identical to 41 exact evaluations (tests/test_parity_gpu.py::test_adaptive_filter_equals_exact_path and
// every step of the full cfg4 run), at a tenth of the round trips.
#include "pa_common.cuh"
#include <math.h>

// ---- count-only energy histogram of the current population, privatised per CTA in shared memory -------------------------
// Hd[m] += #{j : (E_j + 2N - e0)/4 = m}.  Bins inside the window [m_min, m_min + PA_HWIN) are counted in shared memory and
// flushed once per CTA; anything outside (never seen in practice: the window spans 4 PA_HWIN in energy) goes to global atomics.
#define PA_HWIN 4096
__global__ void __launch_bounds__(256)
pa_ehist_kernel(const int32_t* __restrict__ E, long long R, int N /* nlev */, int e0, const PaScalars* __restrict__ sc, uint32_t* __restrict__ Hd) {
    __shared__ uint32_t bins[PA_HWIN];
    for (int b = threadIdx.x; b < PA_HWIN; b += blockDim.x) bins[b] = 0u;
    __syncthreads();
    const int m_lo = (int)(0xffffffffu - sc->mmin_inv);
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < R; j += (long long)gridDim.x * blockDim.x) {
        const int m = (E[j] + 2 * N - e0) >> 2;
        const int b = m - m_lo;
        if (b >= 0 && b < PA_HWIN) atomicAdd(&bins[b], 1u); else atomicAdd(&Hd[m], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < PA_HWIN; b += blockDim.x) {
        const uint32_t c = bins[b];
        if (c) atomicAdd(&Hd[m_lo + b], c);
    }
}

// ---- the bisection on the histogram -------------------------------------------------------------------------------------
__device__ __forceinline__ double pa_block_sum_all(double v, double* sh) {      // every thread returns the same bits
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();                                                             // sh may still be read from the previous call
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = (threadIdx.x & 31) < (blockDim.x >> 5) ? sh[threadIdx.x & 31] : 0.0;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    return t;
}

// alpha'(x) from the histogram in shared memory (hs[d], d = 0..dmax) with the weights cached in ws[]
__device__ __forceinline__ double pa_alpha_hist(const uint32_t* hs, double* ws, int dmax, double x, double R_target, double R_cur, double* sh) {
    double acc = 0.0;
    for (int d = threadIdx.x; d <= dmax; d += blockDim.x) {
        const double w = exp(-(x * (double)(4 * d)));                            // the oracle's argument, the device's exp (<= 1 ulp)
        ws[d] = w;
        acc += (double)hs[d] * w;
    }
    const double W = pa_block_sum_all(acc, sh);
    acc = 0.0;
    for (int d = threadIdx.x; d <= dmax; d += blockDim.x) {
        const double tau = (R_target * ws[d]) / W;
        acc += (double)hs[d] * (tau < 1.0 ? tau : 1.0);
    }
    return pa_block_sum_all(acc, sh) / R_cur;
}

__global__ void __launch_bounds__(1024)
pa_adapt_kernel(const uint32_t* __restrict__ Hd, const PaScalars* __restrict__ sc, double R_target, double R_cur, double target,
                double bound, const PaAdaptState in, PaAdaptState* __restrict__ st) {
    // the bisection state comes in as a kernel argument and goes out into mapped host memory: no copy operation either way
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double sh[32];
    const int m_lo = (int)(0xffffffffu - sc->mmin_inv), dmax = (int)sc->mmax - m_lo;
    double lo = in.lo, hi = in.hi, margin = in.margin, a_last = 0.0;
    int it = in.it;
    if (dmax + 1 > PA_ADAPT_BINS) {                                              // wider than the shared-memory table: all exact
        if (threadIdx.x == 0) { st->lo = lo; st->hi = hi; st->it = it; st->status = it < 0 ? PA_ADAPT_AMBIG_FIRST : PA_ADAPT_AMBIG; st->margin = margin; st->a_last = target; }
        return;
    }
    double* ws = reinterpret_cast<double*>(smem_raw);
    uint32_t* hs = reinterpret_cast<uint32_t*>(ws + PA_ADAPT_BINS);
    for (int d = threadIdx.x; d <= dmax; d += blockDim.x) hs[d] = Hd[m_lo + d];
    __syncthreads();
    int status = PA_ADAPT_DONE;
    if (it < 0) {                                                                // O10: if alpha(hi) >= alpha* return hi
        const double a = pa_alpha_hist(hs, ws, dmax, hi, R_target, R_cur, sh);
        if (a >= target + bound) status = PA_ADAPT_RETURN_HI;
        else if (a < target - bound) it = 0;
        else { status = PA_ADAPT_AMBIG_FIRST; a_last = a; }
        if (status != PA_ADAPT_AMBIG_FIRST) margin = fmin(margin, fabs(a - target) / bound);
    }
    if (status == PA_ADAPT_DONE) {
        for (; it < 40; ++it) {                                                  // O10: exactly 40 bisection steps
            const double mid = 0.5 * (lo + hi);
            const double a = pa_alpha_hist(hs, ws, dmax, mid, R_target, R_cur, sh);
            if (a >= target + bound) lo = mid;
            else if (a < target - bound) hi = mid;
            else { status = PA_ADAPT_AMBIG; a_last = a; break; }
            margin = fmin(margin, fabs(a - target) / bound);
        }
    }
    if (threadIdx.x == 0) { st->lo = lo; st->hi = hi; st->it = it; st->status = status; st->margin = margin; st->a_last = a_last; }
}

int pa_launch_ehist(pa_handle* h) {
    PA_CUDA(h, cudaMemsetAsync(h->Hd, 0, ((size_t)h->nlev + 1) * 4, h->stream));
    long long blocks = (h->R_cur + 256 * 16 - 1) / (256 * 16);
    if (blocks > 2 * h->n_sm) blocks = 2 * h->n_sm;
    if (blocks < 1) blocks = 1;
    pa_ehist_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->E, h->R_cur, h->nlev, h->e0, h->d_scal, h->Hd);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}

// One launch of the bisection filter from the state *h->h_adapt (pinned), result back in the same place.  Synchronises.
int pa_run_adapt_filter(pa_handle* h, double target, double bound) {
    const size_t smem = (size_t)PA_ADAPT_BINS * (8 + 4);
    PA_CUDA(h, cudaFuncSetAttribute(pa_adapt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    pa_adapt_kernel<<<1, 1024, smem, h->stream>>>(h->Hd, h->d_scal, (double)h->R_target, (double)h->R_cur, target, bound, *h->h_adapt,
                                                  h->h_adapt_dev);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    PA_CUDA(h, cudaStreamSynchronize(h->stream));
    return PA_OK;
}
