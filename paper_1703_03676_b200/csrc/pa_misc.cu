// pa_misc.cu -- initial population (a0), energy histogram and multi-histogram
// accumulation (a9), spin import/export, and the integer-pipe calibration kernels.
#include "pa_common.cuh"
#include <stdint.h>
#include <math.h>


// a0 (L55, L65; O1): word(g, s) = philox(s, g>>2, 0, TAG_INIT)[g&3]; lanes >= R are cleared.
__global__ void pa_init_kernel(uint32_t* __restrict__ pop, PaGeom L, int N, long long R, PhiloxKeys K) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long G = (R + 31) / 32;
    if (i >= G * N) return;
    const long long g = i / N;
    const int idx = (int)(i - g * N);
    const int s = pa_site_of_index(idx, L);
    uint4 x = pa_philox((uint32_t)s, (uint32_t)(g >> 2), 0u, PA_TAG_INIT, K);
    const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
    uint32_t w = xs[g & 3];
    const long long live = R - g * 32;
    if (live < 32) w &= (1u << live) - 1u;
    pop[i] = w;
}

int pa_launch_init(pa_handle* h) {
    const long long n = ((h->R_cur + 31) / 32) * (long long)h->N;
    pa_init_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(h->spins[h->cur], h->geom, h->N, h->R_cur, h->keys);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}

// a9 (Eq. 9; O9)
// also O14 (L129): the microcanonical magnetisation sums A1[m] += |M_j|, A2[m] += M_j^2 (exact integers, order-free)
// Privatised per CTA (three global atomics per replica into a few hundred hot bins): a CTA of 1024 threads takes up to
// PA_HIST_PER_CTA = 8192 replicas and accumulates the levels inside the window [m_min, m_min + PA_HIST_WIN) -- m_min from the
// measure kernel's device scalars -- in shared memory with native 32-bit atomics: the count, sum |M| (< 2^18 * 2^13) and M^2 in
// three 12-bit slices (M^2 < 2^36; each slice sum < 2^12 * 2^13), then flushes one global atomic per occupied level and sum.
// A level outside the window (a population spanning more than 4 PA_HIST_WIN in energy) goes to global atomics directly.
#define PA_HIST_WIN 2048
#define PA_HIST_PER_CTA 8192
__global__ void __launch_bounds__(1024)
pa_hist_kernel(const int32_t* __restrict__ E, const int32_t* __restrict__ M, long long R, int N /* nlev */, const PaScalars* __restrict__ sc,
               uint32_t* __restrict__ Hcur, unsigned long long* __restrict__ A1, unsigned long long* __restrict__ A2) {
    __shared__ uint32_t cnt[PA_HIST_WIN], s1[PA_HIST_WIN], q0[PA_HIST_WIN], q1[PA_HIST_WIN], q2[PA_HIST_WIN];
    for (int b = threadIdx.x; b < PA_HIST_WIN; b += blockDim.x) { cnt[b] = 0u; s1[b] = 0u; q0[b] = 0u; q1[b] = 0u; q2[b] = 0u; }
    __syncthreads();
    const int m_lo = (int)(0xffffffffu - sc->mmin_inv);
    const long long j0 = (long long)blockIdx.x * PA_HIST_PER_CTA, j1 = min(R, j0 + PA_HIST_PER_CTA);
    for (long long j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        const int m = (E[j] + 2 * N) >> 2;
        const long long mj = M[j];
        const unsigned long long a = (unsigned long long)(mj < 0 ? -mj : mj), a2 = a * a;
        const int b = m - m_lo;
        if (b >= 0 && b < PA_HIST_WIN) {
            atomicAdd(&cnt[b], 1u); atomicAdd(&s1[b], (uint32_t)a);
            atomicAdd(&q0[b], (uint32_t)(a2 & 0xfffu)); atomicAdd(&q1[b], (uint32_t)((a2 >> 12) & 0xfffu)); atomicAdd(&q2[b], (uint32_t)(a2 >> 24));
        } else { atomicAdd(&Hcur[m], 1u); atomicAdd(&A1[m], a); atomicAdd(&A2[m], a2); }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < PA_HIST_WIN; b += blockDim.x) {
        const uint32_t c = cnt[b];
        if (c) {
            atomicAdd(&Hcur[m_lo + b], c); atomicAdd(&A1[m_lo + b], (unsigned long long)s1[b]);
            atomicAdd(&A2[m_lo + b], (unsigned long long)q0[b] + ((unsigned long long)q1[b] << 12) + ((unsigned long long)q2[b] << 24));
        }
    }
}
__global__ void pa_hist_fold_kernel(uint32_t* __restrict__ Hcur, unsigned long long* __restrict__ Hsum,
                                    double* __restrict__ lnD, int N /* nlev */, double lnR_minus_lnZ, double beta, int e0) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m > N) return;
    Hsum[m] += Hcur[m];
    Hcur[m] = 0;
    const double Em = (double)(-2 * N + 4 * m + e0);
    const double term = lnR_minus_lnZ - beta * Em;
    const double a = lnD[m];
    double out;
    if (a == -INFINITY) out = term;
    else { const double hi = fmax(a, term), lo = fmin(a, term); out = hi + log1p(exp(lo - hi)); }
    lnD[m] = out;
}

int pa_launch_hist(pa_handle* h, double beta) {
    const long long blocks = (h->R_cur + PA_HIST_PER_CTA - 1) / PA_HIST_PER_CTA;
    pa_hist_kernel<<<(unsigned)blocks, 1024, 0, h->stream>>>(h->E, h->M, h->R_cur, h->nlev, h->d_scal, h->Hcur, h->A1, h->A2);
    const double c = log((double)h->R_cur) - h->lnZ;
    pa_hist_fold_kernel<<<(h->nlev + 1 + 255) / 256, 256, 0, h->stream>>>(h->Hcur, h->Hsum, h->lnD, h->nlev, c, beta, h->e0);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 2;
    return PA_OK;
}

// ------------------------------------------------------------------------------------------------
// O12 (Sec. 2.4, Eq. 9): canonical averages at any beta from the accumulated sums.
// ln Omega_m = ln Hsum[m] - lnD[m]; one CTA per beta; three passes over the N+1 levels (largest exponent,
// Z and <E>, variance about the mean) with fixed-shape block reductions (shuffle tree, then the tree over the
// warp results), so the result does not depend on scheduling.
// ------------------------------------------------------------------------------------------------
template <bool IS_MAX>
__device__ __forceinline__ double pa_block_reduce(double v, double* sh) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const double o = __shfl_down_sync(0xffffffffu, v, off);
        v = IS_MAX ? fmax(v, o) : v + o;
    }
    __syncthreads();                                   // sh may still be read from the previous reduction
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : (IS_MAX ? -INFINITY : 0.0);
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

__global__ void __launch_bounds__(256)
pa_reweight_kernel(const unsigned long long* __restrict__ Hsum, const double* __restrict__ lnD,
                   const unsigned long long* __restrict__ A1, const unsigned long long* __restrict__ A2, int N /* nlev */, int nsites, int e0,
                   const double* __restrict__ betas, double* __restrict__ lnZ, double* __restrict__ e, double* __restrict__ C,
                   double* __restrict__ absm, double* __restrict__ m2) {
    __shared__ double sh[33];
    const double beta = betas[blockIdx.x];
    double amax = -INFINITY;
    for (int m = threadIdx.x; m <= N; m += blockDim.x) {
        const unsigned long long H = Hsum[m];
        if (H == 0ull) continue;
        amax = fmax(amax, (log((double)H) - lnD[m]) - beta * (double)(-2 * N + 4 * m + e0));
    }
    amax = pa_block_reduce<true>(amax, sh);
    double s0 = 0.0, s1 = 0.0, sa = 0.0, sq = 0.0;
    for (int m = threadIdx.x; m <= N; m += blockDim.x) {
        const unsigned long long H = Hsum[m];
        if (H == 0ull) continue;
        const double Em = (double)(-2 * N + 4 * m + e0);
        const double p = exp(((log((double)H) - lnD[m]) - beta * Em) - amax);
        s0 += p; s1 += Em * p;
        sa += p * ((double)A1[m] / (double)H);           // O14: microcanonical mean of |M| at level m
        sq += p * ((double)A2[m] / (double)H);
    }
    s0 = pa_block_reduce<false>(s0, sh);
    s1 = pa_block_reduce<false>(s1, sh);
    sa = pa_block_reduce<false>(sa, sh);
    sq = pa_block_reduce<false>(sq, sh);
    const double mean = s1 / s0;
    double s2 = 0.0;
    for (int m = threadIdx.x; m <= N; m += blockDim.x) {
        const unsigned long long H = Hsum[m];
        if (H == 0ull) continue;
        const double Em = (double)(-2 * N + 4 * m + e0);
        const double p = exp(((log((double)H) - lnD[m]) - beta * Em) - amax);
        s2 += (Em - mean) * (Em - mean) * p;
    }
    s2 = pa_block_reduce<false>(s2, sh);
    if (threadIdx.x == 0) {
        lnZ[blockIdx.x] = amax + log(s0);
        e[blockIdx.x] = mean / (double)nsites;
        C[blockIdx.x] = beta * beta * (s2 / s0) / (double)nsites;
        absm[blockIdx.x] = (sa / s0) / (double)nsites;
        m2[blockIdx.x] = (sq / s0) / ((double)nsites * (double)nsites);
    }
}

// d_io: [betas(n) | lnZ(n) | e(n) | C(n) | absm(n) | m2(n)] in device memory
int pa_launch_reweight(pa_handle* h, int n, double* d_io) {
    const size_t z = (size_t)n;
    pa_reweight_kernel<<<n, 256, 0, h->stream>>>(h->Hsum, h->lnD, h->A1, h->A2, h->nlev, h->N, h->e0, d_io, d_io + z, d_io + 2 * z, d_io + 3 * z,
                                                 d_io + 4 * z, d_io + 5 * z);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}

// O13 (Sec. 2.2, Eq. 6-7): omega_m = exp(lnZ_m - max) / sum, A~_k = sum_m omega_m A[m][k].  One CTA.
__global__ void __launch_bounds__(256)
pa_wavg_kernel(int M, const double* __restrict__ lnZ, const double* __restrict__ A, int nobs,
               double* __restrict__ A_out, double* __restrict__ omega) {
    __shared__ double sh[33];
    double zmax = -INFINITY;
    for (int m = threadIdx.x; m < M; m += blockDim.x) zmax = fmax(zmax, lnZ[m]);
    zmax = pa_block_reduce<true>(zmax, sh);
    double s = 0.0;
    for (int m = threadIdx.x; m < M; m += blockDim.x) s += exp(lnZ[m] - zmax);
    s = pa_block_reduce<false>(s, sh);
    for (int m = threadIdx.x; m < M; m += blockDim.x) omega[m] = exp(lnZ[m] - zmax) / s;
    __syncthreads();
    for (int k = 0; k < nobs; ++k) {
        double acc = 0.0;
        for (int m = threadIdx.x; m < M; m += blockDim.x) acc += omega[m] * A[(size_t)m * nobs + k];
        acc = pa_block_reduce<false>(acc, sh);
        if (threadIdx.x == 0) A_out[k] = acc;
    }
}

cudaError_t pa_run_wavg(int M, const double* d_lnZ, const double* d_A, int nobs, double* d_out, double* d_omega, cudaStream_t st) {
    pa_wavg_kernel<<<1, 256, 0, st>>>(M, d_lnZ, d_A, nobs, d_out, d_omega);
    return cudaGetLastError();
}

// ---- spin export / import ------------------------------------------------------------------------
__global__ void pa_unpack_kernel(const uint32_t* __restrict__ pop, PaGeom L, int N, const long long* __restrict__ slots,
                                 long long j0, long long n, int8_t* __restrict__ out) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n * N) return;
    const long long r = i / N;
    const int s = (int)(i - r * N);
    const long long j = slots ? slots[r] : j0 + r;
    const uint32_t w = pop[(j >> 5) * N + pa_index_of_site(s, L)];
    out[i] = ((w >> (j & 31)) & 1u) ? 1 : -1;
}
__global__ void pa_pack_kernel(uint32_t* __restrict__ pop, PaGeom L, int N, long long j0, long long n, const int8_t* __restrict__ in) {
    // one thread per (group, site): rewrites the bits of replicas j0..j0+n-1 that fall in this word
    const long long g0 = j0 >> 5, g1 = (j0 + n - 1) >> 5;
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= (g1 - g0 + 1) * N) return;
    const long long g = g0 + i / N;
    const int s = (int)(i % N);
    const long long idx = g * N + pa_index_of_site(s, L);
    uint32_t w = pop[idx];
    for (int b = 0; b < 32; ++b) {
        const long long j = g * 32 + b;
        if (j >= j0 && j < j0 + n) {
            const uint32_t bit = in[(j - j0) * N + s] > 0 ? 1u : 0u;
            w = (w & ~(1u << b)) | (bit << b);
        }
    }
    pop[idx] = w;
}
// The sweep kernels flip all 32 lanes of the last group, so the resident lanes past the population hold arbitrary bits (every
// reader masks by j < R); the interchange words are canonical: dead lanes read as 0.
// One thread per PAIR of sites (x = 2 xh, 2 xh + 1) of a lattice row: in the interchange layout the pair is 8 contiguous bytes, in the
// resident layout its words sit at the same index (r, xh) of the two colour arrays -- which of the two takes the even x depends on the
// parity of y + z.  Both sides are coalesced (the first version moved one word per thread with a 64-bit division and a stride-2
// access: 1.7 TB/s; this one runs at the copy kernel's rate).  grid = (groups, pair blocks); V2: 8-byte accesses (aligned buffers).
template <bool V2>
__global__ void __launch_bounds__(256)
pa_words_out_kernel(const uint32_t* __restrict__ pop, PaGeom L, int N, long long R, uint32_t* __restrict__ out) {
    const long long g = blockIdx.x;
    const int pr = blockIdx.y * blockDim.x + threadIdx.x, half = N >> 1;
    if (pr >= half) return;
    const int Lh = L.Lx >> 1;
    const int r = pr / Lh, z = r / L.Ly, y = r - z * L.Ly;
    const int q = (y + z) & 1;                                   // colour 0 holds x = 2 xh + q
    const uint32_t* base = pop + g * (long long)N;
    uint32_t w0 = base[pr], w1 = base[half + pr];                // colour 0, colour 1
    const long long live = R - g * 32;
    if (live < 32) { const uint32_t m = (1u << live) - 1u; w0 &= m; w1 &= m; }
    const uint32_t we = q ? w1 : w0, wo = q ? w0 : w1;           // even x, odd x
    uint32_t* o = out + g * (long long)N + 2 * (long long)pr;
    if (V2) *reinterpret_cast<uint2*>(o) = make_uint2(we, wo);
    else { o[0] = we; o[1] = wo; }
}
template <bool V2>
__global__ void __launch_bounds__(256)
pa_words_in_kernel(uint32_t* __restrict__ pop, PaGeom L, int N, long long R, const uint32_t* __restrict__ in) {
    const long long g = blockIdx.x;
    const int pr = blockIdx.y * blockDim.x + threadIdx.x, half = N >> 1;
    if (pr >= half) return;
    const int Lh = L.Lx >> 1;
    const int r = pr / Lh, z = r / L.Ly, y = r - z * L.Ly;
    const int q = (y + z) & 1;
    const uint32_t* i2 = in + g * (long long)N + 2 * (long long)pr;
    uint32_t we, wo;
    if (V2) { const uint2 v = *reinterpret_cast<const uint2*>(i2); we = v.x; wo = v.y; }
    else { we = i2[0]; wo = i2[1]; }
    const long long live = R - g * 32;
    if (live < 32) { const uint32_t m = (1u << live) - 1u; we &= m; wo &= m; }
    uint32_t* base = pop + g * (long long)N;
    base[pr] = q ? wo : we;
    base[half + pr] = q ? we : wo;
}

int pa_launch_unpack(pa_handle* h, const int64_t* d_slots, int64_t j0, int64_t n, int8_t* d_out) {
    const long long tot = n * (long long)h->N;
    if (tot == 0) return PA_OK;
    pa_unpack_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, h->stream>>>(h->spins[h->cur], h->geom, h->N,
                                                                          (const long long*)d_slots, j0, n, d_out);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}
int pa_launch_pack(pa_handle* h, int64_t j0, int64_t n, const int8_t* d_in) {
    if (n == 0) return PA_OK;
    const long long ng = ((j0 + n - 1) >> 5) - (j0 >> 5) + 1;
    const long long tot = ng * h->N;
    pa_pack_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, h->stream>>>(h->spins[h->cur], h->geom, h->N, j0, n, d_in);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}
static bool pa_aligned8(const void* p) { return ((uintptr_t)p & 7u) == 0; }
static int pa_words_out_groups(pa_handle* h, const uint32_t* pop, long long R_rel, uint32_t* d_words) {
    const long long G = (R_rel + 31) / 32;
    if (G <= 0) return PA_OK;
    const dim3 grid((unsigned)G, (unsigned)((h->N / 2 + 255) / 256), 1);
    if (pa_aligned8(d_words)) pa_words_out_kernel<true><<<grid, 256, 0, h->stream>>>(pop, h->geom, h->N, R_rel, d_words);
    else pa_words_out_kernel<false><<<grid, 256, 0, h->stream>>>(pop, h->geom, h->N, R_rel, d_words);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}
int pa_launch_words_out(pa_handle* h, uint32_t* d_words) { return pa_words_out_groups(h, h->spins[h->cur], h->R_cur, d_words); }
int pa_launch_words_out_range(pa_handle* h, uint32_t* d_words, int64_t g0, int64_t ng) {
    long long R_rel = h->R_cur - 32 * g0;                       // the kernel counts groups and live lanes from its base pointers
    if (R_rel > 32 * ng) R_rel = 32 * ng;
    return pa_words_out_groups(h, h->spins[h->cur] + g0 * (long long)h->N, R_rel, d_words + g0 * (long long)h->N);
}
int pa_launch_words_in(pa_handle* h, int64_t R, const uint32_t* d_words) {
    const long long G = (R + 31) / 32;
    const dim3 grid((unsigned)G, (unsigned)((h->N / 2 + 255) / 256), 1);
    if (pa_aligned8(d_words)) pa_words_in_kernel<true><<<grid, 256, 0, h->stream>>>(h->spins[h->cur], h->geom, h->N, R, d_words);
    else pa_words_in_kernel<false><<<grid, 256, 0, h->stream>>>(h->spins[h->cur], h->geom, h->N, R, d_words);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return PA_OK;
}

// ---- integer-pipe calibration -------------------------------------------------
// Dependent chains with enough independent copies per thread to saturate a pipe; the result is
// written so nothing is optimised away.  Each loop iteration issues `PER_ITER` instructions of the kind.
template <int KIND>
__global__ void __launch_bounds__(256)
pa_calib_kernel(uint32_t* out, int iters, uint32_t seed, unsigned long long* cycles) {
    uint32_t a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed + threadIdx.x * 8 + i;
    unsigned long long q[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) q[i] = ((unsigned long long)a[i] << 32) | (seed * 2654435761u + i);
    uint32_t k = seed ^ 0x9E3779B9u;
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (KIND == 0) {                       // LOP3: 3-input xor chain (volatile: xor chains are linear and would be folded)
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) & 7]), "r"(k));
                } else if (KIND == 1) {                // IMAD.WIDE.U32 chain without addend, as in Philox: p = hi(p) * M0
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(q[i]) : "r"((uint32_t)(q[i] >> 32) | 1u), "r"(PA_PHILOX_M0));
                } else {                               // the Philox round mix: 2 IMAD.WIDE + 2 LOP3
                    uint32_t h0, l0, h1, l1;
                    pa_mulhilo(PA_PHILOX_M0, a[i], h0, l0);
                    pa_mulhilo(PA_PHILOX_M1, a[(i + 4) & 7], h1, l1);
                    a[i] = h1 ^ l0 ^ k;
                    a[(i + 4) & 7] = h0 ^ l1 ^ k;
                }
            }
        }
    }
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    uint32_t r = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r ^= a[i] ^ (uint32_t)q[i] ^ (uint32_t)(q[i] >> 32);
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0 && blockIdx.x == 0) { cycles[0] = (unsigned long long)(t1 - t0); cycles[1] = g1 - g0; }   // SM cycles, ns
}

int pa_run_calibrate(int kind, double* ginstr_per_ns, double* sm_mhz) {
    if (kind < 0 || kind > 2) return PA_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return PA_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // exactly one wave: as many CTAs per SM as are resident at once, so that block 0's cycle count spans the kernel
    const int threads = 256, iters = 4096;
    int per_sm = 0;
    cudaError_t oe = kind == 0 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pa_calib_kernel<0>, threads, 0)
                   : kind == 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pa_calib_kernel<1>, threads, 0)
                               : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pa_calib_kernel<2>, threads, 0);
    if (oe != cudaSuccess || per_sm < 1) return PA_ERR_CUDA;
    const int blocks = sms * per_sm;
    uint32_t* d_out = nullptr; unsigned long long* d_cyc = nullptr;
    if (cudaMalloc(&d_out, (size_t)blocks * threads * 4) != cudaSuccess) return PA_ERR_CUDA;
    if (cudaMalloc(&d_cyc, 16) != cudaSuccess) { cudaFree(d_out); return PA_ERR_CUDA; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    unsigned long long cyc[2] = {0, 1};
    for (int rep = 0; rep < 6; ++rep) {                 // the first launches also bring the clocks up
        cudaEventRecord(e0);
        if (kind == 0) pa_calib_kernel<0><<<blocks, threads>>>(d_out, iters, 12345u + rep, d_cyc);
        else if (kind == 1) pa_calib_kernel<1><<<blocks, threads>>>(d_out, iters, 12345u + rep, d_cyc);
        else pa_calib_kernel<2><<<blocks, threads>>>(d_out, iters, 12345u + rep, d_cyc);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d_out); cudaFree(d_cyc); return PA_ERR_CUDA; }
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 1 && ms < best) {
            best = ms;
            cudaMemcpy(cyc, d_cyc, 16, cudaMemcpyDeviceToHost);
        }
    }
    // instructions of the measured kind per thread per iteration
    const double per_iter = (kind == 2) ? 4.0 * 8.0 * 4.0 : 4.0 * 8.0;   // kind 2: 4 reps x 8 x (2 IMAD.WIDE + 2 LOP3)
    const double total = per_iter * (double)iters * (double)blocks * (double)threads;
    if (ginstr_per_ns) *ginstr_per_ns = total / ((double)best * 1e6);
    if (sm_mhz) *sm_mhz = cyc[1] ? (double)cyc[0] * 1e3 / (double)cyc[1] : 0.0;   // block 0: SM cycles per ns of the global timer
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_out); cudaFree(d_cyc);
    return PA_OK;
}
