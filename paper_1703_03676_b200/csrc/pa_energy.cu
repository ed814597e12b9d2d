// pa_energy.cu -- per-replica energy and magnetisation from the packed words (
// PAPER.md Eq. 10).  The paper unpacks the bits ("quite costly", L305); here the 32
// replicas of a word are counted in parallel with bit-sliced (vertical) counters:
//   unsat_j = number of bonds (right, down) with anti-parallel ends,  E_j = 2*unsat_j - 2N,
//   up_j    = number of up spins,                                       M_j = 2*up_j - N.
// One CTA per group; each thread folds its words into carry-save counters (Harley-Seal blocks of 8),
// the warp adds the 32 threads' counters with a bit-sliced ripple adder over shuffles, lane b then
// extracts replica b's count, and the warps' results are summed in shared memory.
#include "pa_common.cuh"
#include <stddef.h>

#define PA_EPLANES 20   // counts up to 2N = 2^19 (L = 512)

__device__ __forceinline__ void pa_csa(uint32_t& h, uint32_t& l, uint32_t a, uint32_t b, uint32_t c) {
    uint32_t u = a ^ b;
    h = (a & b) | (u & c);
    l = u ^ c;
}

struct BitCounter {          // per-thread bit-sliced counter: planes[k] holds bit k of 32 counts
    uint32_t ones, twos, fours;
    uint32_t hi[PA_EPLANES - 3];   // planes 3..
    __device__ __forceinline__ void clear() {
        ones = twos = fours = 0;
#pragma unroll
        for (int k = 0; k < PA_EPLANES - 3; ++k) hi[k] = 0;
    }
    // add eight 1-bit-per-lane inputs
    __device__ __forceinline__ void add8(const uint32_t x[8]) {
        uint32_t tA, tB, fA, fB, e;
        pa_csa(tA, ones, ones, x[0], x[1]);
        pa_csa(tB, ones, ones, x[2], x[3]);
        pa_csa(fA, twos, twos, tA, tB);
        pa_csa(tA, ones, ones, x[4], x[5]);
        pa_csa(tB, ones, ones, x[6], x[7]);
        pa_csa(fB, twos, twos, tA, tB);
        pa_csa(e, fours, fours, fA, fB);
        // ripple the eights into the upper planes (per-thread counts stay below 2^12)
#pragma unroll
        for (int k = 0; k < 9; ++k) { uint32_t t = hi[k] & e; hi[k] ^= e; e = t; }
    }
    __device__ __forceinline__ uint32_t plane(int k) const {
        return k == 0 ? ones : k == 1 ? twos : k == 2 ? fours : hi[k - 3];
    }
};

// Sum the bit-sliced counters of the 32 threads of a warp; afterwards every lane holds the warp total.
__device__ __forceinline__ void pa_warp_add_planes(uint32_t p[PA_EPLANES]) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < PA_EPLANES; ++k) {
            uint32_t b = __shfl_xor_sync(0xffffffffu, p[k], off);
            uint32_t u = p[k] ^ b;
            uint32_t s = u ^ carry;
            carry = (p[k] & b) | (u & carry);
            p[k] = s;
        }
    }
}

// The kernel also folds in everything else that is measured from (E_j, M_j) -- the paper's energyKer +
// CalcAverages (L173) and the first stage of QKer's range (our E_min, O5) -- so that a temperature step
// needs one launch and one device-to-host read for its observables:
//   exact integer sums  SE = sum E, SE2 = sum E^2, SA = sum |M|, SM2 = sum M^2   (order-independent atomics),
//   m_min / m_max of m = (E + 2N)/4                                             (atomicMax, order-independent),
//   sum_j (M_j/N)^4 in the TREE1024 order (O5, O8): the warp that finishes a group holds one replica per lane,
//   so its __shfl_down tree IS the aligned-run-of-32 level; the run sums go to runsum[g], and the last CTA
//   to finish (atomic ticket) does the tree over each 32 run sums and the sequential sum over 1024-blocks.
__global__ void __launch_bounds__(256)
pa_measure_kernel(const uint32_t* __restrict__ pop, int L, int N, long long R_cur,
                  int32_t* __restrict__ E, int32_t* __restrict__ M, PaScalars* __restrict__ sc,
                  double* __restrict__ runsum, double* __restrict__ blocksum) {
    const long long g = blockIdx.x;
    const uint32_t* base = pop + g * (long long)N;
    const int Lh = L >> 1, half = N >> 1;
    const int T = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    BitCounter cE, cM;
    cE.clear(); cM.clear();
    for (int b0 = tid * 8; b0 < N; b0 += T * 8) {
        uint32_t xa[8], xb[8], xs[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            int idx = b0 + q;
            uint32_t s = 0, a = 0, b = 0;
            if (idx < N) {
                int c = idx >= half ? 1 : 0;
                int rem = idx - c * half;
                int y = rem / Lh, xh = rem - y * Lh;
                int p = (y + c) & 1;
                const uint32_t* oth = base + (1 - c) * half;
                s = base[idx];
                // right neighbour (x+1, y): other colour, same row; down neighbour (x, y+1)
                int xr = p ? (xh + 1 == Lh ? 0 : xh + 1) : xh;
                int yd = (y + 1 == L) ? 0 : y + 1;
                a = s ^ oth[y * Lh + xr];
                b = s ^ oth[yd * Lh + xh];
            }
            xs[q] = s; xa[q] = a; xb[q] = b;
        }
        cE.add8(xa); cE.add8(xb); cM.add8(xs);
    }
    __shared__ int sE[8][32], sM[8][32];
    __shared__ bool s_last;
    uint32_t p[PA_EPLANES];
#pragma unroll
    for (int k = 0; k < PA_EPLANES; ++k) p[k] = cE.plane(k);
    pa_warp_add_planes(p);
    int vE = 0;
#pragma unroll
    for (int k = 0; k < PA_EPLANES; ++k) vE += (int)((p[k] >> lane) & 1u) << k;
#pragma unroll
    for (int k = 0; k < PA_EPLANES; ++k) p[k] = cM.plane(k);
    pa_warp_add_planes(p);
    int vM = 0;
#pragma unroll
    for (int k = 0; k < PA_EPLANES; ++k) vM += (int)((p[k] >> lane) & 1u) << k;
    sE[warp][lane] = vE; sM[warp][lane] = vM;
    __syncthreads();
    if (warp == 0) {
        int nw = T >> 5, unsat = 0, up = 0;
        for (int w = 0; w < nw; ++w) { unsat += sE[w][lane]; up += sM[w][lane]; }
        const long long j = g * 32 + lane;
        const bool live = j < R_cur;
        const int e = 2 * unsat - 2 * N, m = 2 * up - N;
        if (live) { E[j] = e; M[j] = m; }
        long long se = live ? e : 0, se2 = live ? (long long)e * e : 0, sa = live ? (m < 0 ? -m : m) : 0, sm2 = live ? (long long)m * m : 0;
        unsigned mlo = live ? 0xffffffffu - (unsigned)unsat / 2u : 0u;      // m = (E + 2N)/4 = unsat/2; max of (2^32-1 - m) = min m
        unsigned mhi = live ? (unsigned)unsat / 2u : 0u;
        double v = 0.0;
        if (live) {
            const double mm = __ddiv_rn((double)m, (double)N);
            const double m2 = __dmul_rn(mm, mm);
            v = __dmul_rn(m2, m2);
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            se += __shfl_xor_sync(0xffffffffu, se, off);
            se2 += __shfl_xor_sync(0xffffffffu, se2, off);
            sa += __shfl_xor_sync(0xffffffffu, sa, off);
            sm2 += __shfl_xor_sync(0xffffffffu, sm2, off);
            mlo = max(mlo, __shfl_xor_sync(0xffffffffu, mlo, off));
            mhi = max(mhi, __shfl_xor_sync(0xffffffffu, mhi, off));
            v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));         // TREE1024, run-of-32 level
        }
        if (lane == 0) {
            atomicAdd((unsigned long long*)&sc->SE, (unsigned long long)se);
            atomicAdd((unsigned long long*)&sc->SE2, (unsigned long long)se2);
            atomicAdd((unsigned long long*)&sc->SA, (unsigned long long)sa);
            atomicAdd((unsigned long long*)&sc->SM2, (unsigned long long)sm2);
            atomicMax(&sc->mmin_inv, mlo);
            atomicMax(&sc->mmax, mhi);
            runsum[g] = v;
            __threadfence();
            s_last = atomicAdd(&sc->done_counter, 1u) == gridDim.x - 1;
        }
    }
    __syncthreads();
    if (!s_last) return;
    // ---- last CTA: second and third level of TREE1024 over the run sums ----
    __threadfence();
    const long long G = gridDim.x;
    const int nblk = (int)((G + 31) / 32);
    for (int blk = warp; blk < nblk; blk += (T >> 5)) {
        const long long i = (long long)blk * 32 + lane;
        double v = i < G ? __ldcg(runsum + i) : 0.0;
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));
        if (lane == 0) blocksum[blk] = v;
    }
    __syncthreads();
    if (tid == 0) {
        double total = 0.0;
        for (int i = 0; i < nblk; ++i) total = __dadd_rn(total, blocksum[i]);   // ascending block index
        sc->m4sum = total;
    }
}

int pa_launch_measure(pa_handle* h) {
    const int64_t G = (h->R_cur + 31) / 32;
    int T = 256;
    while (T > 32 && T * 8 > h->N) T >>= 1;
    PA_CUDA(h, cudaMemsetAsync(h->d_scal, 0, offsetof(PaScalars, R_new), h->stream));
    pa_measure_kernel<<<(unsigned)G, T, 0, h->stream>>>(h->spins[h->cur], h->L, h->N, h->R_cur, h->E, h->M, h->d_scal,
                                                        h->runsum, h->partials);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    h->em_valid = true;
    h->host_scal_valid = false;
    return PA_OK;
}
