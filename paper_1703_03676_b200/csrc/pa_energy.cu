// pa_energy.cu -- per-replica energy and magnetisation from the packed words (
// PAPER.md Eq. 10).  The paper unpacks the bits ("quite costly", L305); here the 32
// replicas of a word are counted in parallel with bit-sliced (vertical) counters:
//   unsat_j = number of bonds (right, down) with anti-parallel ends,  E_j = 2*unsat_j - 2N,
//   up_j    = number of up spins,                                       M_j = 2*up_j - N.
// One CTA per group; each thread folds its words into carry-save counters (Harley-Seal blocks of 8),
// the warp adds the 32 threads' counters with a bit-sliced ripple adder over shuffles, lane b then
// extracts replica b's count, and the warps' results are summed in shared memory.
#include "pa_common.cuh"

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

__global__ void __launch_bounds__(256)
pa_energy_kernel(const uint32_t* __restrict__ pop, int L, int N, long long R_cur,
                 int32_t* __restrict__ E, int32_t* __restrict__ M) {
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
        long long j = g * 32 + lane;
        if (j < R_cur) { E[j] = 2 * unsat - 2 * N; M[j] = 2 * up - N; }
    }
}

int pa_launch_energy(pa_handle* h) {
    const int64_t G = (h->R_cur + 31) / 32;
    int T = 256;
    while (T > 32 && T * 8 > h->N) T >>= 1;
    pa_energy_kernel<<<(unsigned)G, T, 0, h->stream>>>(h->spins[h->cur], h->L, h->N, h->R_cur, h->E, h->M);
    PA_CUDA(h, cudaGetLastError());
    h->launches += 1;
    h->em_valid = true;
    return PA_OK;
}
