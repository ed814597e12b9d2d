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
#include <stdlib.h>

#define PA_EPLANES 20   // bit planes of the per-replica counters: counts up to 2N = 2^19 (L = 512) on the square lattice and up to
                        // 3N = 3 * 2^18 on the largest cubic box (pa_create_box: at most 2^18 sites)
static_assert(3 * (1 << 18) < (1 << PA_EPLANES), "the energy counters of the largest cubic box must fit PA_EPLANES bit planes");

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
template <int NPL>
__device__ __forceinline__ void pa_warp_add_planes(uint32_t (&p)[NPL]) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < NPL; ++k) {
            uint32_t b = __shfl_xor_sync(0xffffffffu, p[k], off);
            uint32_t u = p[k] ^ b;
            uint32_t s = u ^ carry;
            carry = (p[k] & b) | (u & carry);
            p[k] = s;
        }
    }
}

// Everything after the per-thread bit-sliced counters, shared by both measure kernels.  pe / pm hold NPL planes
// of the thread's unsatisfied-bond and up-spin counts (bit b of plane k = bit k of replica b's count).
template <int NPL>
__device__ __forceinline__ void pa_measure_tail(uint32_t (&pe)[NPL], uint32_t (&pm)[NPL], long long g, int N, int nlev, long long R_cur,
                                                int32_t* __restrict__ E, int32_t* __restrict__ M, PaScalars* __restrict__ sc,
                                                double* __restrict__ runsum, double* __restrict__ blocksum, PaScalars* __restrict__ snap) {
    const int T = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ int sE[8][32], sM[8][32];
    __shared__ bool s_last;
    pa_warp_add_planes<NPL>(pe);
    int vE = 0;
#pragma unroll
    for (int k = 0; k < NPL; ++k) vE += (int)((pe[k] >> lane) & 1u) << k;
    pa_warp_add_planes<NPL>(pm);
    int vM = 0;
#pragma unroll
    for (int k = 0; k < NPL; ++k) vM += (int)((pm[k] >> lane) & 1u) << k;
    sE[warp][lane] = vE; sM[warp][lane] = vM;
    __syncthreads();
    if (warp == 0) {
        int nw = T >> 5, unsat = 0, up = 0;
        for (int w = 0; w < nw; ++w) { unsat += sE[w][lane]; up += sM[w][lane]; }
        const long long j = g * 32 + lane;
        const bool live = j < pa_live_R(R_cur, sc);
        const int e = 2 * unsat - 2 * nlev, m = 2 * up - N;          // E = 2 unsat - (number of bonds), M = 2 up - N
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
    for (int blk0 = warp * 8; blk0 < nblk; blk0 += (T >> 5) * 8) {       // 8 blocks of 32 run sums in flight per warp
        double v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const long long i = (long long)(blk0 + u) * 32 + lane;
            v[u] = i < G ? __ldcg(runsum + i) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) v[u] = __dadd_rn(v[u], __shfl_down_sync(0xffffffffu, v[u], off));
            if (lane == 0 && blk0 + u < nblk) blocksum[blk0 + u] = v[u];
        }
    }
    __syncthreads();
    if (tid == 0) {
        double total = 0.0;
        for (int i = 0; i < nblk; ++i) total = __dadd_rn(total, blocksum[i]);   // ascending block index
        sc->m4sum = total;
        if (snap) {                                                      // pa_anneal: this step's scalars, complete now
            const unsigned long long* s8 = reinterpret_cast<const unsigned long long*>(sc);
            unsigned long long* d8 = reinterpret_cast<unsigned long long*>(snap);
#pragma unroll
            for (int i = 0; i < (int)(sizeof(PaScalars) / 8); ++i) d8[i] = __ldcg(s8 + i);
            snap->m4sum = total;
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
// LOG_LH, LOG_LY >= 0: Lx/2 and Ly are these powers of two (cubes: shifts instead of two integer divisions per word); -1: any.
template <int LOG_LH, int LOG_LY>
__global__ void __launch_bounds__(256)
pa_measure_generic_kernel(const uint32_t* __restrict__ pop, PaGeom geo, int N, long long R_cur,
                  int32_t* __restrict__ E, int32_t* __restrict__ M, PaScalars* __restrict__ sc,
                  double* __restrict__ runsum, double* __restrict__ blocksum, const uint8_t* __restrict__ jmask,
                  PaScalars* __restrict__ snap, int nlev) {
    pa_pdl_wait(); pa_pdl_launch();
    const long long g = blockIdx.x;
    const uint32_t* base = pop + g * (long long)N;
    const int Lh = LOG_LH >= 0 ? (1 << LOG_LH) : geo.Lx >> 1, Ly = LOG_LY >= 0 ? (1 << LOG_LY) : geo.Ly, Lz = geo.Lz, half = N >> 1;
    const int T = blockDim.x, tid = threadIdx.x;
    BitCounter cE, cM;
    cE.clear(); cM.clear();
    for (int b0 = tid * 8; b0 < N; b0 += T * 8) {
        uint32_t xa[8], xb[8], xc[8], xs[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            int idx = b0 + q;
            uint32_t s = 0, a = 0, b = 0, cz = 0;
            if (idx < N) {
                int c = idx >= half ? 1 : 0;
                int rem = idx - c * half;
                int r = LOG_LH >= 0 ? (rem >> LOG_LH) : rem / Lh, xh = rem - r * Lh;          // row r = z*Ly + y (z = 0 on the square lattice)
                int z = LOG_LY >= 0 ? (r >> LOG_LY) : r / Ly, y = r - z * Ly;
                int p = (y + z + c) & 1;
                const uint32_t* oth = base + (1 - c) * half;
                s = base[idx];
                // every site owns its +x, +y (and, O16, +z) bond: right neighbour (x+1): other colour, same row;
                // an edge of length 2 makes the bond a double bond, owned by both of its sites
                int xr = p ? (xh + 1 == Lh ? 0 : xh + 1) : xh;
                int yd = (y + 1 == Ly) ? 0 : y + 1;
                a = s ^ oth[r * Lh + xr];
                b = s ^ oth[(z * Ly + yd) * Lh + xh];
                if (Lz > 1) { int zd = (z + 1 == Lz) ? 0 : z + 1; cz = s ^ oth[(zd * Ly + y) * Lh + xh]; }
                if (jmask) {                     // O15: a J = -1 bond is unsatisfied when its ends are parallel
                    const uint32_t j = jmask[idx];
                    a ^= 0u - ((j >> 4) & 1u);   // right bond
                    b ^= 0u - ((j >> 3) & 1u);   // down bond
                }
            }
            xs[q] = s; xa[q] = a; xb[q] = b; xc[q] = cz;
        }
        cE.add8(xa); cE.add8(xb); cM.add8(xs);
        if (Lz > 1) cE.add8(xc);
    }
    uint32_t pe[PA_EPLANES], pm[PA_EPLANES];
#pragma unroll
    for (int k = 0; k < PA_EPLANES; ++k) { pe[k] = cE.plane(k); pm[k] = cM.plane(k); }
    pa_measure_tail<PA_EPLANES>(pe, pm, g, N, nlev, R_cur, E, M, sc, runsum, blocksum, snap);
}


// ------------------------------------------------------------------------------------------------
// Fast path for L = 8, 16, ..., 256 (powers of two; every BASELINE.json config).
// A thread owns one quad column (four consecutive xh of both colours = two uint4 per lattice row) and walks
// down RS rows; lanes of a warp hold consecutive quads of a row (QPR = L/8 quads per row), so the one word a
// row's horizontal bonds need from the next quad comes from a shuffle, and the row below is the thread's own
// next load: every word is read from memory exactly once (plus one extra row per strip), two rows ahead of
// its use.  Per row and thread: 16 bond words -> one 16-input carry-save block, 8 spin words -> one 8-input
// block; about 12 instructions per word against 82 in the generic kernel, which made it ALU-bound
// (profiles/r01b_summary.md).
// ------------------------------------------------------------------------------------------------
template <int NP>
struct PlaneCounter {           // planes[k] holds bit k of 32 per-lane counts, counts < 2^NP
    uint32_t pl[NP];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int k = 0; k < NP; ++k) pl[k] = 0;
    }
    // ripple a carry word of weight 2^K0 into the planes K0..NP-1
    template <int K0>
    __device__ __forceinline__ void ripple(uint32_t e) {
#pragma unroll
        for (int k = K0; k < NP; ++k) { const uint32_t t = pl[k] & e; pl[k] ^= e; e = t; }
    }
    __device__ __forceinline__ uint32_t block8(const uint32_t* x) {     // returns the weight-8 carry
        uint32_t tA, tB, fA, fB, e;
        pa_csa(tA, pl[0], pl[0], x[0], x[1]);
        pa_csa(tB, pl[0], pl[0], x[2], x[3]);
        pa_csa(fA, pl[1], pl[1], tA, tB);
        pa_csa(tA, pl[0], pl[0], x[4], x[5]);
        pa_csa(tB, pl[0], pl[0], x[6], x[7]);
        pa_csa(fB, pl[1], pl[1], tA, tB);
        pa_csa(e, pl[2], pl[2], fA, fB);
        return e;
    }
    __device__ __forceinline__ void add8(const uint32_t* x) { ripple<3>(block8(x)); }
    // the weight-16 carry of sixteen inputs (planes 0..3 absorb the rest)
    __device__ __forceinline__ uint32_t block16(const uint32_t* x) {
        const uint32_t e1 = block8(x), e2 = block8(x + 8);
        uint32_t s;
        pa_csa(s, pl[3], pl[3], e1, e2);
        return s;
    }
    // Eight carries of weight 2^K0 (one per row of a block of eight rows) folded in by a carry-save ladder: seven full adders and ONE
    // ripple per eight rows instead of a ripple through all upper planes per row (the ripple was a quarter of the kernel's instructions)
    template <int K0>
    __device__ __forceinline__ void ladder8(const uint32_t* c) {
        uint32_t a, b, d, e, f, g2, h;
        pa_csa(a, pl[K0], pl[K0], c[0], c[1]);
        pa_csa(b, pl[K0], pl[K0], c[2], c[3]);
        pa_csa(d, pl[K0], pl[K0], c[4], c[5]);
        pa_csa(e, pl[K0], pl[K0], c[6], c[7]);
        pa_csa(f, pl[K0 + 1], pl[K0 + 1], a, b);
        pa_csa(g2, pl[K0 + 1], pl[K0 + 1], d, e);
        pa_csa(h, pl[K0 + 2], pl[K0 + 2], f, g2);
        ripple<K0 + 3>(h);
    }
    __device__ __forceinline__ void add16(const uint32_t* x) {
        const uint32_t e1 = block8(x), e2 = block8(x + 8);
        uint32_t s;
        pa_csa(s, pl[3], pl[3], e1, e2);
        ripple<4>(s);
    }
};

__host__ __device__ constexpr int pa_msr_threads(int L) { return (L * L / 8 >= 64) ? 64 : 32; }
__host__ __device__ constexpr int pa_msr_strips(int L) { return (pa_msr_threads(L) / (L / 8) < L) ? pa_msr_threads(L) / (L / 8) : L; }
__host__ __device__ constexpr int pa_bits(int v) { return v <= 1 ? 1 : 1 + pa_bits(v >> 1); }

// HASJ (O15): jm16[y * QPR + q] carries one bit per bond word of the row (bit i <-> xb[i] below): J = -1 on that bond,
// so the word is complemented (a negative bond is unsatisfied when its ends are parallel).
template <int LOG_QPR, bool HASJ>
__global__ void __launch_bounds__(64)
pa_measure_kernel(const uint32_t* __restrict__ pop, int N, long long R_cur,
                  int32_t* __restrict__ E, int32_t* __restrict__ M, PaScalars* __restrict__ sc,
                  double* __restrict__ runsum, double* __restrict__ blocksum, const uint16_t* __restrict__ jm16,
                  PaScalars* __restrict__ snap) {
    constexpr int QPR = 1 << LOG_QPR, L = 8 * QPR, Lq = L / 8;          // Lq = uint4 per colour row
    constexpr int S = pa_msr_strips(L), RS = L / S;                      // strips per group, rows per strip
    constexpr int NPE = pa_bits(16 * RS), NPM = pa_bits(8 * RS);         // planes per thread
    constexpr int NPW = NPE + 5;                                         // planes after the warp sum
    pa_pdl_wait(); pa_pdl_launch();
    const long long g = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool act = tid < S * QPR;
    const int q = tid & (QPR - 1), strip = act ? (tid >> LOG_QPR) : 0;
    const uint4* c0 = reinterpret_cast<const uint4*>(pop + g * (long long)N);
    const uint4* c1 = c0 + (N >> 3);
    const int y0 = strip * RS;
    const int nxt_lane = (lane & ~(QPR - 1)) | ((lane + 1) & (QPR - 1));  // next quad of the same row (periodic)
    const uint4 zero = make_uint4(0, 0, 0, 0);
    PlaneCounter<NPE> cE; PlaneCounter<NPM> cM;
    cE.clear(); cM.clear();
    uint4 a = zero, b = zero, na = zero, nb = zero;
    if (act) {
        a = __ldg(c0 + y0 * Lq + q); b = __ldg(c1 + y0 * Lq + q);
        const int y1 = (y0 + 1) & (L - 1);
        na = __ldg(c0 + y1 * Lq + q); nb = __ldg(c1 + y1 * Lq + q);
    }
    constexpr bool LADDER = RS % 8 == 0 && NPE >= 7 && NPM >= 6;        // L >= 64
    uint32_t ce[8], cm[8];                                                // the rows' top carries, folded in every eight rows
#pragma unroll 8
    for (int r = 0; r < RS; ++r) {
        const int y = y0 + r;
        uint4 fa = zero, fb = zero;                                       // row y + 2, in flight while row y is counted
        if (act && r + 1 < RS) {
            const int y2 = (y + 2) & (L - 1);
            fa = __ldg(c0 + y2 * Lq + q); fb = __ldg(c1 + y2 * Lq + q);
        }
        // colour-0 sites of row y sit at x = 2 xh + (y & 1): the bond to the right of the odd-x site of a pair
        // leads into the next xh of the other colour
        const bool odd = (y & 1) != 0;
        const uint4 t = odd ? b : a, u = odd ? a : b;                     // bond u[xh] - t[xh + 1]
        const uint32_t tn = __shfl_sync(0xffffffffu, t.x, nxt_lane);
        uint32_t xb[16];
        xb[0] = a.x ^ b.x; xb[1] = a.y ^ b.y; xb[2] = a.z ^ b.z; xb[3] = a.w ^ b.w;        // bonds inside a pair
        xb[4] = u.x ^ t.y; xb[5] = u.y ^ t.z; xb[6] = u.z ^ t.w; xb[7] = u.w ^ tn;         // bonds between pairs
        xb[8] = a.x ^ nb.x; xb[9] = a.y ^ nb.y; xb[10] = a.z ^ nb.z; xb[11] = a.w ^ nb.w;  // down bonds of colour 0
        xb[12] = b.x ^ na.x; xb[13] = b.y ^ na.y; xb[14] = b.z ^ na.z; xb[15] = b.w ^ na.w; // down bonds of colour 1
        if (HASJ) {
            const uint32_t j = act ? (uint32_t)__ldg(jm16 + (y & (L - 1)) * QPR + q) : 0u;
#pragma unroll
            for (int i = 0; i < 16; ++i) xb[i] ^= 0u - ((j >> i) & 1u);
        }
        const uint32_t xs[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
        if (LADDER) {
            ce[r & 7] = cE.block16(xb);
            cm[r & 7] = cM.block8(xs);
            if ((r & 7) == 7) { cE.template ladder8<4>(ce); cM.template ladder8<3>(cm); }
        } else {
            cE.add16(xb);
            cM.add8(xs);
        }
        a = na; b = nb; na = fa; nb = fb;
    }
    uint32_t pe[NPW], pm[NPW];
#pragma unroll
    for (int k = 0; k < NPW; ++k) { pe[k] = k < NPE ? cE.pl[k < NPE ? k : 0] : 0u; pm[k] = k < NPM ? cM.pl[k < NPM ? k : 0] : 0u; }
    pa_measure_tail<NPW>(pe, pm, g, N, N, R_cur, E, M, sc, runsum, blocksum, snap);
}

// ------------------------------------------------------------------------------------------------
// The quad-column walk for cubes of 8, 16, 32 (O16): a thread owns one quad column of ONE z-plane and walks down y; the row below is
// its own next load, the row of the plane above (+z bond) a second stream of loads, the +y bond of the plane's last row leads back
// to its first.  Per row and thread: 24 bond words (x, y, z) -> three 8-input carry-save blocks, 8 spin words -> one; the rows' top
// carries go through the eight-row ladder.  (The any-edge kernel spends 91 instructions per word on index arithmetic: 0.44 ms at
// 32^3, R = 10^5, against a 0.07 ms HBM floor.)
// ------------------------------------------------------------------------------------------------
template <int LOG_QPR>
__global__ void __launch_bounds__(128)
pa_measure3d_kernel(const uint32_t* __restrict__ pop, int N, long long R_cur, int32_t* __restrict__ E, int32_t* __restrict__ M,
                    PaScalars* __restrict__ sc, double* __restrict__ runsum, double* __restrict__ blocksum,
                    PaScalars* __restrict__ snap, int nlev) {
    constexpr int QPR = 1 << LOG_QPR, L = 8 * QPR, Lq = QPR;             // Lq = uint4 per colour row
    constexpr int NPE = pa_bits(24 * L), NPM = pa_bits(8 * L), NPW = NPE + 5;
    static_assert(NPE >= 8 && NPM >= 6, "ladder planes");
    pa_pdl_wait(); pa_pdl_launch();
    const long long g = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool act = tid < L * QPR;
    const int q = tid & (QPR - 1), z = act ? (tid >> LOG_QPR) : 0;
    const uint4* c0 = reinterpret_cast<const uint4*>(pop + g * (long long)N);
    const uint4* c1 = c0 + (N >> 3);
    const int r0 = z * L, rz = ((z + 1) & (L - 1)) * L;                   // first row of this plane / of the plane above
    const int nxt_lane = (lane & ~(QPR - 1)) | ((lane + 1) & (QPR - 1));
    const uint4 zero = make_uint4(0, 0, 0, 0);
    PlaneCounter<NPE> cE; PlaneCounter<NPM> cM;
    cE.clear(); cM.clear();
    uint4 a = zero, b = zero, na = zero, nb = zero, za = zero, zb = zero;
    if (act) {
        a = __ldg(c0 + r0 * Lq + q); b = __ldg(c1 + r0 * Lq + q);
        na = __ldg(c0 + (r0 + 1) * Lq + q); nb = __ldg(c1 + (r0 + 1) * Lq + q);
        za = __ldg(c0 + rz * Lq + q); zb = __ldg(c1 + rz * Lq + q);
    }
    uint32_t ce[8], cm[8];
#pragma unroll 8
    for (int y = 0; y < L; ++y) {
        uint4 fa = zero, fb = zero, fza = zero, fzb = zero;               // rows (z, y+2) and (z+1, y+1), in flight while row y is counted
        if (act) {
            const int y2 = (y + 2) & (L - 1), y1 = (y + 1) & (L - 1);
            fa = __ldg(c0 + (r0 + y2) * Lq + q); fb = __ldg(c1 + (r0 + y2) * Lq + q);
            fza = __ldg(c0 + (rz + y1) * Lq + q); fzb = __ldg(c1 + (rz + y1) * Lq + q);
        }
        const bool odd = ((y + z) & 1) != 0;                               // colour 0 holds x = 2 xh + ((y + z) & 1)
        const uint4 t = odd ? b : a, u = odd ? a : b;                      // bond u[xh] - t[xh + 1]
        const uint32_t tn = __shfl_sync(0xffffffffu, t.x, nxt_lane);
        uint32_t xb[24];
        xb[0] = a.x ^ b.x; xb[1] = a.y ^ b.y; xb[2] = a.z ^ b.z; xb[3] = a.w ^ b.w;          // x bonds inside a pair
        xb[4] = u.x ^ t.y; xb[5] = u.y ^ t.z; xb[6] = u.z ^ t.w; xb[7] = u.w ^ tn;           // x bonds between pairs
        xb[8] = a.x ^ nb.x; xb[9] = a.y ^ nb.y; xb[10] = a.z ^ nb.z; xb[11] = a.w ^ nb.w;    // +y bonds
        xb[12] = b.x ^ na.x; xb[13] = b.y ^ na.y; xb[14] = b.z ^ na.z; xb[15] = b.w ^ na.w;
        xb[16] = a.x ^ zb.x; xb[17] = a.y ^ zb.y; xb[18] = a.z ^ zb.z; xb[19] = a.w ^ zb.w;  // +z bonds
        xb[20] = b.x ^ za.x; xb[21] = b.y ^ za.y; xb[22] = b.z ^ za.z; xb[23] = b.w ^ za.w;
        const uint32_t xs[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
        {   // 24 inputs: three blocks of eight, their weight-8 carries into plane 3, the two weight-16 carries into plane 4
            const uint32_t e1 = cE.block8(xb), e2 = cE.block8(xb + 8), e3 = cE.block8(xb + 16);
            uint32_t c16, c32;
            pa_csa(c16, cE.pl[3], cE.pl[3], e1, e2);
            const uint32_t t16 = cE.pl[3] & e3;
            cE.pl[3] ^= e3;
            pa_csa(c32, cE.pl[4], cE.pl[4], c16, t16);
            ce[y & 7] = c32;
        }
        cm[y & 7] = cM.block8(xs);
        if ((y & 7) == 7) { cE.template ladder8<5>(ce); cM.template ladder8<3>(cm); }
        a = na; b = nb; na = fa; nb = fb; za = fza; zb = fzb;
    }
    uint32_t pe[NPW], pm[NPW];
#pragma unroll
    for (int k = 0; k < NPW; ++k) { pe[k] = k < NPE ? cE.pl[k < NPE ? k : 0] : 0u; pm[k] = k < NPM ? cM.pl[k < NPM ? k : 0] : 0u; }
    pa_measure_tail<NPW>(pe, pm, g, N, nlev, R_cur, E, M, sc, runsum, blocksum, snap);
}

int pa_launch_measure(pa_handle* h) {
    const int64_t G = h->dev_R ? h->G_cap : (h->R_cur + 31) / 32;      // dead groups contribute zeros (and +0.0 to the m^4 tree)
    const long long Rarg = h->dev_R ? -1 : h->R_cur;
    const int L = h->L;
    if (!h->scal_zeroed) PA_CUDA(h, cudaMemsetAsync(h->d_scal, 0, offsetof(PaScalars, R_new), h->stream));
    h->scal_zeroed = false;
    const bool timed = (h->timing & PA_TIME_MEASURE) != 0;
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[7], h->stream));
    // single calls: the last CTA writes the finished scalars straight into mapped host memory (pa_read_measure_scalars)
    const bool to_host = !h->dev_R && !h->snap_out && h->h_snap_dev && pa_sw(h, PA_SW_SNAP_HOST, 1) != 0;   // PA_SNAP_HOST=0: device-to-host copy instead
    PaScalars* const snap_save = h->snap_out;
    if (to_host) h->snap_out = h->h_snap_dev;
    h->snap_on_host = to_host;
    cudaError_t le = cudaSuccess;
    const bool pow2 = h->D == 2 && (L & (L - 1)) == 0 && L >= 8 && L <= 256 && !h->sw.set[PA_SW_MEASURE_GENERIC];
    if (pow2) {
#define PA_MSR_CASE(LOG) case (8 << LOG): \
        if (h->has_j) le = pa_launch(h, pa_measure_kernel<LOG, true>, dim3((unsigned)G), dim3(pa_msr_threads(8 << LOG)), 0, \
            (const uint32_t*)h->spins[h->cur], h->N, Rarg, h->E, h->M, h->d_scal, h->runsum, h->partials, (const uint16_t*)h->jm16, h->snap_out); \
        else le = pa_launch(h, pa_measure_kernel<LOG, false>, dim3((unsigned)G), dim3(pa_msr_threads(8 << LOG)), 0, \
            (const uint32_t*)h->spins[h->cur], h->N, Rarg, h->E, h->M, h->d_scal, h->runsum, h->partials, (const uint16_t*)nullptr, h->snap_out); \
        break;
        switch (L) { PA_MSR_CASE(0) PA_MSR_CASE(1) PA_MSR_CASE(2) PA_MSR_CASE(3) PA_MSR_CASE(4) PA_MSR_CASE(5) default: break; }
#undef PA_MSR_CASE
    } else if (h->D == 3 && !h->has_j && h->geom.Lx == h->geom.Ly && h->geom.Lx == h->geom.Lz && (L == 8 || L == 16 || L == 32) &&
               !h->sw.set[PA_SW_MEASURE_GENERIC]) {
        const int T3 = L * (L / 8) < 32 ? 32 : L * (L / 8);
#define PA_M3_CASE(LOG) le = pa_launch(h, pa_measure3d_kernel<LOG>, dim3((unsigned)G), dim3(T3), 0, (const uint32_t*)h->spins[h->cur], h->N, Rarg, \
            h->E, h->M, h->d_scal, h->runsum, h->partials, h->snap_out, h->nlev)
        if (L == 8) PA_M3_CASE(0); else if (L == 16) PA_M3_CASE(1); else PA_M3_CASE(2);
#undef PA_M3_CASE
    } else {
        int T = 256;
        while (T > 32 && T * 8 > h->N) T >>= 1;
#define PA_MG_CASE(LOGH, LOGY) le = pa_launch(h, pa_measure_generic_kernel<LOGH, LOGY>, dim3((unsigned)G), dim3(T), 0, (const uint32_t*)h->spins[h->cur], \
            h->geom, h->N, Rarg, h->E, h->M, h->d_scal, h->runsum, h->partials, h->has_j ? (const uint8_t*)h->jmask : (const uint8_t*)nullptr, h->snap_out, h->nlev)
        const int cube = h->D == 3 && h->geom.Lx == h->geom.Ly && !h->sw.set[PA_SW_MEASURE_GENERIC] ? h->geom.Lx : 0;
        switch (cube) {
            case 8: PA_MG_CASE(2, 3); break;
            case 16: PA_MG_CASE(3, 4); break;
            case 32: PA_MG_CASE(4, 5); break;
            case 64: PA_MG_CASE(5, 6); break;
            default: PA_MG_CASE(-1, -1); break;
        }
#undef PA_MG_CASE
    }
    h->snap_out = snap_save;
    PA_CUDA(h, le);
    PA_CUDA(h, cudaGetLastError());
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[8], h->stream));
    h->measure_timed = timed;
    h->launches += 1;
    h->em_valid = true;
    h->host_scal_valid = false;
    return PA_OK;
}
