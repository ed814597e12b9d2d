// pa_sweep.cu -- the checkerboard Metropolis sweep kernel.
//
// One thread-block cluster of C CTAs owns one group (32 replicas, one uint32 per site).  Each CTA
// stages H = L/C lattice rows of both colours in shared memory, runs all theta sweeps of the launch
// on chip (colour 0, barrier, colour 1, barrier -- the paper's "blue, synchronise, white", L157) and
// writes the rows back: HBM traffic is one read and one write of the population per launch.  Rows
// at a strip boundary read their vertical neighbour from the adjacent CTA's shared memory (DSMEM).
//
// Per word (32 spins) the work is: 8 Philox4x32-10 calls sharing their first rounds (the 8 counters
// differ only in c1 = 8g+i), 64 threshold tests, and a dozen bit-sliced logic ops for the neighbour
// count.  The kernel is bound by integer issue (IMAD.WIDE on the FMA pipe, LOP3 on the ALU pipe);
// see DESIGN.md Sec. 6 for the instruction budget.
#include "pa_common.cuh"
#include <cooperative_groups.h>
#include <math.h>
#include <stdlib.h>
namespace cg = cooperative_groups;

struct SweepParams {
    PhiloxKeys K;
    uint32_t T4, T8;                 // acceptance thresholds for dE = 4, 8 (O2)
    uint32_t T12;                    // ... and dE = 12 (simple-cubic lattice, O16)
    int Ly, Lz;                      // O16: rows per plane and planes (Lz = 1: square lattice); H = rows per CTA
    uint32_t t0;                     // sweep counter at launch
    uint32_t two;                    // the constant 2, opaque to ptxas (see pa_shift_in_ge)
    int theta;
    int L, Lh, H, C, N;
    long long R;                     // population size, or -1: read sc->R_dev (pa_anneal)
    const PaScalars* sc;
    long long Gcap;                  // groups the population buffer holds (p = 64 experiment: the second group of a pair may not exist)
    const uint8_t* jmask;            // O15: per resident word, bit k = bond to neighbour k (same, x, up, down) has J = -1; NULL = ferromagnet
    int whole;                       // host side: the launch covers the whole population (not a range of pa_step_host)
    long long g0;                    // column-walk kernels: first group of this launch (pa_launch_sweep_range: a step in chunks of groups); else 0
    const uint32_t* src;             // lane-split kernel with GATHER: the population before resampling and its parent map (new[d] = old[parent[d]])
    const uint32_t* parent;
    long long n_main;                // column-walk kernels without clusters, mixed launch (pa_sweep_pick_C): CTAs 0 .. n_main-1 own a whole group each, every
                                     // later group is shared by four lane-split CTAs; -1: uniform launch
};

// m = 2*m + (x >= T).  "sub.cc" leaves the hardware carry of x + ~T + 1 in CC.CF, i.e. NOT borrow, and
// "madc" adds it: ptxas emits one carry-out IADD3 (ALU pipe) and one IMAD.X (FMA pipe).  The multiplier is
// passed as a register holding 2 (a kernel parameter) so that ptxas cannot turn the shift-in into an ALU-pipe
// LEA.X / IADD3.X: on B200 every IMAD.WIDE also blocks the ALU pipe for two cycles, which makes the ALU pipe
// the binding one, so the insert has to stay on the FMA pipe.  Exact for every T
// including 0 (always 1) -- checked on the device by tests/test_parity_gpu.py::test_sweep_threshold_extremes.
__device__ __forceinline__ void pa_shift_in_ge(uint32_t& m, uint32_t x, uint32_t T, uint32_t two) {
    asm("{\n\t.reg .u32 t;\n\tsub.cc.u32 t, %1, %2;\n\tmadc.lo.u32 %0, %0, %3, 0;\n\t}" : "+r"(m) : "r"(x), "r"(T), "r"(two));
}

// m |= bit if x < T, with both instructions on the ALU pipe (ISETP + predicated LOP3).  The FMA pipe is
// the bottleneck of this kernel (IMAD.WIDE.U32 issues at 32 lanes/clk/SM), so the acceptance test must
// not add to it.
template <uint32_t BIT>
__device__ __forceinline__ void pa_or_if_lt(uint32_t& m, uint32_t x, uint32_t T) {
    asm("{\n\t.reg .pred q;\n\tsetp.lt.u32 q, %1, %2;\n\t@q or.b32 %0, %0, %3;\n\t}" : "+r"(m) : "r"(x), "r"(T), "n"(BIT));
}

// Flip mask of one word: bit b set iff replica 32g+b flips its spin at `site` (O3).
//   s: centre word, n0..n3: the four neighbour words.
//   c0base = hi(M1*c2) ^ k0[0] ^ 8g, lo1u = lo(M1*c2), c2 = 2t+colour (uniform per half-sweep).
template <int CMP>
__device__ __forceinline__ uint32_t pa_flip_mask(uint32_t s, uint32_t n0, uint32_t n1, uint32_t n2, uint32_t n3,
                                                 uint32_t site, uint32_t c0base, uint32_t lo1u,
                                                 const SweepParams& P) {
    // bit-sliced count u of anti-parallel neighbours per lane: dE = 8 - 4u (Eq. 10)
    uint32_t a0 = s ^ n0, a1 = s ^ n1, a2 = s ^ n2, a3 = s ^ n3;
    uint32_t U1 = a0 | a1 | a2 | a3;                                   // u >= 1
    uint32_t U2 = (a0 & a1) | (a2 & a3) | ((a0 ^ a1) & (a2 ^ a3));     // u >= 2: always flips

    // ---- 8 Philox4x32-10 calls, counters (site, 8g+i, 2t+c, TAG_SWEEP), i = 0..7 (O1) ----
    uint32_t x0[8], x1[8], x2[8], x3[8];
    // round 1: only c0' depends on i
    uint32_t hi0, lo0;
    pa_mulhilo(PA_PHILOX_M0, site, hi0, lo0);
    const uint32_t c2w = hi0 ^ PA_TAG_SWEEP ^ P.K.k1[0];
    const uint32_t c3w = lo0;
    // round 2: the M1 product and c0'', c1'' are shared by the 8 calls
    uint32_t hi1w, lo1w;
    pa_mulhilo(PA_PHILOX_M1, c2w, hi1w, lo1w);
    const uint32_t c0w = hi1w ^ lo1u ^ P.K.k0[1];
    const uint32_t c1w = lo1w;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M0, c0base ^ (uint32_t)i, h, l);
        x2[i] = h ^ c3w ^ P.K.k1[1];
        x3[i] = l;
    }
    // round 3: the M0 product is shared
    uint32_t hi0w, lo0w;
    pa_mulhilo(PA_PHILOX_M0, c0w, hi0w, lo0w);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M1, x2[i], h, l);
        x0[i] = h ^ c1w ^ P.K.k0[2];
        x1[i] = l;
        x2[i] = hi0w ^ x3[i] ^ P.K.k1[2];
        x3[i] = lo0w;
    }
    // rounds 4..10
#pragma unroll
    for (int r = 3; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            uint32_t h0, l0, h1, l1;
            pa_mulhilo(PA_PHILOX_M0, x0[i], h0, l0);
            pa_mulhilo(PA_PHILOX_M1, x2[i], h1, l1);
            x0[i] = h1 ^ x1[i] ^ P.K.k0[r];
            x1[i] = l1;
            x2[i] = h0 ^ x3[i] ^ P.K.k1[r];
            x3[i] = l0;
        }
    }
    // ---- acceptance: flip iff u >= 2, or u = 1 and x < T4, or u = 0 and x < T8 (O3) ----
    uint32_t acc = 0;
    if (CMP == 1) {
        uint32_t g4 = 0, g8 = 0;               // bit b = (x_b >= T): built most-significant bit first
#pragma unroll
        for (int i = 7; i >= 0; --i) {
            const uint32_t xs[4] = {x0[i], x1[i], x2[i], x3[i]};
#pragma unroll
            for (int q = 3; q >= 0; --q) {
                pa_shift_in_ge(g4, xs[q], P.T4, P.two);
                pa_shift_in_ge(g8, xs[q], P.T8, P.two);
            }
        }
        acc = ~g4 & (U1 | ~g8);                // (x < T4) and (u >= 1 or x < T8)
    } else if (CMP == 2) {
        uint32_t m4 = 0, m8 = 0;
#define PA_CMP4(I, Q, X) pa_or_if_lt<(1u << (4 * I + Q))>(m4, X, P.T4); pa_or_if_lt<(1u << (4 * I + Q))>(m8, X, P.T8);
#define PA_CMPI(I) PA_CMP4(I, 0, x0[I]) PA_CMP4(I, 1, x1[I]) PA_CMP4(I, 2, x2[I]) PA_CMP4(I, 3, x3[I])
        PA_CMPI(0) PA_CMPI(1) PA_CMPI(2) PA_CMPI(3) PA_CMPI(4) PA_CMPI(5) PA_CMPI(6) PA_CMPI(7)
#undef PA_CMPI
#undef PA_CMP4
        acc = m4 & (U1 | m8);
    } else {
        uint32_t m4 = 0, m8 = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const uint32_t xs[4] = {x0[i], x1[i], x2[i], x3[i]};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (xs[q] < P.T4) m4 |= 1u << (4 * i + q);
                if (xs[q] < P.T8) m8 |= 1u << (4 * i + q);
            }
        }
        acc = m4 & (U1 | m8);
    }
    return U2 | acc;
}

// LCG-assisted stream (O11; Sec. 4): the 32 lanes of the word take the next 32 outputs of
// r <- 1664525 r + 1013904223 (mod 2^32), most significant lane first (the first output is shifted in first and
// ends up in bit 31).  One 32-bit IMAD (FMA pipe, 2 cycles) per lane replaces a quarter of a Philox call
// (5 IMAD.WIDE + 5 LOP3); the acceptance test is the same carry-out compare with the shift-in on the FMA pipe.
// r <- A r + C as ONE multiply-add: written in PTX so that the compiler cannot re-associate the recurrence into
// s <- A s + C', x = s + C'' (it does, which costs an extra ALU-pipe add per lane).
__device__ __forceinline__ uint32_t pa_lcg_step(uint32_t r) {
    uint32_t o;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(o) : "r"(r), "n"(PA_LCG_A), "n"(PA_LCG_C));
    return o;
}

// NOR = number of leading lanes (31, 30, ...) whose two threshold tests run on the ALU pipe alone (ISETP +
// predicated OR) instead of carry-out IADD3 (ALU) + IMAD.X (FMA): balances the two pipes.
template <int NOR>
__device__ __forceinline__ uint32_t pa_flip_mask_lcg(uint32_t s, uint32_t n0, uint32_t n1, uint32_t n2, uint32_t n3,
                                                     uint32_t r, const SweepParams& P) {
    uint32_t a0 = s ^ n0, a1 = s ^ n1, a2 = s ^ n2, a3 = s ^ n3;
    uint32_t U1 = a0 | a1 | a2 | a3;                                   // u >= 1
    uint32_t U2 = (a0 & a1) | (a2 & a3) | ((a0 ^ a1) & (a2 ^ a3));     // u >= 2: always flips
    uint32_t m4 = 0, m8 = 0;                                           // bit b = (x_b <  T), lanes 31 .. 32-NOR
    uint32_t g4 = 0, g8 = 0;                                           // bit b = (x_b >= T), lanes 31-NOR .. 0
#define PA_LCG_OR(B) if (NOR > 31 - (B)) { r = pa_lcg_step(r); pa_or_if_lt<(1u << (B))>(m4, r, P.T4); pa_or_if_lt<(1u << (B))>(m8, r, P.T8); }
    PA_LCG_OR(31) PA_LCG_OR(30) PA_LCG_OR(29) PA_LCG_OR(28) PA_LCG_OR(27) PA_LCG_OR(26) PA_LCG_OR(25) PA_LCG_OR(24)
#undef PA_LCG_OR
#pragma unroll
    for (int b = 31 - NOR; b >= 0; --b) {
        r = pa_lcg_step(r);
        pa_shift_in_ge(g4, r, P.T4, P.two);
        pa_shift_in_ge(g8, r, P.T8, P.two);
    }
    constexpr uint32_t LOW = NOR == 0 ? 0xffffffffu : (0xffffffffu >> (NOR & 31));
    const uint32_t lt4 = (~g4 & LOW) | m4, lt8 = (~g8 & LOW) | m8;
    return U2 | (lt4 & (U1 | lt8));                                    // u >= 2, or x < T4 and (u >= 1 or x < T8)
}

// Lane-split CTAs (see pa_flip_mask_part): the eight lanes 8 sub + 7 ... 8 sub of the word take the LCG outputs number
// 25 - 8 sub ... 32 - 8 sub (O11: output n goes to lane 32 - n), reached by one jump r <- A^n r + C (A^n - 1)/(A - 1), n = 24 - 8 sub.
__host__ __device__ constexpr uint32_t pa_lcg_jump_mul(int n) { uint32_t a = 1u; for (int i = 0; i < n; ++i) a *= PA_LCG_A; return a; }
__host__ __device__ constexpr uint32_t pa_lcg_jump_add(int n) { uint32_t c = 0u; for (int i = 0; i < n; ++i) c = c * PA_LCG_A + PA_LCG_C; return c; }
template <int NL = 8>
__device__ __forceinline__ uint32_t pa_flip_mask_lcg_part(uint32_t s, uint32_t n0, uint32_t n1, uint32_t n2, uint32_t n3,
                                                          uint32_t r, uint32_t jmul, uint32_t jadd, uint32_t sh, const SweepParams& P) {
    uint32_t a0 = s ^ n0, a1 = s ^ n1, a2 = s ^ n2, a3 = s ^ n3;
    uint32_t U1 = a0 | a1 | a2 | a3;
    uint32_t U2 = (a0 & a1) | (a2 & a3) | ((a0 ^ a1) & (a2 ^ a3));
    r = r * jmul + jadd;
    uint32_t g4 = 0, g8 = 0;
#pragma unroll
    for (int b = NL - 1; b >= 0; --b) {
        r = pa_lcg_step(r);
        pa_shift_in_ge(g4, r, P.T4, P.two);
        pa_shift_in_ge(g8, r, P.T8, P.two);
    }
    const uint32_t acc = ~g4 & ((U1 >> sh) | ~g8);
    return (((U2 >> sh) | acc) & ((1u << NL) - 1u)) << sh;
}

// The four LCG seeds of a quad of rows (y & ~3 .. +3) in column xh of one sub-lattice: one Philox call (O11).
__device__ __forceinline__ uint4 pa_lcg_seeds(uint32_t quad, uint32_t g, uint32_t c2, const PhiloxKeys& K) {
    return pa_philox(quad, g, c2, PA_TAG_LCG, K);
}

// O15: neighbour word as the acceptance logic must see it: complemented if bond k of this site has J = -1
__device__ __forceinline__ uint32_t pa_jx(uint32_t n, uint32_t j, int k) { return n ^ (0u - ((j >> k) & 1u)); }

template <int CMP, bool CLUSTER, int RNG, bool HASJ>
__global__ void __launch_bounds__(256)
pa_sweep_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint32_t tile[];   // [2][H][Lh]
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    const long long g = blockIdx.x / C;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;        // past the population (capacity-sized grid in pa_anneal); uniform per cluster
    const int H = P.H, Lh = P.Lh, L = P.L;
    const int y0 = (int)cr * H;
    const int half = H * Lh;
    uint32_t* gbase = pop + g * (long long)P.N;
    const int goff = y0 * Lh, gcol = P.N >> 1;

    // stage both colours of this strip
    if ((Lh & 3) == 0) {
        for (int c = 0; c < 2; ++c) {
            const uint4* src = reinterpret_cast<const uint4*>(gbase + c * gcol + goff);
            uint4* dst = reinterpret_cast<uint4*>(tile + c * half);
            for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
        }
    } else {
        for (int c = 0; c < 2; ++c)
            for (int i = tid; i < half; i += T) tile[c * half + i] = gbase[c * gcol + goff + i];
    }
    const uint32_t* up_tile = tile;
    const uint32_t* dn_tile = tile;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }

    const int dy = T / Lh, dx = T % Lh;
    const uint32_t g8 = (uint32_t)(8 * g);
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t hi1u, lo1u;
            pa_mulhilo(PA_PHILOX_M1, c2, hi1u, lo1u);
            const uint32_t c0base = hi1u ^ P.K.k0[0] ^ g8;
            uint32_t* mine = tile + c * half;
            const uint32_t* oth = tile + (1 - c) * half;
            const uint32_t* up_oth = up_tile + (1 - c) * half;
            const uint32_t* dn_oth = dn_tile + (1 - c) * half;
            int yl = tid / Lh, xh = tid % Lh;
#pragma unroll 1
            for (int w = tid; w < half; w += T) {
                const int y = y0 + yl;
                const int p = (y + c) & 1;
                const int row = yl * Lh;
                const uint32_t s = mine[row + xh];
                const uint32_t nS = oth[row + xh];
                const int xh2 = p ? (xh + 1 == Lh ? 0 : xh + 1) : (xh == 0 ? Lh - 1 : xh - 1);
                const uint32_t nX = oth[row + xh2];
                uint32_t nU, nD;
                if (yl > 0) nU = oth[row - Lh + xh]; else nU = up_oth[(H - 1) * Lh + xh];
                if (yl < H - 1) nD = oth[row + Lh + xh]; else nD = dn_oth[xh];
                uint32_t nS_ = nS, nX_ = nX;
                if (HASJ) {
                    // O15: a bond with J = -1 is unsatisfied when the spins are parallel: complement that neighbour's word
                    const uint32_t j = P.jmask[c * gcol + y * Lh + xh];
                    nS_ ^= 0u - (j & 1u); nX_ ^= 0u - ((j >> 1) & 1u); nU ^= 0u - ((j >> 2) & 1u); nD ^= 0u - ((j >> 3) & 1u);
                }
                uint32_t flip;
                if (RNG == PA_RNG_LCG) {
                    const uint4 sd = pa_lcg_seeds((uint32_t)((y >> 2) * Lh + xh), (uint32_t)g, c2, P.K);
                    const int q = y & 3;
                    flip = pa_flip_mask_lcg<0>(s, nS_, nX_, nU, nD, q == 0 ? sd.x : q == 1 ? sd.y : q == 2 ? sd.z : sd.w, P);
                } else {
                    const uint32_t site = (uint32_t)(y * L + 2 * xh + p);
                    flip = pa_flip_mask<CMP>(s, nS_, nX_, nU, nD, site, c0base, lo1u, P);
                }
                mine[row + xh] = s ^ flip;
                xh += dx; yl += dy;
                if (xh >= Lh) { xh -= Lh; yl += 1; }
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }

    if ((Lh & 3) == 0) {
        for (int c = 0; c < 2; ++c) {
            uint4* dst = reinterpret_cast<uint4*>(gbase + c * gcol + goff);
            const uint4* src = reinterpret_cast<const uint4*>(tile + c * half);
            for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
        }
    } else {
        for (int c = 0; c < 2; ++c)
            for (int i = tid; i < half; i += T) gbase[c * gcol + goff + i] = tile[c * half + i];
    }
}

// ------------------------------------------------------------------------------------------------
// Lane-split CTAs.  The 32 replicas of a word are independent, so a group can be shared out by LANES instead of by rows: S CTAs
// (on S different SMs) each stage the whole group but advance only the 32/S lanes of byte(s) `sub` of every word -- the 8/S
// Philox calls i = sub*8/S ... of the word's eight (lanes 4i .. 4i+3, O1) -- and write back only those bytes.  No halo, no cluster
// barrier, no atomics; the price is that rounds 1-3 are shared by fewer calls (1 + 2 (NC+1) + 14 NC wide multiplies for NC calls:
// 35 x 4 instead of 131) and that the neighbour logic is repeated per CTA.  Used where whole groups cannot fill the SMs: small
// populations on the generic path (cfg1: 32 groups -> 128 CTAs), and the last, incomplete round of a medium population on the
// column-walk path (pa_sweep_pick_C).
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ uint32_t pa_flip_mask_part(uint32_t s, uint32_t n0, uint32_t n1, uint32_t n2, uint32_t n3,
                                                      uint32_t site, uint32_t c0base, uint32_t lo1u, uint32_t i0,
                                                      const SweepParams& P) {
    uint32_t a0 = s ^ n0, a1 = s ^ n1, a2 = s ^ n2, a3 = s ^ n3;
    uint32_t U1 = a0 | a1 | a2 | a3;
    uint32_t U2 = (a0 & a1) | (a2 & a3) | ((a0 ^ a1) & (a2 ^ a3));
    uint32_t x0[NC], x1[NC], x2[NC], x3[NC];
    uint32_t hi0, lo0;
    pa_mulhilo(PA_PHILOX_M0, site, hi0, lo0);
    const uint32_t c2w = hi0 ^ PA_TAG_SWEEP ^ P.K.k1[0];
    const uint32_t c3w = lo0;
    uint32_t hi1w, lo1w;
    pa_mulhilo(PA_PHILOX_M1, c2w, hi1w, lo1w);
    const uint32_t c0w = hi1w ^ lo1u ^ P.K.k0[1];
    const uint32_t c1w = lo1w;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M0, c0base ^ (i0 + (uint32_t)i), h, l);
        x2[i] = h ^ c3w ^ P.K.k1[1];
        x3[i] = l;
    }
    uint32_t hi0w, lo0w;
    pa_mulhilo(PA_PHILOX_M0, c0w, hi0w, lo0w);
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M1, x2[i], h, l);
        x0[i] = h ^ c1w ^ P.K.k0[2];
        x1[i] = l;
        x2[i] = hi0w ^ x3[i] ^ P.K.k1[2];
        x3[i] = lo0w;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            uint32_t h0, l0, h1, l1;
            pa_mulhilo(PA_PHILOX_M0, x0[i], h0, l0);
            pa_mulhilo(PA_PHILOX_M1, x2[i], h1, l1);
            x0[i] = h1 ^ x1[i] ^ P.K.k0[r];
            x1[i] = l1;
            x2[i] = h0 ^ x3[i] ^ P.K.k1[r];
            x3[i] = l0;
        }
    }
    uint32_t g4 = 0, g8 = 0;                   // bit 4i+q (relative to lane 4 i0) = (x >= T), most significant first
#pragma unroll
    for (int i = NC - 1; i >= 0; --i) {
        const uint32_t xs[4] = {x0[i], x1[i], x2[i], x3[i]};
#pragma unroll
        for (int q = 3; q >= 0; --q) {
            pa_shift_in_ge(g4, xs[q], P.T4, P.two);
            pa_shift_in_ge(g8, xs[q], P.T8, P.two);
        }
    }
    constexpr uint32_t LM = NC == 8 ? 0xffffffffu : ((1u << (4 * (NC & 7))) - 1u);
    const uint32_t sh = 4u * i0;
    const uint32_t acc = ~g4 & ((U1 >> sh) | ~g8);
    return (((U2 >> sh) | acc) & LM) << sh;
}

// write back the lanes of lane block `sub` (of S) of n words: byte / halfword stores, little-endian lane order
template <int S>
__device__ __forceinline__ void pa_store_lanes(uint32_t* gdst, const uint32_t* src, int n, int sub, int tid, int T) {
    if (S == 4) {
        uint8_t* d = reinterpret_cast<uint8_t*>(gdst) + sub;
        for (int i = tid; i < n; i += T) d[4 * i] = (uint8_t)(src[i] >> (8 * sub));
    } else {
        uint16_t* d = reinterpret_cast<uint16_t*>(gdst) + sub;
        for (int i = tid; i < n; i += T) d[2 * i] = (uint16_t)(src[i] >> (16 * sub));
    }
}

// GATHER (pa_anneal, small populations): `pop` is the NEW population buffer; the strip is staged from the old population P.src
// through the parent map -- the replica copy of the resampling step (L165-L171, O7: new[d] = old[parent(d)], dead lanes 0) done by
// the kernel that needs the words anyway, which saves the launch-bound step a kernel.
template <int S, bool GATHER, int RNG, bool HASJ>
__global__ void __launch_bounds__(256)
pa_sweep_split_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    constexpr int NC = 8 / S;
    extern __shared__ __align__(16) uint32_t tile[];   // [2][L][Lh]: the whole group (only this CTA's lanes are kept current)
    const int T = blockDim.x, tid = threadIdx.x;
    const long long g = blockIdx.x / S;
    const int sub = blockIdx.x % S;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;
    const int Lh = P.Lh, L = P.L, half = P.N >> 1;
    uint32_t* gbase = pop + g * (long long)P.N;
    if (GATHER) {
        constexpr int NL = 32 / S;                     // this CTA's lanes: NL * sub ... NL * sub + NL - 1
        __shared__ uint32_t s_par[NL];
        if (tid < NL) {
            const long long d = g * 32 + sub * NL + tid;
            s_par[tid] = d < pa_live_R(P.R, P.sc) ? P.parent[d] : 0xffffffffu;
        }
        __syncthreads();
        for (int i = tid; i < P.N; i += T) {
            uint32_t wd = 0u, q_last = 0xffffffffu, ws = 0u;
#pragma unroll
            for (int k = 0; k < NL; ++k) {
                const uint32_t pr = s_par[k];
                if (pr != 0xffffffffu) {
                    const uint32_t q = pr >> 5;
                    if (q != q_last) { ws = P.src[(size_t)q * P.N + i]; q_last = q; }    // parents are non-decreasing: each source word once
                    wd |= ((ws >> (pr & 31u)) & 1u) << (sub * NL + k);
                }
            }
            tile[i] = wd;
        }
    } else {
        for (int i = tid; i < P.N; i += T) tile[i] = gbase[i];
    }
    __syncthreads();
    const uint32_t g8 = (uint32_t)(8 * g);
    // LCG stream (O11): skip the outputs that belong to the lanes above this CTA's block of 32/S lanes
    constexpr int NLN = 32 / S;
    const int nskip = 32 - NLN * (sub + 1);
    const uint32_t jmul = nskip == 24 ? pa_lcg_jump_mul(24) : nskip == 16 ? pa_lcg_jump_mul(16) : nskip == 8 ? pa_lcg_jump_mul(8) : 1u;
    const uint32_t jadd = nskip == 24 ? pa_lcg_jump_add(24) : nskip == 16 ? pa_lcg_jump_add(16) : nskip == 8 ? pa_lcg_jump_add(8) : 0u;
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t hi1u, lo1u;
            pa_mulhilo(PA_PHILOX_M1, c2, hi1u, lo1u);
            const uint32_t c0base = hi1u ^ P.K.k0[0] ^ g8;
            uint32_t* mine = tile + c * half;
            const uint32_t* oth = tile + (1 - c) * half;
            int y = tid / Lh, xh = tid % Lh;
            const int dy = T / Lh, dx = T % Lh;
#pragma unroll 1
            for (int w = tid; w < half; w += T) {
                const int p = (y + c) & 1;
                const int xh2 = p ? (xh + 1 == Lh ? 0 : xh + 1) : (xh == 0 ? Lh - 1 : xh - 1);
                const uint32_t s = mine[w];
                uint32_t nS = oth[w];
                uint32_t nX = oth[w - xh + xh2];
                uint32_t nU = oth[(y == 0 ? L - 1 : y - 1) * Lh + xh];
                uint32_t nD = oth[(y + 1 == L ? 0 : y + 1) * Lh + xh];
                if (HASJ) {                                   // O15: complement the neighbour across a bond with J = -1
                    const uint32_t j = P.jmask[c * half + w];
                    nS = pa_jx(nS, j, 0); nX = pa_jx(nX, j, 1); nU = pa_jx(nU, j, 2); nD = pa_jx(nD, j, 3);
                }
                if (RNG == PA_RNG_LCG) {
                    const uint4 sd = pa_lcg_seeds((uint32_t)((y >> 2) * Lh + xh), (uint32_t)g, c2, P.K);
                    const int q = y & 3;
                    mine[w] = s ^ pa_flip_mask_lcg_part<NLN>(s, nS, nX, nU, nD, q == 0 ? sd.x : q == 1 ? sd.y : q == 2 ? sd.z : sd.w,
                                                             jmul, jadd, (uint32_t)(sub * NLN), P);
                } else {
                    const uint32_t site = (uint32_t)(y * L + 2 * xh + p);
                    mine[w] = s ^ pa_flip_mask_part<NC>(s, nS, nX, nU, nD, site, c0base, lo1u, (uint32_t)(sub * NC), P);
                }
                xh += dx; y += dy;
                if (xh >= Lh) { xh -= Lh; y += 1; }
            }
            __syncthreads();
        }
    }
    pa_store_lanes<S>(gbase, tile, P.N, sub, tid, T);
}

// ------------------------------------------------------------------------------------------------
// Column-walk variant for power-of-two L >= 64 (all of BASELINE.json's configs but L = 16).
// A thread owns one column xh of the strip and walks down `rpt` consecutive rows, two rows per
// iteration (the two rows have opposite x-parity, so the pair is the natural unit).  Every shared-memory
// address is the thread's base pointer plus a compile-time immediate, the up-neighbour of the second row
// and the down-neighbour of the first are words the pair has loaded anyway, and the site index advances by
// a constant: the per-word addressing overhead of the generic kernel (about 35 ALU-pipe instructions per
// word, 8 % of the kernel) disappears.  The ALU pipe is the binding one.
// Requirements (checked by pa_sweep_configure): Lh = 2^LOG_LH >= 32, T >= Lh, H*Lh/T even and >= 2, H even.
// ------------------------------------------------------------------------------------------------
// Block size: 256 threads, and 512 for L = 256 (LOG_LH = 7), where a cluster of TWO CTAs with 128 KB strips and one CTA of 16
// warps per SM beats four CTAs with 64 KB strips (clusters of 4 cannot be placed on 16 of the 148 SMs; measured in
// profiles/r02_sweep_L256.md: 1 586 -> 1 679 updates/ns at cfg5).
#define PA_SWEEP_BOUNDS __launch_bounds__(LOG_LH == 7 ? 512 : 256)
template <int CMP, int LOG_LH, bool CLUSTER, bool HASJ>
__global__ void PA_SWEEP_BOUNDS
pa_sweep_col_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint32_t tile[];   // [2][H][Lh]
    constexpr int Lh = 1 << LOG_LH;
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    long long g = blockIdx.x / C;
    int sub = -1;                                      // >= 0: this CTA advances only the lanes of byte `sub` of its group (lane-split CTAs)
    if (!CLUSTER && P.n_main >= 0 && g >= P.n_main) {  // mixed launch: n_main whole groups, then four CTAs per remaining group
        sub = (int)((g - P.n_main) & 3);
        g = P.n_main + ((g - P.n_main) >> 2);
    }
    g += P.g0;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;        // past the population (capacity-sized grid in pa_anneal); uniform per cluster
    const int H = P.H;
    const int y0 = (int)cr * H;
    const int half = H * Lh;
    uint32_t* gbase = pop + g * (long long)P.N;
    const int goff = y0 * Lh, gcol = P.N >> 1;

    for (int c = 0; c < 2; ++c) {
        const uint4* src = reinterpret_cast<const uint4*>(gbase + c * gcol + goff);
        uint4* dst = reinterpret_cast<uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
    const uint32_t* up_tile = tile;
    const uint32_t* dn_tile = tile;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }

    const int xh = tid & (Lh - 1), rb = tid >> LOG_LH;
    const int rpt = half / T;                          // rows per thread: even, >= 2
    const int ya = rb * rpt;                           // first local row (even)
    const int dL = ((xh - 1) & (Lh - 1)) - xh, dR = ((xh + 1) & (Lh - 1)) - xh;
    const int b0 = ya * Lh + xh;
    const uint32_t g8 = (uint32_t)(8 * g);
    const uint32_t site_base = 2u * (uint32_t)((y0 + ya) * Lh + xh);   // site of (row y0+ya, x = 2 xh)
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t hi1u, lo1u;
            pa_mulhilo(PA_PHILOX_M1, c2, hi1u, lo1u);
            const uint32_t c0base = hi1u ^ P.K.k0[0] ^ g8;
            uint32_t* mine = tile + c * half + b0;
            const uint32_t* oth = tile + (1 - c) * half + b0;
            // rows y0+ya+2k have x-parity p = c (x = 2 xh + c), rows y0+ya+2k+1 have p = 1 - c
            const int dA = c ? dR : dL, dB = c ? dL : dR;
            uint32_t site = site_base + (uint32_t)c;
            const uint8_t* jm = HASJ ? P.jmask + c * gcol + goff + b0 : nullptr;     // bond masks of this thread's column (O15)
#pragma unroll 1
            for (int k = 0; k < rpt; k += 2) {
                const uint32_t s0 = mine[0], s1 = mine[Lh];
                const uint32_t nS0 = oth[0], nS1 = oth[Lh];
                const uint32_t nX0 = oth[dA], nX1 = oth[Lh + dB];
                uint32_t nU0, nD1;
                if (ya + k > 0) nU0 = oth[-Lh]; else nU0 = up_tile[(1 - c) * half + (H - 1) * Lh + xh];
                if (ya + k + 2 < H) nD1 = oth[2 * Lh]; else nD1 = dn_tile[(1 - c) * half + xh];
                uint32_t f0, f1;
                if (HASJ) {
                    const uint32_t j0 = jm[0], j1 = jm[Lh];
                    f0 = pa_flip_mask<CMP>(s0, pa_jx(nS0, j0, 0), pa_jx(nX0, j0, 1), pa_jx(nU0, j0, 2), pa_jx(nS1, j0, 3), site, c0base, lo1u, P);
                    f1 = pa_flip_mask<CMP>(s1, pa_jx(nS1, j1, 0), pa_jx(nX1, j1, 1), pa_jx(nS0, j1, 2), pa_jx(nD1, j1, 3),
                                           site + (uint32_t)(2 * Lh + 1 - 2 * c), c0base, lo1u, P);
                    jm += 2 * Lh;
                } else if (!CLUSTER && sub >= 0) {
                    f0 = pa_flip_mask_part<2>(s0, nS0, nX0, nU0, nS1, site, c0base, lo1u, 2u * (uint32_t)sub, P);
                    f1 = pa_flip_mask_part<2>(s1, nS1, nX1, nS0, nD1, site + (uint32_t)(2 * Lh + 1 - 2 * c), c0base, lo1u, 2u * (uint32_t)sub, P);
                } else {
                    f0 = pa_flip_mask<CMP>(s0, nS0, nX0, nU0, nS1, site, c0base, lo1u, P);
                    f1 = pa_flip_mask<CMP>(s1, nS1, nX1, nS0, nD1, site + (uint32_t)(2 * Lh + 1 - 2 * c), c0base, lo1u, P);
                }
                mine[0] = s0 ^ f0;
                mine[Lh] = s1 ^ f1;
                mine += 2 * Lh; oth += 2 * Lh; site += 4u * Lh;
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }

    if (!CLUSTER && sub >= 0) {                        // only this CTA's lanes are current
        for (int c = 0; c < 2; ++c) pa_store_lanes<4>(gbase + c * gcol + goff, tile + c * half, half, sub, tid, T);
        return;
    }
    for (int c = 0; c < 2; ++c) {
        uint4* dst = reinterpret_cast<uint4*>(gbase + c * gcol + goff);
        const uint4* src = reinterpret_cast<const uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
}

// ------------------------------------------------------------------------------------------------
// Column-walk kernel for the LCG-assisted stream (O11): the same strip / cluster layout, but a thread walks
// FOUR rows per iteration -- the quad of rows that shares one Philox call for its four LCG seeds.  The six
// vertical-neighbour words of the quad are loaded once.  Requirements (pa_col_ok): as above and rows per thread
// a multiple of 4, strip height a multiple of 4.
// ------------------------------------------------------------------------------------------------
template <int LOG_LH, bool CLUSTER, int NOR, bool HASJ>
__global__ void PA_SWEEP_BOUNDS
pa_sweep_lcg_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint32_t tile[];   // [2][H][Lh]
    constexpr int Lh = 1 << LOG_LH;
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    long long g = blockIdx.x / C;
    int sub = -1;                                      // >= 0: this CTA advances only the lanes of byte `sub` of its group (lane-split CTAs)
    if (!CLUSTER && P.n_main >= 0 && g >= P.n_main) {  // mixed launch: n_main whole groups, then four CTAs per remaining group
        sub = (int)((g - P.n_main) & 3);
        g = P.n_main + ((g - P.n_main) >> 2);
    }
    g += P.g0;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;        // past the population (capacity-sized grid in pa_anneal); uniform per cluster
    const int H = P.H;
    const int y0 = (int)cr * H;
    const int half = H * Lh;
    uint32_t* gbase = pop + g * (long long)P.N;
    const int goff = y0 * Lh, gcol = P.N >> 1;

    for (int c = 0; c < 2; ++c) {
        const uint4* src = reinterpret_cast<const uint4*>(gbase + c * gcol + goff);
        uint4* dst = reinterpret_cast<uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
    const uint32_t* up_tile = tile;
    const uint32_t* dn_tile = tile;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }

    const int xh = tid & (Lh - 1), rb = tid >> LOG_LH;
    const int rpt = half / T;                          // rows per thread: multiple of 4
    const int ya = rb * rpt;                           // first local row (multiple of 4)
    const int dL = ((xh - 1) & (Lh - 1)) - xh, dR = ((xh + 1) & (Lh - 1)) - xh;
    const int b0 = ya * Lh + xh;
    const uint32_t quad_base = (uint32_t)(((y0 + ya) >> 2) * Lh + xh);
    // lane-split CTA: skip the 24 - 8 sub LCG outputs that belong to the lanes above this CTA's byte
    const uint32_t jmul = sub == 0 ? pa_lcg_jump_mul(24) : sub == 1 ? pa_lcg_jump_mul(16) : sub == 2 ? pa_lcg_jump_mul(8) : 1u;
    const uint32_t jadd = sub == 0 ? pa_lcg_jump_add(24) : sub == 1 ? pa_lcg_jump_add(16) : sub == 2 ? pa_lcg_jump_add(8) : 0u;
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t* mine = tile + c * half + b0;
            const uint32_t* oth = tile + (1 - c) * half + b0;
            // rows y0+ya+2k have x-parity p = c (x = 2 xh + c), rows y0+ya+2k+1 have p = 1 - c
            const int dA = c ? dR : dL, dB = c ? dL : dR;
            uint32_t quad = quad_base;
            const uint8_t* jm = HASJ ? P.jmask + c * gcol + goff + b0 : nullptr;     // bond masks of this thread's column (O15)
#pragma unroll 1
            for (int k = 0; k < rpt; k += 4) {
                const uint4 sd = pa_lcg_seeds(quad, (uint32_t)g, c2, P.K);
                const uint32_t s0 = mine[0], s1 = mine[Lh], s2 = mine[2 * Lh], s3 = mine[3 * Lh];
                const uint32_t o0 = oth[0], o1 = oth[Lh], o2 = oth[2 * Lh], o3 = oth[3 * Lh];
                const uint32_t x0 = oth[dA], x1 = oth[Lh + dB], x2 = oth[2 * Lh + dA], x3 = oth[3 * Lh + dB];
                uint32_t oU, oD;
                if (ya + k > 0) oU = oth[-Lh]; else oU = up_tile[(1 - c) * half + (H - 1) * Lh + xh];
                if (ya + k + 4 < H) oD = oth[4 * Lh]; else oD = dn_tile[(1 - c) * half + xh];
                uint32_t f0, f1, f2, f3;
                if (HASJ) {
                    const uint32_t j0 = jm[0], j1 = jm[Lh], j2 = jm[2 * Lh], j3 = jm[3 * Lh];
                    f0 = pa_flip_mask_lcg<NOR>(s0, pa_jx(o0, j0, 0), pa_jx(x0, j0, 1), pa_jx(oU, j0, 2), pa_jx(o1, j0, 3), sd.x, P);
                    f1 = pa_flip_mask_lcg<NOR>(s1, pa_jx(o1, j1, 0), pa_jx(x1, j1, 1), pa_jx(o0, j1, 2), pa_jx(o2, j1, 3), sd.y, P);
                    f2 = pa_flip_mask_lcg<NOR>(s2, pa_jx(o2, j2, 0), pa_jx(x2, j2, 1), pa_jx(o1, j2, 2), pa_jx(o3, j2, 3), sd.z, P);
                    f3 = pa_flip_mask_lcg<NOR>(s3, pa_jx(o3, j3, 0), pa_jx(x3, j3, 1), pa_jx(o2, j3, 2), pa_jx(oD, j3, 3), sd.w, P);
                    jm += 4 * Lh;
                } else if (!CLUSTER && sub >= 0) {
                    f0 = pa_flip_mask_lcg_part(s0, o0, x0, oU, o1, sd.x, jmul, jadd, 8u * (uint32_t)sub, P);
                    f1 = pa_flip_mask_lcg_part(s1, o1, x1, o0, o2, sd.y, jmul, jadd, 8u * (uint32_t)sub, P);
                    f2 = pa_flip_mask_lcg_part(s2, o2, x2, o1, o3, sd.z, jmul, jadd, 8u * (uint32_t)sub, P);
                    f3 = pa_flip_mask_lcg_part(s3, o3, x3, o2, oD, sd.w, jmul, jadd, 8u * (uint32_t)sub, P);
                } else {
                    f0 = pa_flip_mask_lcg<NOR>(s0, o0, x0, oU, o1, sd.x, P);
                    f1 = pa_flip_mask_lcg<NOR>(s1, o1, x1, o0, o2, sd.y, P);
                    f2 = pa_flip_mask_lcg<NOR>(s2, o2, x2, o1, o3, sd.z, P);
                    f3 = pa_flip_mask_lcg<NOR>(s3, o3, x3, o2, oD, sd.w, P);
                }
                mine[0] = s0 ^ f0;
                mine[Lh] = s1 ^ f1;
                mine[2 * Lh] = s2 ^ f2;
                mine[3 * Lh] = s3 ^ f3;
                mine += 4 * Lh; oth += 4 * Lh; quad += Lh;
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }

    if (!CLUSTER && sub >= 0) {                        // only this CTA's lanes are current
        for (int c = 0; c < 2; ++c) pa_store_lanes<4>(gbase + c * gcol + goff, tile + c * half, half, sub, tid, T);
        return;
    }
    for (int c = 0; c < 2; ++c) {
        uint4* dst = reinterpret_cast<uint4*>(gbase + c * gcol + goff);
        const uint4* src = reinterpret_cast<const uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
}

// ------------------------------------------------------------------------------------------------
// p = 64 experiment (Sec. 4, Table 1 L196 / L200 / L204: 64-bit words were SLOWER than 32-bit ones on Kepler; SURVEY
// 8(f) row 4 asks for the measurement on B200).  The LCG column-walk kernel with a 64-replica word = the words of two adjacent
// groups side by side (uint2 in shared memory, 64-bit LDS / STS); the random stream is unchanged (O11: one seed per 32-replica
// word), so the result is bit-identical to the p = 32 kernel.  What a wider word can share on a 32-bit integer datapath is the
// addressing, the loop and half of the shared-memory instructions; every LCG step, compare, insert and logic op doubles.
// Taken automatically at L = 64 for large populations (pa_sweep_dispatch_lcg); PA_LCG_P64=1 / 0 force it on (power-of-two L, ferromagnet) / off.
// ------------------------------------------------------------------------------------------------
template <int LOG_LH, bool CLUSTER, int NOR>
__global__ void __launch_bounds__(LOG_LH == 7 ? 512 : 256)
pa_sweep_lcg64_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint2 tile2[];     // [2][H][Lh], .x = group 2q, .y = group 2q+1
    constexpr int Lh = 1 << LOG_LH;
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    const long long ga = 2 * (long long)(blockIdx.x / C), gb = ga + 1;
    pa_pdl_wait(); pa_pdl_launch();
    if (ga * 32 >= pa_live_R(P.R, P.sc)) return;
    const bool vb = gb < P.Gcap;
    const int H = P.H;
    const int y0 = (int)cr * H;
    const int half = H * Lh;
    uint32_t* abase = pop + ga * (long long)P.N;
    uint32_t* bbase = pop + gb * (long long)P.N;
    const int goff = y0 * Lh, gcol = P.N >> 1;
    for (int c = 0; c < 2; ++c)
        for (int i = tid; i < half; i += T)
            tile2[c * half + i] = make_uint2(abase[c * gcol + goff + i], vb ? bbase[c * gcol + goff + i] : 0u);
    const uint2* up_tile = tile2;
    const uint2* dn_tile = tile2;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile2, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile2, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }
    const int xh = tid & (Lh - 1), rb = tid >> LOG_LH;
    const int rpt = half / T;
    const int ya = rb * rpt;
    const int dL = ((xh - 1) & (Lh - 1)) - xh, dR = ((xh + 1) & (Lh - 1)) - xh;
    const int b0 = ya * Lh + xh;
    const uint32_t quad_base = (uint32_t)(((y0 + ya) >> 2) * Lh + xh);
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint2* mine = tile2 + c * half + b0;
            const uint2* oth = tile2 + (1 - c) * half + b0;
            const int dA = c ? dR : dL, dB = c ? dL : dR;
            uint32_t quad = quad_base;
#pragma unroll 1
            for (int k = 0; k < rpt; k += 4) {
                const uint4 sa = pa_lcg_seeds(quad, (uint32_t)ga, c2, P.K);
                const uint4 sb = pa_lcg_seeds(quad, (uint32_t)gb, c2, P.K);
                const uint2 s0 = mine[0], s1 = mine[Lh], s2 = mine[2 * Lh], s3 = mine[3 * Lh];
                const uint2 o0 = oth[0], o1 = oth[Lh], o2 = oth[2 * Lh], o3 = oth[3 * Lh];
                const uint2 x0 = oth[dA], x1 = oth[Lh + dB], x2 = oth[2 * Lh + dA], x3 = oth[3 * Lh + dB];
                uint2 oU, oD;
                if (ya + k > 0) oU = oth[-Lh]; else oU = up_tile[(1 - c) * half + (H - 1) * Lh + xh];
                if (ya + k + 4 < H) oD = oth[4 * Lh]; else oD = dn_tile[(1 - c) * half + xh];
                uint2 f0, f1, f2, f3;
                f0.x = pa_flip_mask_lcg<NOR>(s0.x, o0.x, x0.x, oU.x, o1.x, sa.x, P);
                f1.x = pa_flip_mask_lcg<NOR>(s1.x, o1.x, x1.x, o0.x, o2.x, sa.y, P);
                f2.x = pa_flip_mask_lcg<NOR>(s2.x, o2.x, x2.x, o1.x, o3.x, sa.z, P);
                f3.x = pa_flip_mask_lcg<NOR>(s3.x, o3.x, x3.x, o2.x, oD.x, sa.w, P);
                f0.y = pa_flip_mask_lcg<NOR>(s0.y, o0.y, x0.y, oU.y, o1.y, sb.x, P);
                f1.y = pa_flip_mask_lcg<NOR>(s1.y, o1.y, x1.y, o0.y, o2.y, sb.y, P);
                f2.y = pa_flip_mask_lcg<NOR>(s2.y, o2.y, x2.y, o1.y, o3.y, sb.z, P);
                f3.y = pa_flip_mask_lcg<NOR>(s3.y, o3.y, x3.y, o2.y, oD.y, sb.w, P);
                mine[0] = make_uint2(s0.x ^ f0.x, s0.y ^ f0.y);
                mine[Lh] = make_uint2(s1.x ^ f1.x, s1.y ^ f1.y);
                mine[2 * Lh] = make_uint2(s2.x ^ f2.x, s2.y ^ f2.y);
                mine[3 * Lh] = make_uint2(s3.x ^ f3.x, s3.y ^ f3.y);
                mine += 4 * Lh; oth += 4 * Lh; quad += Lh;
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }
    for (int c = 0; c < 2; ++c)
        for (int i = tid; i < half; i += T) {
            const uint2 v = tile2[c * half + i];
            abase[c * gcol + goff + i] = v.x;
            if (vb) bbase[c * gcol + goff + i] = v.y;
        }
}

// ------------------------------------------------------------------------------------------------
// Simple-cubic lattice (O16).  The same scheme one dimension up: a cluster of C CTAs owns a group, each CTA
// stages Lz/C whole z-planes of both colours (rows r = z*Ly + y, H = Ly*Lz/C of them), and only the z-neighbours of a strip's
// first and last plane live in the neighbouring CTA's shared memory.  Per word: six neighbour words, a bit-sliced count of the
// six anti-parallel flags (two full adders and a half adder), the same 8 Philox calls, and THREE threshold tests per lane
// (dE = 12 - 4u in {4, 8, 12}):  flip = [u>=3] | (x<T4 & [u>=2]) | (x<T8 & [u>=1]) | x<T12   (T12 <= T8 <= T4).
// An edge of length 2 makes the two neighbour slots of that direction the same word: it simply enters the count twice.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t pa_flip_mask3d(uint32_t s, uint32_t n0, uint32_t n1, uint32_t n2, uint32_t n3, uint32_t n4,
                                                   uint32_t n5, uint32_t site, uint32_t c0base, uint32_t lo1u, const SweepParams& P) {
    const uint32_t a0 = s ^ n0, a1 = s ^ n1, a2 = s ^ n2, a3 = s ^ n3, a4 = s ^ n4, a5 = s ^ n5;
    const uint32_t s1 = a0 ^ a1 ^ a2, c1 = (a0 & a1) | (a2 & (a0 ^ a1));
    const uint32_t s2 = a3 ^ a4 ^ a5, c2 = (a3 & a4) | (a5 & (a3 ^ a4));
    const uint32_t low = s1 ^ s2, c3 = s1 & s2;                       // u = low + 2 (c1 + c2 + c3)
    const uint32_t b1 = c1 ^ c2 ^ c3, b2 = (c1 & c2) | (c3 & (c1 ^ c2));
    const uint32_t U1 = low | b1 | b2, U2 = b1 | b2, U3 = b2 | (b1 & low);
    // ---- 8 Philox4x32-10 calls, counters (site, 8g+i, 2t+c, TAG_SWEEP), i = 0..7 (O1): as in pa_flip_mask ----
    uint32_t x0[8], x1[8], x2[8], x3[8];
    uint32_t hi0, lo0;
    pa_mulhilo(PA_PHILOX_M0, site, hi0, lo0);
    const uint32_t c2w = hi0 ^ PA_TAG_SWEEP ^ P.K.k1[0];
    const uint32_t c3w = lo0;
    uint32_t hi1w, lo1w;
    pa_mulhilo(PA_PHILOX_M1, c2w, hi1w, lo1w);
    const uint32_t c0w = hi1w ^ lo1u ^ P.K.k0[1];
    const uint32_t c1w = lo1w;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M0, c0base ^ (uint32_t)i, h, l);
        x2[i] = h ^ c3w ^ P.K.k1[1];
        x3[i] = l;
    }
    uint32_t hi0w, lo0w;
    pa_mulhilo(PA_PHILOX_M0, c0w, hi0w, lo0w);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t h, l;
        pa_mulhilo(PA_PHILOX_M1, x2[i], h, l);
        x0[i] = h ^ c1w ^ P.K.k0[2];
        x1[i] = l;
        x2[i] = hi0w ^ x3[i] ^ P.K.k1[2];
        x3[i] = lo0w;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            uint32_t h0, l0, h1, l1;
            pa_mulhilo(PA_PHILOX_M0, x0[i], h0, l0);
            pa_mulhilo(PA_PHILOX_M1, x2[i], h1, l1);
            x0[i] = h1 ^ x1[i] ^ P.K.k0[r];
            x1[i] = l1;
            x2[i] = h0 ^ x3[i] ^ P.K.k1[r];
            x3[i] = l0;
        }
    }
    uint32_t g4 = 0, g8 = 0, g12 = 0;              // bit b = (x_b >= T): built most-significant bit first
#pragma unroll
    for (int i = 7; i >= 0; --i) {
        const uint32_t xs[4] = {x0[i], x1[i], x2[i], x3[i]};
#pragma unroll
        for (int q = 3; q >= 0; --q) {
            pa_shift_in_ge(g4, xs[q], P.T4, P.two);
            pa_shift_in_ge(g8, xs[q], P.T8, P.two);
            pa_shift_in_ge(g12, xs[q], P.T12, P.two);
        }
    }
    return U3 | (~g4 & U2) | (~g8 & U1) | ~g12;
}

// LOG_LH, LOG_LY >= 0: Lx/2 and Ly are these powers of two (cubes 8^3 .. 64^3: the index arithmetic is shifts and masks);
// -1: any even edges (two integer divisions per word).
template <bool CLUSTER, int LOG_LH, int LOG_LY>
__global__ void __launch_bounds__(256, 3)
pa_sweep3d_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint32_t tile[];   // [2][H][Lh], H = Ly * (Lz / C) rows
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    const long long g = blockIdx.x / C;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;        // uniform per cluster
    const int H = P.H, Lh = LOG_LH >= 0 ? (1 << LOG_LH) : P.Lh, Lx = 2 * Lh, Ly = LOG_LY >= 0 ? (1 << LOG_LY) : P.Ly;
    const int Pz = LOG_LY >= 0 ? (H >> LOG_LY) : H / Ly;  // planes of this CTA
    const int z0 = (int)cr * Pz;
    const int half = H * Lh;
    uint32_t* gbase = pop + g * (long long)P.N;
    const int goff = z0 * Ly * Lh, gcol = P.N >> 1;
    if ((half & 3) == 0) {
        for (int c = 0; c < 2; ++c) {
            const uint4* src = reinterpret_cast<const uint4*>(gbase + c * gcol + goff);
            uint4* dst = reinterpret_cast<uint4*>(tile + c * half);
            for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
        }
    } else {
        for (int c = 0; c < 2; ++c)
            for (int i = tid; i < half; i += T) tile[c * half + i] = gbase[c * gcol + goff + i];
    }
    const uint32_t* up_tile = tile;
    const uint32_t* dn_tile = tile;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }
    const uint32_t g8 = (uint32_t)(8 * g);
    const int plane = Ly * Lh;
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t hi1u, lo1u;
            pa_mulhilo(PA_PHILOX_M1, c2, hi1u, lo1u);
            const uint32_t c0base = hi1u ^ P.K.k0[0] ^ g8;
            uint32_t* mine = tile + c * half;
            const uint32_t* oth = tile + (1 - c) * half;
            const uint32_t* up_oth = up_tile + (1 - c) * half;
            const uint32_t* dn_oth = dn_tile + (1 - c) * half;
#pragma unroll 1
            for (int w = tid; w < half; w += T) {
                const int rl = LOG_LH >= 0 ? (w >> LOG_LH) : w / Lh, xh = w - rl * Lh;
                const int zl = LOG_LY >= 0 ? (rl >> LOG_LY) : rl / Ly, y = rl - zl * Ly;
                const int z = z0 + zl;
                const int p = (y + z + c) & 1;
                const int in_plane = y * Lh + xh, pl = zl * plane;
                const uint32_t s = mine[w];
                const uint32_t nS = oth[w];
                const int xh2 = p ? (xh + 1 == Lh ? 0 : xh + 1) : (xh == 0 ? Lh - 1 : xh - 1);
                const uint32_t nX = oth[w - xh + xh2];
                const uint32_t nYm = oth[pl + (y == 0 ? Ly - 1 : y - 1) * Lh + xh];
                const uint32_t nYp = oth[pl + (y + 1 == Ly ? 0 : y + 1) * Lh + xh];
                uint32_t nZm, nZp;
                if (zl > 0) nZm = oth[w - plane]; else nZm = up_oth[(Pz - 1) * plane + in_plane];
                if (zl < Pz - 1) nZp = oth[w + plane]; else nZp = dn_oth[in_plane];
                const uint32_t site = (uint32_t)((z * Ly + y) * Lx + 2 * xh + p);
                mine[w] = s ^ pa_flip_mask3d(s, nS, nX, nYm, nYp, nZm, nZp, site, c0base, lo1u, P);
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }
    if ((half & 3) == 0) {
        for (int c = 0; c < 2; ++c) {
            uint4* dst = reinterpret_cast<uint4*>(gbase + c * gcol + goff);
            const uint4* src = reinterpret_cast<const uint4*>(tile + c * half);
            for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
        }
    } else {
        for (int c = 0; c < 2; ++c)
            for (int i = tid; i < half; i += T) gbase[c * gcol + goff + i] = tile[c * half + i];
    }
}

// Column walk for cubes of 8 .. 64 (edges 2 Lh = Ly = Lz): a thread owns the column (y, xh) of its CTA's planes and walks down z two
// planes at a time, as pa_sweep_col_kernel walks down the rows.  Every shared-memory address is the thread's pointer plus a
// compile-time immediate (x and y wrap offsets are per-thread constants, the z neighbours of a pair are words the pair has loaded
// anyway), the site index advances by a constant: the two dozen index instructions per word of pa_sweep3d_kernel disappear.
// Requirements (pa_launch_sweep_3d): planes per CTA even, T = min(256, columns * planes / 2).
template <bool CLUSTER, int LOG_LH>
__global__ void __launch_bounds__(LOG_LH == 5 ? 512 : 256, LOG_LH == 5 ? 1 : 3)      // 64^3: 128 KB strips, one CTA of 16 warps per SM
pa_sweep3d_col_kernel(uint32_t* __restrict__ pop, const SweepParams P) {
    extern __shared__ __align__(16) uint32_t tile[];   // [2][Pz][Ly][Lh]
    constexpr int Lh = 1 << LOG_LH, Ly = 2 * Lh, Lx = 2 * Lh, LOG_COLS = 2 * LOG_LH + 1, cols = 1 << LOG_COLS, plane = cols;
    const int T = blockDim.x, tid = threadIdx.x;
    const int C = CLUSTER ? P.C : 1;
    unsigned cr = 0;
    if (CLUSTER) cr = cg::this_cluster().block_rank();
    const long long g = blockIdx.x / C;
    pa_pdl_wait(); pa_pdl_launch();
    if (g * 32 >= pa_live_R(P.R, P.sc)) return;        // uniform per cluster
    const int Pz = P.H >> (LOG_LH + 1);                // planes of this CTA (even)
    const int z0 = (int)cr * Pz;
    const int half = Pz * plane;
    uint32_t* gbase = pop + g * (long long)P.N;
    const int goff = z0 * plane, gcol = P.N >> 1;
    for (int c = 0; c < 2; ++c) {
        const uint4* src = reinterpret_cast<const uint4*>(gbase + c * gcol + goff);
        uint4* dst = reinterpret_cast<uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
    const uint32_t* up_tile = tile;
    const uint32_t* dn_tile = tile;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        up_tile = cl.map_shared_rank(tile, (cr + C - 1) % C);
        dn_tile = cl.map_shared_rank(tile, (cr + 1) % C);
        cl.sync();
    } else {
        __syncthreads();
    }
    const uint32_t g8 = (uint32_t)(8 * g);
    const int nseg = T > cols ? (T >> LOG_COLS) : 1;   // z segments per column when there are more threads than columns
    const int zps = Pz / nseg;                         // planes per thread and column: even, >= 2
    const int items = cols * nseg;
    for (int it = 0; it < P.theta; ++it) {
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const uint32_t c2 = 2u * (P.t0 + (uint32_t)it) + (uint32_t)c;
            uint32_t hi1u, lo1u;
            pa_mulhilo(PA_PHILOX_M1, c2, hi1u, lo1u);
            const uint32_t c0base = hi1u ^ P.K.k0[0] ^ g8;
#pragma unroll 1
            for (int item = tid; item < items; item += T) {
                const int col = item & (cols - 1), seg = item >> LOG_COLS;
                const int y = col >> LOG_LH, xh = col & (Lh - 1);
                const int za = seg * zps;                                       // first local plane: even, and z0 is even
                const int dYm = y == 0 ? (Ly - 1) * Lh : -Lh, dYp = y == Ly - 1 ? -(Ly - 1) * Lh : Lh;
                const int dL = ((xh - 1) & (Lh - 1)) - xh, dR = ((xh + 1) & (Lh - 1)) - xh;
                const int p0 = (y + c) & 1;                                     // x-parity of the even planes; odd planes: 1 - p0
                const int dA = p0 ? dR : dL, dB = p0 ? dL : dR;
                uint32_t* m = tile + c * half + za * plane + col;
                const uint32_t* o = tile + (1 - c) * half + za * plane + col;
                uint32_t site = (uint32_t)(((z0 + za) * Ly + y) * Lx + 2 * xh + p0);
                const uint32_t dsite = (uint32_t)(Ly * Lx + 1 - 2 * p0);        // to the site of the next plane in this column
#pragma unroll 1
                for (int k = 0; k < zps; k += 2) {
                    const uint32_t s0 = m[0], s1 = m[plane];
                    const uint32_t o0 = o[0], o1 = o[plane];
                    const uint32_t x0 = o[dA], x1 = o[plane + dB];
                    const uint32_t ym0 = o[dYm], yp0 = o[dYp], ym1 = o[plane + dYm], yp1 = o[plane + dYp];
                    uint32_t zm0, zp1;
                    if (za + k > 0) zm0 = o[-plane]; else zm0 = up_tile[(1 - c) * half + (Pz - 1) * plane + col];
                    if (za + k + 2 < Pz) zp1 = o[2 * plane]; else zp1 = dn_tile[(1 - c) * half + col];
                    const uint32_t f0 = pa_flip_mask3d(s0, o0, x0, ym0, yp0, zm0, o1, site, c0base, lo1u, P);
                    const uint32_t f1 = pa_flip_mask3d(s1, o1, x1, ym1, yp1, o0, zp1, site + dsite, c0base, lo1u, P);
                    m[0] = s0 ^ f0;
                    m[plane] = s1 ^ f1;
                    m += 2 * plane; o += 2 * plane; site += (uint32_t)(2 * Ly * Lx);
                }
            }
            if (CLUSTER) cg::this_cluster().sync(); else __syncthreads();
        }
    }
    for (int c = 0; c < 2; ++c) {
        uint4* dst = reinterpret_cast<uint4*>(gbase + c * gcol + goff);
        const uint4* src = reinterpret_cast<const uint4*>(tile + c * half);
        for (int i = tid; i < (half >> 2); i += T) dst[i] = src[i];
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------

// Launch geometry.  C_min = the smallest cluster size in {1,2,4,8} dividing L whose strip (L/C rows of both
// colours, L*L*4/C bytes) fits the shared-memory budget per CTA; threads = min(256, words per colour).
// kind 1 = column-walk kernel (power-of-two L >= 64), kind 0 = generic kernel (any even L).
// Environment overrides (tests, tuning): PA_SWEEP_C, PA_SWEEP_T, PA_SWEEP_KIND, PA_SWEEP_CMP, PA_SWEEP_SMEM_KB.
static bool pa_col_ok(int L, int C, int T, int rng_mode = PA_RNG_PHILOX) {
    if ((L & (L - 1)) != 0 || L < 64 || L % C != 0) return false;
    const int Lh = L / 2, H = L / C, half = H * Lh;
    const int q = rng_mode == PA_RNG_LCG ? 4 : 2;          // rows per iteration of the column walk
    return H % q == 0 && T >= Lh && (T & (T - 1)) == 0 && half % T == 0 && half / T >= q && (half / T) % q == 0;
}

// O16: the smallest cluster size C in {1,2,4,8} dividing Lz whose Lz/C planes fit the preferred 64 KB (else 224 KB).
static int pa_sweep_configure_3d(pa_handle* h) {
    const size_t bytes = (size_t)h->N * 4;
    const int Lz = h->geom.Lz;
    int C = 0;
    for (int lim = 64; lim <= 224 && !C; lim += 160)
        for (int c = 1; c <= 8 && !C; c *= 2)
            if (Lz % c == 0 && bytes / c <= (size_t)lim * 1024) C = c;
    const int forceC = (int)pa_sw(h, PA_SW_SWEEP_C, 0);
    h->sweep_C_forced = false;
    if (forceC > 0 && forceC <= 8 && (forceC & (forceC - 1)) == 0 && Lz % forceC == 0 && bytes / forceC <= (size_t)224 * 1024) { C = forceC; h->sweep_C_forced = true; }
    if (!C) return PA_ERR_INVALID_ARG;
    const int half = h->N / 2 / C;
    int T = 256;
    while (T > 32 && T > half) T >>= 1;
    const int forceT = (int)pa_sw(h, PA_SW_SWEEP_T, 0);
    if (forceT >= 32 && forceT <= 256) T = forceT;
    h->sweep_C = C; h->sweep_T = T; h->sweep_kind = 0; h->sweep_cmp = 1;
    return PA_OK;
}

int pa_sweep_configure(pa_handle* h) {
    if (h->D == 3) return pa_sweep_configure_3d(h);
    const int L = h->L;
    // strips of up to 64 KB (three CTAs of 256 threads per SM); L = 256: 128 KB strips, clusters of two, one CTA of 512 threads per SM
    const bool big = L == 256;
    const size_t budget = (size_t)(int)pa_sw(h, PA_SW_SWEEP_SMEM_KB, big ? 128 : 64) * 1024;
    int C = 1;
    while (C <= 8 && (((L % C) != 0) || (size_t)L * L * 4 / C > budget)) C *= 2;
    if (C > 8) {                                   // L = 512: no strip fits the preferred budget; take the largest that fits an SM
        C = 1;
        while (C <= 8 && (((L % C) != 0) || (size_t)L * L * 4 / C > (size_t)224 * 1024)) C *= 2;
    }
    h->sweep_C_forced = false;
    int forceC = (int)pa_sw(h, PA_SW_SWEEP_C, 0);
    if (forceC > 0 && L % forceC == 0) { C = forceC; h->sweep_C_forced = true; }
    if (C > 8 || (size_t)L * L * 4 / C > 224 * 1024) return PA_ERR_INVALID_ARG;
    int half = (L / C) * (L / 2);
    int T = big ? 512 : 256;
    while (T > 32 && T > half) T >>= 1;
    int forceT = (int)pa_sw(h, PA_SW_SWEEP_T, 0);
    if (forceT >= 32 && forceT <= (big ? 512 : 256)) T = forceT;
    int kind = pa_col_ok(L, C, T) ? 1 : 0;
    kind = (int)pa_sw(h, PA_SW_SWEEP_KIND, kind);
    if (kind == 1 && !pa_col_ok(L, C, T)) kind = 0;
    if (kind == 0 && T > 256) T = 256;                       // the generic kernel is compiled for blocks of up to 256 threads
    h->sweep_C = C; h->sweep_T = T; h->sweep_kind = kind;
    h->sweep_cmp = (int)pa_sw(h, PA_SW_SWEEP_CMP, 1);
    if (h->sweep_cmp < 0 || h->sweep_cmp > 2) h->sweep_cmp = 1;
    return PA_OK;
}

// Small and medium populations: the kernel is pipe-bound, so an SM's time is proportional to the number of CTAs it works
// through, whatever their residency: n CTAs on 148 SMs run at (n/148) / ceil(n/148) of the full-machine rate (measured, round 1:
// cfg2 with one CTA per group 625/148 -> 4.22/5 = 0.845 against 0.835 measured; two CTAs per group 8.45/9 x 0.97 = 0.91 against
// 0.90; L = 128, R = 50 000 with one CTA per group 10.6/11 = 0.96 against 0.977).  Splitting every group over a cluster of C CTAs
// makes the work items smaller at a measured cluster cost (C = 2: 0.97; C = 4: 0.93, 0.85 when a thread is left with one row
// pair; C = 8: 0.85).  The earlier "waves of resident CTAs" model mispredicted L = 128 at R = 50 000 (chose C = 4: 1 536
// updates/ns; C = 1: 1 644).
static double pa_cluster_cost(int C, int rows_per_thread) {
    return C == 1 ? 1.0 : C == 2 ? 0.97 : C == 4 ? (rows_per_thread >= 4 ? 0.93 : 0.85) : 0.85;
}

// Returns the cluster size; *n_main >= 0 selects a MIXED launch without clusters: CTAs 0 .. n_main-1 own a whole group each and
// fill floor(G/148) complete rounds of the 148 SMs; every remaining group -- which would otherwise occupy a round of its own on a
// fraction of the SMs -- is shared by four lane-split CTAs (pa_flip_mask_part), scheduled last by block order (cfg2: 625 groups =
// 4 rounds of 148 + 33 groups in lane quarters instead of 9 rounds of half-groups).  Needs a whole group in one CTA (C_min = 1,
// i.e. L <= 128).  PA_SWEEP_MIXED=0 switches it off.
static int pa_sweep_pick_C(const pa_handle* h, int64_t G, long long* n_main) {
    *n_main = -1;
    const int Cmin = h->sweep_C;
    if (h->sweep_C_forced || h->sweep_kind != 1) return Cmin;
    const int L = h->L;
    const double S = (double)h->n_sm;
    if ((double)G * Cmin / S >= 24.0) return Cmin;                 // quantisation below 4 %
    double best = -1.0; int bestC = Cmin;
    for (int C = Cmin; C <= 8; C *= 2) {
        if (!pa_col_ok(L, C, h->sweep_T, h->rng_mode)) break;
        const int rows_per_thread = (L / C) * (L / 2) / h->sweep_T;
        const double per_sm = (double)G * C / S;
        const double eff = per_sm / ceil(per_sm) * pa_cluster_cost(C, rows_per_thread) * (C == Cmin ? 1.0 : 0.995);   // ties go to the smaller cluster
        if (eff > best) { best = eff; bestC = C; }
    }
    if (Cmin != 1 || h->has_j || (int)pa_sw(h, PA_SW_SWEEP_MIXED, 1) == 0 || !pa_col_ok(L, 1, h->sweep_T, h->rng_mode)) return bestC;
    if (h->rng_mode == PA_RNG_LCG && (int)pa_sw(h, PA_SW_LCG_P64, 0) == 1) return bestC;
    // inside pa_anneal the grid covers the capacity; the live population is about the target
    const int64_t G_live = h->dev_R ? (h->R_target + 31) / 32 : G;
    const int64_t rounds = G_live / h->n_sm;
    const int64_t Gm = rounds * h->n_sm, Gt = G_live - Gm;
    if (rounds < 1 || Gt <= 0) return bestC;
    // a lane quarter costs about 0.3 of a whole group (35 instead of 131/4 wide multiplies, repeated neighbour logic)
    const double time = (double)rounds + ceil((double)Gt * 4 / S) * 0.30;
    const double eff = ((double)G_live / S) / time * 0.985;         // must beat the uniform launch by 1.5 % to be taken
    if (eff > best) { bestC = 1; *n_main = Gm; }
    return bestC;
}

template <typename Kern>
static cudaError_t pa_sweep_launch_k(pa_handle* h, Kern kern, const SweepParams& P, size_t smem, unsigned grid, bool cluster, int T = 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3((unsigned)(T > 0 ? T : h->sweep_T), 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cluster ? (unsigned)P.C : 1u;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;       // see pa_common.cuh
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = h->pdl ? 2 : 1;
    return cudaLaunchKernelEx(&cfg, kern, h->spins[h->cur], P);
}

template <int NOR, bool HASJ>
static cudaError_t pa_sweep_dispatch_lcg_col(pa_handle* h, const SweepParams& P, size_t smem, unsigned grid) {
    const bool cl = P.C > 1;
    switch (P.Lh) {
#define PA_COL_CASE(LOG) case (1 << LOG): return cl ? pa_sweep_launch_k(h, pa_sweep_lcg_kernel<LOG, true, NOR, HASJ>, P, smem, grid, true) \
                                                  : pa_sweep_launch_k(h, pa_sweep_lcg_kernel<LOG, false, NOR, HASJ>, P, smem, grid, false);
        PA_COL_CASE(5) PA_COL_CASE(6) PA_COL_CASE(7) PA_COL_CASE(8)
#undef PA_COL_CASE
        default: return cudaErrorInvalidValue;
    }
}

static cudaError_t pa_sweep_dispatch_lcg(pa_handle* h, const SweepParams& P, size_t smem, unsigned grid) {
    const bool cl = P.C > 1;
    // p = 64 words: PA_LCG_P64=1 wherever the kernel applies, =0 never; unset: at L = 64 (+2.7 % there, -12 % at L = 128:
    // profiles/r02b_p64.md) for a uniform launch of the whole population (the mixed launch and pa_step_host's ranges stay on p = 32)
    const int p64 = (int)pa_sw(h, PA_SW_LCG_P64, -1);
    const bool p64_on = p64 == 1 || (p64 < 0 && P.L == 64 && P.C == 1 && P.n_main < 0 && P.whole != 0 && grid >= 24u * (unsigned)h->n_sm);
    if (h->sweep_kind == 1 && !h->has_j && p64_on && pa_col_ok(P.L, P.C, h->sweep_T, PA_RNG_LCG) &&
        P.Lh >= 32 && P.Lh <= 128 && 2 * smem <= (size_t)224 * 1024) {
        // p = 64 experiment: one CTA (cluster) per PAIR of groups, twice the shared memory
        const unsigned grid2 = (unsigned)(((grid / P.C) + 1) / 2 * P.C);
        if (P.Lh == 32 || P.Lh == 64 || P.Lh == 128) h->last_sweep_kind |= PA_SWEEP_RAN_P64;
        switch (P.Lh) {
#define PA_COL_CASE(LOG) case (1 << LOG): return cl ? pa_sweep_launch_k(h, pa_sweep_lcg64_kernel<LOG, true, 4>, P, 2 * smem, grid2, true) \
                                                  : pa_sweep_launch_k(h, pa_sweep_lcg64_kernel<LOG, false, 4>, P, 2 * smem, grid2, false);
            PA_COL_CASE(5) PA_COL_CASE(6) PA_COL_CASE(7)
#undef PA_COL_CASE
            default: break;
        }
    }
    if (h->sweep_kind == 1 && pa_col_ok(P.L, P.C, h->sweep_T, PA_RNG_LCG) && P.Lh >= 32 && P.Lh <= 256) {
        if (h->has_j) return pa_sweep_dispatch_lcg_col<4, true>(h, P, smem, grid);
        switch ((int)pa_sw(h, PA_SW_LCG_NOR, 4)) {       // tuning knob; every value gives the same bytes
            case 0: return pa_sweep_dispatch_lcg_col<0, false>(h, P, smem, grid);
            case 2: return pa_sweep_dispatch_lcg_col<2, false>(h, P, smem, grid);
            case 6: return pa_sweep_dispatch_lcg_col<6, false>(h, P, smem, grid);
            case 8: return pa_sweep_dispatch_lcg_col<8, false>(h, P, smem, grid);
            default: return pa_sweep_dispatch_lcg_col<4, false>(h, P, smem, grid);
        }
    }
    if (h->has_j)
        return cl ? pa_sweep_launch_k(h, pa_sweep_kernel<1, true, PA_RNG_LCG, true>, P, smem, grid, true)
                  : pa_sweep_launch_k(h, pa_sweep_kernel<1, false, PA_RNG_LCG, true>, P, smem, grid, false);
    return cl ? pa_sweep_launch_k(h, pa_sweep_kernel<1, true, PA_RNG_LCG, false>, P, smem, grid, true)
              : pa_sweep_launch_k(h, pa_sweep_kernel<1, false, PA_RNG_LCG, false>, P, smem, grid, false);
}

template <int CMP>
static cudaError_t pa_sweep_dispatch(pa_handle* h, const SweepParams& P, size_t smem, unsigned grid) {
    const bool cl = P.C > 1;
    if (h->sweep_kind == 1) {
        switch (P.Lh) {
#define PA_COL_CASE(LOG) case (1 << LOG): return cl ? pa_sweep_launch_k(h, pa_sweep_col_kernel<CMP, LOG, true, false>, P, smem, grid, true) \
                                                      : pa_sweep_launch_k(h, pa_sweep_col_kernel<CMP, LOG, false, false>, P, smem, grid, false);
            PA_COL_CASE(5) PA_COL_CASE(6) PA_COL_CASE(7) PA_COL_CASE(8)
#undef PA_COL_CASE
            default: break;
        }
    }
    return cl ? pa_sweep_launch_k(h, pa_sweep_kernel<CMP, true, PA_RNG_PHILOX, false>, P, smem, grid, true)
              : pa_sweep_launch_k(h, pa_sweep_kernel<CMP, false, PA_RNG_PHILOX, false>, P, smem, grid, false);
}

// O15 with one Philox number per spin: column-walk kernel where it applies, else the generic kernel
static cudaError_t pa_sweep_dispatch_j(pa_handle* h, const SweepParams& P, size_t smem, unsigned grid) {
    const bool cl = P.C > 1;
    if (h->sweep_kind == 1) {
        switch (P.Lh) {
#define PA_COL_CASE(LOG) case (1 << LOG): return cl ? pa_sweep_launch_k(h, pa_sweep_col_kernel<1, LOG, true, true>, P, smem, grid, true) \
                                                      : pa_sweep_launch_k(h, pa_sweep_col_kernel<1, LOG, false, true>, P, smem, grid, false);
            PA_COL_CASE(5) PA_COL_CASE(6) PA_COL_CASE(7) PA_COL_CASE(8)
#undef PA_COL_CASE
            default: break;
        }
    }
    return cl ? pa_sweep_launch_k(h, pa_sweep_kernel<1, true, PA_RNG_PHILOX, true>, P, smem, grid, true)
              : pa_sweep_launch_k(h, pa_sweep_kernel<1, false, PA_RNG_PHILOX, true>, P, smem, grid, false);
}

static int pa_launch_sweep_3d(pa_handle* h, uint32_t T4, uint32_t T8, int theta) {
    SweepParams P;
    P.K = h->keys;
    P.T4 = T4; P.T8 = T8; P.T12 = h->T12;
    P.t0 = h->t; P.theta = theta; P.two = 2u;
    const int64_t G = h->dev_R ? h->G_cap : (h->R_cur + 31) / 32;
    P.R = h->dev_R ? -1 : h->R_cur; P.sc = h->d_scal;
    P.L = h->geom.Lx; P.Lh = h->geom.Lx / 2; P.Ly = h->geom.Ly; P.Lz = h->geom.Lz; P.N = h->N;
    P.C = h->sweep_C; P.H = h->geom.Ly * (h->geom.Lz / P.C);
    P.jmask = nullptr; P.Gcap = h->G_cap; P.n_main = -1; P.g0 = 0; P.whole = 1; P.src = nullptr; P.parent = nullptr;
    const size_t smem = (size_t)h->N * 4 / P.C;
    const unsigned grid = (unsigned)(G * P.C);
    cudaError_t e = cudaErrorInvalidValue;
    const bool cl = P.C > 1;
    const int kind = (int)pa_sw(h, PA_SW_SWEEP_KIND, 1);                                    // 1: column walk, 2: shift/mask index arithmetic, 0: generic
    const int lx = P.L == P.Ly && kind != 0 ? P.L : 0;
    const int Pz = P.Lz / P.C;
    if (kind == 1 && P.L == P.Ly && P.L == P.Lz && (P.L == 8 || P.L == 16 || P.L == 32 || P.L == 64) && Pz >= 2 && (Pz & 1) == 0 &&
        (int)pa_sw(h, PA_SW_SWEEP_T, 0) == 0) {
        const int cols = P.Ly * P.Lh;
        int T = P.L == 64 ? 512 : 256;
        while (T > 32 && T > cols * Pz / 2) T >>= 1;
        if (T <= cols * Pz / 2 && (cols >= T || (Pz % (T / cols) == 0 && ((Pz / (T / cols)) & 1) == 0))) {
#define PA_3DC_CASE(LOGH) e = cl ? pa_sweep_launch_k(h, pa_sweep3d_col_kernel<true, LOGH>, P, smem, grid, true, T) \
                                  : pa_sweep_launch_k(h, pa_sweep3d_col_kernel<false, LOGH>, P, smem, grid, false, T)
            switch (P.L) {
                case 8: PA_3DC_CASE(2); break;
                case 16: PA_3DC_CASE(3); break;
                case 32: PA_3DC_CASE(4); break;
                default: PA_3DC_CASE(5); break;
            }
#undef PA_3DC_CASE
            PA_CUDA(h, e);
            h->launches += 1;
            h->last_sweep_kind = PA_SWEEP_RAN_COL;
            return PA_OK;
        }
    }
#define PA_3D_CASE(LOGH, LOGY) e = cl ? pa_sweep_launch_k(h, pa_sweep3d_kernel<true, LOGH, LOGY>, P, smem, grid, true) \
                                      : pa_sweep_launch_k(h, pa_sweep3d_kernel<false, LOGH, LOGY>, P, smem, grid, false)
    switch (lx) {
        case 8: PA_3D_CASE(2, 3); break;
        case 16: PA_3D_CASE(3, 4); break;
        case 32: PA_3D_CASE(4, 5); break;
        case 64: PA_3D_CASE(5, 6); break;
        default: PA_3D_CASE(-1, -1); break;
    }
#undef PA_3D_CASE
    PA_CUDA(h, e);
    h->launches += 1;
    return PA_OK;
}

// Lane split S (CTAs per group) for a small population on the generic path, 0 = one CTA per group: the largest S in {2, 4} that
// still gives every CTA an SM of its own (measured on B200, sweep of theta = 10: L = 16, R = 1000 22.2 -> 14.7 us with S = 4,
// L = 32, R = 1000 45.5 -> 23.2 us; with more groups than SMs the split only adds work: L = 16, R = 10 000 35.8 -> 39.5 us).
// PA_SWEEP_SPLIT forces 0/2/4.
static int pa_sweep_pick_split(const pa_handle* h, int64_t G) {
    if (h->D != 2 || h->sweep_kind != 0 || h->sweep_C != 1 || h->sweep_C_forced) return 0;
    if ((size_t)h->N * 4 > (size_t)64 * 1024) return 0;
    const int force = (int)pa_sw(h, PA_SW_SWEEP_SPLIT, -1);
    if (force == 0 || force == 2 || force == 4) return force;
    const int64_t room = h->n_sm + h->n_sm / 12;                 // 160 CTAs on 148 SMs
    return G * 4 <= room ? 4 : G * 2 <= room ? 2 : 0;
}

static int pa_launch_sweep_split(pa_handle* h, SweepParams& P, int S, int64_t G, bool gather) {
    P.C = 1; P.H = h->L;
    const int half = h->N / 2;
    int T = (half + 31) / 32 * 32;
    if (T > 256) T = 256;
    const size_t smem = (size_t)h->N * 4;
    void (*kern)(uint32_t*, const SweepParams) = nullptr;
    const int lcg = h->rng_mode == PA_RNG_LCG ? 1 : 0, hj = h->has_j ? 1 : 0;
#define PA_SPLIT_PICK(SS, GG, RR, JJ) if (S == SS && gather == GG && lcg == (RR == PA_RNG_LCG ? 1 : 0) && hj == (JJ ? 1 : 0)) kern = pa_sweep_split_kernel<SS, GG, RR, JJ>;
#define PA_SPLIT_PICK4(SS, GG) PA_SPLIT_PICK(SS, GG, PA_RNG_PHILOX, false) PA_SPLIT_PICK(SS, GG, PA_RNG_PHILOX, true) \
                               PA_SPLIT_PICK(SS, GG, PA_RNG_LCG, false) PA_SPLIT_PICK(SS, GG, PA_RNG_LCG, true)
    PA_SPLIT_PICK4(2, false) PA_SPLIT_PICK4(2, true) PA_SPLIT_PICK4(4, false) PA_SPLIT_PICK4(4, true)
#undef PA_SPLIT_PICK4
#undef PA_SPLIT_PICK
    if (!kern) return PA_ERR_INVALID_ARG;
    h->last_sweep_kind = PA_SWEEP_RAN_SPLIT;
    PA_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    PA_CUDA(h, pa_launch(h, kern, dim3((unsigned)(G * S)), dim3((unsigned)T), smem, h->spins[h->cur], P));
    h->launches += 1;
    return PA_OK;
}

// pa_anneal: true if the sweep launch of this step runs on the lane-split kernel and the plan kernel can commit the population
// size (small populations), so that the sweep can stage its strips straight from the old population (no pa_copy_kernel launch)
bool pa_sweep_gathers(const pa_handle* h, int theta) {
    return theta > 0 && h->dev_R && pa_small_plan_ok(h) && pa_sweep_pick_split(h, (h->R_target + 31) / 32) != 0;
}

int pa_launch_sweep_gather(pa_handle* h, uint32_t T4, uint32_t T8, int theta) {
    SweepParams P;
    P.K = h->keys;
    P.T4 = T4; P.T8 = T8; P.T12 = 0u; P.Ly = h->L; P.Lz = 1;
    P.t0 = h->t; P.theta = theta; P.two = 2u;
    P.R = -1; P.sc = h->d_scal;
    P.L = h->L; P.Lh = h->L / 2; P.N = h->N; P.jmask = h->has_j ? h->jmask : nullptr; P.Gcap = h->G_cap; P.n_main = -1; P.g0 = 0; P.whole = 1;
    P.src = h->spins[1 - h->cur]; P.parent = h->parent;
    return pa_launch_sweep_split(h, P, pa_sweep_pick_split(h, (h->R_target + 31) / 32), h->G_cap, true);
}

static int pa_launch_sweep_groups(pa_handle* h, uint32_t T4, uint32_t T8, int theta, int64_t g0, int64_t ng);

int pa_launch_sweep(pa_handle* h, uint32_t T4, uint32_t T8, int theta) { return pa_launch_sweep_groups(h, T4, T8, theta, 0, -1); }

// Groups g0 .. g0+ng-1 only (pa_step_host runs a step in chunks of groups so that finished chunks travel to the host while the
// next ones are swept).  Column-walk kernels, uniform launch, host-side population size; PA_ERR_INVALID_ARG otherwise.
int pa_launch_sweep_range(pa_handle* h, uint32_t T4, uint32_t T8, int theta, int64_t g0, int64_t ng) {
    if (theta == 0 || ng <= 0) return PA_OK;
    if (h->D != 2 || h->sweep_kind != 1 || h->dev_R || g0 < 0 || g0 + ng > (h->R_cur + 31) / 32) return PA_ERR_INVALID_ARG;
    if (h->rng_mode == PA_RNG_LCG && ((int)pa_sw(h, PA_SW_LCG_P64, 0) == 1 || !pa_col_ok(h->L, h->sweep_C, h->sweep_T, PA_RNG_LCG))) return PA_ERR_INVALID_ARG;
    return pa_launch_sweep_groups(h, T4, T8, theta, g0, ng);
}

static int pa_launch_sweep_groups(pa_handle* h, uint32_t T4, uint32_t T8, int theta, int64_t g0, int64_t ng) {
    if (theta == 0) return PA_OK;
    if (h->D == 3) return pa_launch_sweep_3d(h, T4, T8, theta);
    SweepParams P;
    P.K = h->keys;
    P.T4 = T4; P.T8 = T8; P.T12 = 0u; P.Ly = h->L; P.Lz = 1;
    P.t0 = h->t; P.theta = theta; P.two = 2u;
    const int64_t G = h->dev_R ? h->G_cap : (h->R_cur + 31) / 32;
    P.R = h->dev_R ? -1 : h->R_cur; P.sc = h->d_scal;
    if (const int S = pa_sweep_pick_split(h, h->dev_R ? (h->R_target + 31) / 32 : G)) {   // pa_anneal: the grid covers the capacity, the population is about the target
        P.L = h->L; P.Lh = h->L / 2; P.N = h->N; P.jmask = h->has_j ? h->jmask : nullptr; P.Gcap = h->G_cap; P.n_main = -1; P.g0 = 0; P.whole = 1;
        P.src = nullptr; P.parent = nullptr;
        return pa_launch_sweep_split(h, P, S, G, false);
    }
    P.L = h->L; P.Lh = h->L / 2; P.N = h->N; P.g0 = 0; P.whole = ng < 0 ? 1 : 0;
    if (ng >= 0) { P.C = h->sweep_C; P.n_main = -1; P.g0 = g0; }       // a range of groups: the configured cluster size, no mixed launch
    else P.C = pa_sweep_pick_C(h, G, &P.n_main);
    P.H = h->L / P.C;
    const size_t smem = (size_t)P.H * h->L * 4;
    // mixed launch: n_main whole groups, then four lane-split CTAs per remaining group
    const unsigned grid = ng >= 0 ? (unsigned)(ng * P.C) : P.n_main >= 0 ? (unsigned)(P.n_main + 4 * (G - P.n_main)) : (unsigned)(G * P.C);
    const int v = h->sweep_cmp;
    P.jmask = h->has_j ? h->jmask : nullptr;
    P.Gcap = h->G_cap; P.src = nullptr; P.parent = nullptr;
    h->last_sweep_kind = (h->sweep_kind == 1 ? PA_SWEEP_RAN_COL : 0) | (P.n_main >= 0 ? PA_SWEEP_RAN_MIXED | PA_SWEEP_RAN_SPLIT : 0);
    const cudaError_t e = (h->has_j && h->rng_mode != PA_RNG_LCG) ? pa_sweep_dispatch_j(h, P, smem, grid)   // O15, Philox per spin
                        : h->rng_mode == PA_RNG_LCG ? pa_sweep_dispatch_lcg(h, P, smem, grid)
                        : v == 2 ? pa_sweep_dispatch<2>(h, P, smem, grid) : v == 1 ? pa_sweep_dispatch<1>(h, P, smem, grid)
                                                                                    : pa_sweep_dispatch<0>(h, P, smem, grid);
    PA_CUDA(h, e);
    h->launches += 1;
    return PA_OK;
}
