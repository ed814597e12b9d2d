// pa_oracle.cpp -- CPU ORACLE for the population-annealing (PA) hot path of the 2D Ising model (and, O16, the simple-cubic one).
//
// THIS FILE IS TEST INFRASTRUCTURE.  It is the plain, slow, step-by-step statement of what the
// method computes, written from the paper (/root/reference/PAPER.md, cited below as "L<line>")
// and from the readings listed in DESIGN.md section 3 ("O1".."O10").  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
// call it.  It shares no code with the CUDA library under paper_1703_03676_b200/csrc/ and
// neither includes the other.
//
// One uint8 per spin (1 = up = sigma +1, 0 = down), spin[j][s] with s = y*L + x, scalar Philox,
// fp64 everywhere a floating-point number appears.  Loops over replicas are marked
// "#pragma omp parallel for": replicas are independent (L149) and the random stream is
// counter-based (L163), so the result does not depend on the thread count.
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"):
//   philox4x32_10 ........ cuRAND's curand_philox4x32_x.h (independent implementation), bijectivity
//   thresholds ........... closed forms (beta = 0, monotonicity, exact powers of two)
//   sweep (O3) ........... L=4 brute-force Boltzmann distribution (chi^2), global-flip symmetry
//   init / beta=0 ........ closed-form moments of i.i.d. spins
//   energies (O4) ........ brute force with numpy.roll, all-up and checkerboard states
//   weights, lnQ (O5) .... dbeta=0 closed form, histogram regrouping, Kaufman lnZ (4 sigma)
//   copy numbers (O6) .... sum tau = R, r in {floor, floor+1}, identity at dbeta=0, |R_i-R| bound
//   scan / copy (O7) ..... serial scan, new[d]==old[parent(d)], monotone parent map
//   observables (O8) ..... L=4 exact enumeration, Kaufman e and C at L=16 (4 sigma over seeds)
//   multi-histogram (O9) . sum H = R_i, sum H*E = SE, ln Omega vs exact ln g(E) at L=4
//   adaptive step (O10) .. alpha(0) closed form, monotonicity, bracket property
//   reweighting (O12) .... exact g(E) of the 4x4 torus in, exact enumeration averages out; Kaufman
//                          e, C, lnZ at off-grid beta from L=16 runs (5 sigma over seeds)
//   magnetisation reweighting (O14) exact g(E) and exact microcanonical |M|, M^2 sums of the 4x4 torus in, exact
//                          enumeration <|m|>, <m^2> out; L=4 runs at off-grid beta (5 sigma over seeds)
//   couplings J = +-1 (O15) gauge invariance (Mattis couplings J_ab = eps_a eps_b reproduce the gauge-transformed ferromagnetic
//                          trajectory and its energies exactly); brute-force enumeration of a frustrated 4x4 sample
//                          (Boltzmann chi^2, whole PA runs, reweighting)
//   weighted averages (O13) closed forms (weight ratios, M = 1, equal F, shift invariance, dominance);
//                          unbiasedness of exp(lnZ_m) and removal of the small-R bias at L=4 (L99)
//   LCG-assisted stream (O11) seed counter, output word, jump length and lane order recomputed from explicit Philox counters
//                          for one whole sweep at L = 8 and 12, plus pairwise-distinct seed draws over an L = 16 lattice
//                          (tests/test_oracle_lcg_pins.py); recurrence against big-integer arithmetic with the constants the
//                          paper prints (L236); the same L=4 Boltzmann chi^2, global-flip symmetry
//                          and Kaufman pins as the Philox-per-spin sweep; variance ratio of C
//                          against the Philox-per-spin mode (Table 1, last column = 1)
//   simple-cubic box (O16) numpy.roll energies on boxes with three different edges and closed-form states; one sweep restated
//                          in numpy from explicit Philox counters on a 6x4x2 box; brute-force enumeration of the 4x2x2 box
//                          (Boltzmann chi^2, whole PA runs for every observable, ln Q sums, ln Omega) -- tests/test_oracle_cubic_pins.py
//   whole method vs the paper's own figures: "parity unpinned" (Figs. 2-3 data and the authors'
//   code are not available); pinned instead by the exact Ising results above.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// O1  Random stream.  L163: "Philox_4x32_10 ... sequence number determined from the grid and
// block indices of the thread and a global iteration parameter".  Philox4x32-10 as published in
// ref. [33] (L368): 10 rounds; per round  (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
// c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is bumped by the Weyl constants between rounds.
// ---------------------------------------------------------------------------------------------
const uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
const uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                   uint32_t k0, uint32_t k1, uint32_t out[4]) {
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Stream tags (O1): the fourth counter word separates the three uses.
const uint32_t TAG_INIT = 0u, TAG_SWEEP = 1u, TAG_RESAMPLE = 2u;

inline uint32_t key0(uint64_t seed) { return (uint32_t)(seed & 0xffffffffull); }
inline uint32_t key1(uint64_t seed) { return (uint32_t)(seed >> 32); }

// INIT: the 32-bit word for (site s, group g) is philox(s, g>>2, 0, TAG_INIT)[g&3]; the spin of
// replica j at site s is bit (j&31) of the word of group j>>5.   (L55, L65: i.i.d. uniform spins)
inline uint8_t x_init(uint64_t seed, int64_t j, uint32_t s) {
    uint32_t g = (uint32_t)(j >> 5), out[4];
    philox4x32_10(s, g >> 2, 0u, TAG_INIT, key0(seed), key1(seed), out);
    return (uint8_t)((out[g & 3u] >> (uint32_t)(j & 31)) & 1u);
}
// SWEEP: x(j,s,t,c) = philox(s, j>>2, 2t+c, TAG_SWEEP)[j&3]; j = replica slot, t = sweep counter.
inline uint32_t x_sweep(uint64_t seed, int64_t j, uint32_t s, uint32_t t, uint32_t c) {
    uint32_t out[4];
    philox4x32_10(s, (uint32_t)(j >> 2), 2u * t + c, TAG_SWEEP, key0(seed), key1(seed), out);
    return out[j & 3];
}
// O11  LCG-assisted stream (Sec. 4: "combining the underlying RNG with a particularly fast
// in-line generator used to supply the p random numbers used to flip the spins stored in the same
// word ... r_{n+1} = A r_n + C mod 2^32 with A = 1664525 and C = 1013904223 ... seeded by a call to
// the underlying, high-quality generator (Philox)").  Reading (O11): the word of group
// g = j>>5 at site s = (x,y) is re-seeded at EVERY visit (sweep t, colour c = (x+y)&1) with
//   r_0 = philox(quad, g, 2t+c, TAG_LCG)[y&3],   quad = (y>>2)*(L/2) + (x>>1)
// (one Philox call serves the four rows of a quad in one column of one sub-lattice), and the 32
// replicas of the word take the next 32 LCG outputs, most significant lane first:
//   x(32g+b) = r_{32-b},  r_{n+1} = A r_n + C mod 2^32.
const uint32_t TAG_LCG = 3u;
const uint32_t LCG_A = 1664525u, LCG_C = 1013904223u;        // L236, ref. [43]
inline uint32_t lcg_next(uint32_t r) { return LCG_A * r + LCG_C; }   // uint32 arithmetic = mod 2^32
inline uint32_t x_sweep_lcg(uint64_t seed, int64_t j, int L, int x, int y, uint32_t t, uint32_t c) {
    uint32_t out[4];
    uint32_t quad = (uint32_t)((y >> 2) * (L / 2) + (x >> 1));
    philox4x32_10(quad, (uint32_t)(j >> 5), 2u * t + c, TAG_LCG, key0(seed), key1(seed), out);
    uint32_t r = out[y & 3];
    int steps = 32 - (int)(j & 31);
    for (int n = 0; n < steps; ++n) r = lcg_next(r);
    return r;
}
// RESAMPLE: x(j,k) = philox(j>>2, 0, k, TAG_RESAMPLE)[j&3]; k = resample counter.
inline uint32_t x_resample(uint64_t seed, int64_t j, uint32_t k) {
    uint32_t out[4];
    philox4x32_10((uint32_t)(j >> 2), 0u, k, TAG_RESAMPLE, key0(seed), key1(seed), out);
    return out[j & 3];
}

// ---------------------------------------------------------------------------------------------
// O2  Thresholds.  L163 "pre-calculated tables of the Metropolis factors exp(-beta dE)".
// T(p) = (uint32) min(floor(p * 2^32), 2^32 - 1); a flip with dE > 0 is accepted iff x < T.
// ---------------------------------------------------------------------------------------------
uint32_t threshold(double p) {
    double v = std::floor(p * 4294967296.0);
    if (v > 4294967295.0) v = 4294967295.0;
    if (v < 0.0) v = 0.0;
    return (uint32_t)v;
}

// ---------------------------------------------------------------------------------------------
// O3  One checkerboard Metropolis sweep of one replica.  L151-L157 (checkerboard, one
// sub-lattice, synchronise, the other), L73 (Metropolis), Eq. 10 L135 (H = -sum s_i s_j,
// periodic, L137).  u = number of the 4 neighbours anti-parallel to the centre spin;
// dE = 2*sigma*sum_nn sigma = 8 - 4u; flip iff dE <= 0 or x < T(dE).
// Colour 0 = (x+y) even is updated first, then colour 1.
// ---------------------------------------------------------------------------------------------
enum { RNG_PHILOX = 0, RNG_LCG = 1 };   // O1 (one Philox number per spin) / O11 (Philox-seeded LCG)

// O15 (L313 "the case of different couplings including spin glasses"): bimodal couplings J = +-1 on the bonds,
// H = -sum_<ab> J_ab s_a s_b.  Jx[s] couples site s = (x,y) to (x+1,y), Jy[s] couples it to (x,y+1) (periodic);
// NULL = ferromagnet (Eq. 10).  u then counts the UNSATISFIED bonds of the centre spin (J s_a s_b = -1) and
// dE = 8 - 4u as before, so the thresholds and the acceptance rule are unchanged.
void sweep_one_replica(uint8_t* sp, int L, uint64_t seed, int64_t slot, uint32_t t,
                       uint32_t T4, uint32_t T8, int rng_mode, const int8_t* Jx = nullptr, const int8_t* Jy = nullptr) {
    for (uint32_t c = 0; c < 2; ++c) {
        for (int y = 0; y < L; ++y) {
            for (int x = 0; x < L; ++x) {
                if ((uint32_t)((x + y) & 1) != c) continue;
                int s = y * L + x;
                int xm = x == 0 ? L - 1 : x - 1, xp = x == L - 1 ? 0 : x + 1;      // periodic, L137
                int ym = y == 0 ? L - 1 : y - 1, yp = y == L - 1 ? 0 : y + 1;
                int u;
                if (!Jx) {
                    u = (sp[y * L + xm] != sp[s]) + (sp[y * L + xp] != sp[s]) +
                        (sp[ym * L + x] != sp[s]) + (sp[yp * L + x] != sp[s]);
                } else {                                      // bond unsatisfied iff (spins differ) xor (J = -1) ... for J = +1: differ
                    u = ((sp[y * L + xm] != sp[s]) != (Jx[y * L + xm] < 0)) + ((sp[y * L + xp] != sp[s]) != (Jx[s] < 0)) +
                        ((sp[ym * L + x] != sp[s]) != (Jy[ym * L + x] < 0)) + ((sp[yp * L + x] != sp[s]) != (Jy[s] < 0));
                }
                uint32_t xr = rng_mode == RNG_LCG ? x_sweep_lcg(seed, slot, L, x, y, t, c)
                                                  : x_sweep(seed, slot, (uint32_t)s, t, c);   // drawn for every (j,s,t)
                bool flip = (u >= 2) || (u == 1 && xr < T4) || (u == 0 && xr < T8);
                if (flip) sp[s] ^= 1u;
            }
        }
    }
}

// O4  Energy and magnetisation of one replica.  Eq. 10 L135 (each bond once: right and down
// neighbour of every site), L173.  E = -sum_bonds sigma_a sigma_b, M = sum sigma.
void energy_one_replica(const uint8_t* sp, int L, int32_t* E, int32_t* M, const int8_t* Jx = nullptr, const int8_t* Jy = nullptr) {
    int32_t e = 0, m = 0;
    for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            int sg = sp[y * L + x] ? 1 : -1;
            int sr = sp[y * L + (x == L - 1 ? 0 : x + 1)] ? 1 : -1;
            int sd = sp[(y == L - 1 ? 0 : y + 1) * L + x] ? 1 : -1;
            e -= Jx ? sg * ((int)Jx[y * L + x] * sr + (int)Jy[y * L + x] * sd) : sg * (sr + sd);
            m += sg;
        }
    *E = e; *M = m;
}

// ---------------------------------------------------------------------------------------------
// O16  Simple-cubic lattice (L313 "models on different lattices in various dimensions", L43 "3D Ising systems"; the paper
// gives no detail beyond "straightforward").  Reading (O16): a periodic box Lx x Ly x Lz, every edge even (so that
// the two-colour checkerboard (x+y+z)&1 survives the wrap), site s = (z*Ly + y)*Lx + x.  A spin has six neighbour SLOTS
// x+-1, y+-1, z+-1 (mod the edge); along an edge of length 2 both slots hold the same site, which then counts twice (the
// usual periodic "double bond").  u = number of anti-parallel slots, dE = 2 sigma sum_slots sigma' = 12 - 4u; Metropolis (L73):
// flip iff u >= 3, or u = 2 and x < T4, or u = 1 and x < T8, or u = 0 and x < T12, T(dE) = threshold(exp(-beta dE)) (O2);
// colour 0 first, the random number of (slot, s, t, c) is the SWEEP stream's x_sweep with this s (O1).
// Energy: every site owns its +x, +y, +z bond: E = -sum_s sigma_s (sigma_{x+1} + sigma_{y+1} + sigma_{z+1}), 3N bonds (a double
// bond is owned by both of its sites), so E = -3N + 4m with m = 0 .. 3N/2.
// ---------------------------------------------------------------------------------------------
void sweep_one_replica_3d(uint8_t* sp, int Lx, int Ly, int Lz, uint64_t seed, int64_t slot, uint32_t t,
                          uint32_t T4, uint32_t T8, uint32_t T12) {
    for (uint32_t c = 0; c < 2; ++c)
        for (int z = 0; z < Lz; ++z)
            for (int y = 0; y < Ly; ++y)
                for (int x = 0; x < Lx; ++x) {
                    if ((uint32_t)((x + y + z) & 1) != c) continue;
                    int s = (z * Ly + y) * Lx + x;
                    int xm = x == 0 ? Lx - 1 : x - 1, xp = x == Lx - 1 ? 0 : x + 1;
                    int ym = y == 0 ? Ly - 1 : y - 1, yp = y == Ly - 1 ? 0 : y + 1;
                    int zm = z == 0 ? Lz - 1 : z - 1, zp = z == Lz - 1 ? 0 : z + 1;
                    int u = (sp[(z * Ly + y) * Lx + xm] != sp[s]) + (sp[(z * Ly + y) * Lx + xp] != sp[s]) +
                            (sp[(z * Ly + ym) * Lx + x] != sp[s]) + (sp[(z * Ly + yp) * Lx + x] != sp[s]) +
                            (sp[(zm * Ly + y) * Lx + x] != sp[s]) + (sp[(zp * Ly + y) * Lx + x] != sp[s]);
                    uint32_t xr = x_sweep(seed, slot, (uint32_t)s, t, c);      // drawn for every (j,s,t)
                    bool flip = (u >= 3) || (u == 2 && xr < T4) || (u == 1 && xr < T8) || (u == 0 && xr < T12);
                    if (flip) sp[s] ^= 1u;
                }
}

void energy_one_replica_3d(const uint8_t* sp, int Lx, int Ly, int Lz, int32_t* E, int32_t* M) {
    int32_t e = 0, m = 0;
    for (int z = 0; z < Lz; ++z)
        for (int y = 0; y < Ly; ++y)
            for (int x = 0; x < Lx; ++x) {
                int sg = sp[(z * Ly + y) * Lx + x] ? 1 : -1;
                int sx = sp[(z * Ly + y) * Lx + (x == Lx - 1 ? 0 : x + 1)] ? 1 : -1;
                int sy = sp[(z * Ly + (y == Ly - 1 ? 0 : y + 1)) * Lx + x] ? 1 : -1;
                int sz = sp[((z == Lz - 1 ? 0 : z + 1) * Ly + y) * Lx + x] ? 1 : -1;
                e -= sg * (sx + sy + sz);
                m += sg;
            }
    *E = e; *M = m;
}

// O5  TREE1024: the fixed summation order of the weight sum (L165: "deterministic ... sum the
// per-block partial results in a subsequent kernel call").  Pad with +0.0 to a multiple of 1024;
// inside every aligned run of 32 values: for off = 16,8,4,2,1: a[i] += a[i+off] for i < off;
// the 32 run sums of an aligned block of 1024 are combined by the same 5-level tree; the block
// sums are added sequentially in ascending block index.
double tree1024(const double* a, int64_t n) {
    double total = 0.0;
    for (int64_t b0 = 0; b0 < n; b0 += 1024) {
        double run[32];
        for (int r = 0; r < 32; ++r) {
            double v[32];
            for (int i = 0; i < 32; ++i) {
                int64_t idx = b0 + 32 * r + i;
                v[i] = (idx < n) ? a[idx] : 0.0;
            }
            for (int off = 16; off >= 1; off >>= 1)
                for (int i = 0; i < off; ++i) v[i] += v[i + off];
            run[r] = v[0];
        }
        for (int off = 16; off >= 1; off >>= 1)
            for (int i = 0; i < off; ++i) run[i] += run[i + off];
        total += run[0];
    }
    return total;
}

int64_t capacity_for(int64_t R) {                       // DESIGN.md O7 (paper silent on capacity)
    int64_t slack = (int64_t)std::ceil(8.0 * std::sqrt((double)R));
    if (slack < 1024) slack = 1024;
    return 32 * ((R + slack + 31) / 32);
}

double logaddexp(double a, double b) {
    if (a == -std::numeric_limits<double>::infinity()) return b;
    if (b == -std::numeric_limits<double>::infinity()) return a;
    double hi = a > b ? a : b, lo = a > b ? b : a;
    return hi + std::log1p(std::exp(lo - hi));
}

struct Oracle {
    int L = 0, N = 0;        // N = number of sites (L*L, or Lx*Ly*Lz for a box, O16)
    int D = 2, Lx = 0, Ly = 0, Lz = 1;   // dimension and edges (2D: Lx = Ly = L, Lz = 1)
    int nlev = 0;            // energies lie on -2 nlev + 4m + e0, m = 0..nlev: nlev = (number of bonds)/2 = N (2D), 3N/2 (3D)
    int64_t R_target = 0, R_cur = 0, R_cap = 0;
    uint64_t seed = 0;
    uint32_t t = 0;          // global sweep counter
    int rng_mode = RNG_PHILOX;
    std::vector<int8_t> Jx, Jy;       // [N] bimodal couplings (O15); empty = ferromagnet
    int e0 = 0;                       // E = -2N + 4m + e0 on every reachable state: e0 = 2 (number of J = -1 bonds) mod 4
    uint32_t k = 0;          // resample counter
    double lnZ = 0.0;        // = -beta F(beta), Eq. 4; starts at N ln 2 (L93)
    double lnQ_last = 0.0;
    std::vector<uint8_t> spin;        // [R_cap][N]
    std::vector<int64_t> Hsum;        // [N+1]  running sum of energy histograms, Eq. 9 numerator
    std::vector<double> lnD;          // [N+1]  log of the Eq. 9 denominator
    std::vector<int64_t> A1sum, A2sum; // [N+1]  sums of |M_j| and M_j^2 over all folded replicas with energy level m (O14)
    // last resample, kept for inspection
    double W_last = 0.0;
    std::vector<double> w_last;
    std::vector<uint32_t> r_last, o_last;
};

void all_energies(const Oracle* o, std::vector<int32_t>& E, std::vector<int32_t>& M) {
    E.resize(o->R_cur); M.resize(o->R_cur);
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < o->R_cur; ++j) {
        if (o->D == 3) energy_one_replica_3d(&o->spin[(size_t)j * o->N], o->Lx, o->Ly, o->Lz, &E[j], &M[j]);
        else energy_one_replica(&o->spin[(size_t)j * o->N], o->L, &E[j], &M[j], o->Jx.empty() ? nullptr : o->Jx.data(),
                                o->Jy.empty() ? nullptr : o->Jy.data());
    }
}

// O5 weights for a given dbeta: E_ref = min_j E_j, wtab[d] = exp(-(dbeta*(double)(4d))),
// w_j = wtab[(E_j-E_ref)/4], W = TREE1024(w).   Eq. 1 L58 with the common factor exp(-dbeta E_ref)
// taken out (paper silent on overflow; O5).
void weights_for(const std::vector<int32_t>& E, double dbeta, int32_t* E_ref_out,
                 std::vector<double>& w, double* W) {
    int64_t R = (int64_t)E.size();
    int32_t E_ref = E[0], E_max = E[0];
    for (int64_t j = 1; j < R; ++j) { if (E[j] < E_ref) E_ref = E[j]; if (E[j] > E_max) E_max = E[j]; }
    int32_t dmax = (E_max - E_ref) / 4;
    std::vector<double> wtab(dmax + 1);
    for (int32_t d = 0; d <= dmax; ++d) wtab[d] = std::exp(-(dbeta * (double)(4 * d)));
    w.resize(R);
    for (int64_t j = 0; j < R; ++j) w[j] = wtab[(E[j] - E_ref) / 4];
    *W = tree1024(w.data(), R);
    *E_ref_out = E_ref;
}

// O10 overlap, Eq. 8: alpha = (1/R_cur) sum_j min(1, tau_hat_j), tau_hat_j = R_target*w_j/W
// (= R exp(-dbeta E_j) / (R_cur Q), Eq. 1), summed in the TREE1024 order.
double overlap_for(const std::vector<int32_t>& E, int64_t R_target, double dbeta) {
    std::vector<double> w; double W; int32_t E_ref;
    weights_for(E, dbeta, &E_ref, w, &W);
    int64_t R = (int64_t)E.size();
    std::vector<double> a(R);
    for (int64_t j = 0; j < R; ++j) {
        double tau = ((double)R_target * w[j]) / W;
        a[j] = tau < 1.0 ? tau : 1.0;
    }
    return tree1024(a.data(), R) / (double)R;
}

// O10, L118 "for instance, bisection": hi = beta_max - beta; if alpha(hi) >= target return hi;
// lo = 0; 40 times: mid = (lo+hi)/2; alpha(mid) >= target ? lo = mid : hi = mid; return lo.
double adapt_for(const std::vector<int32_t>& E, int64_t R_target, double target, double hi) {
    if (overlap_for(E, R_target, hi) >= target) return hi;
    double lo = 0.0;
    for (int it = 0; it < 40; ++it) {
        double mid = 0.5 * (lo + hi);
        if (overlap_for(E, R_target, mid) >= target) lo = mid; else hi = mid;
    }
    return lo;
}

struct obs_values { double e, C, absm, m2, m4, betaF_per_N, S_per_N; };

// step 4, L62; Eq. 3, Eq. 4, Eq. 5 L95 from the vectors E_j, M_j and lnZ = -beta F.
obs_values observables_for(const std::vector<int32_t>& E, const std::vector<int32_t>& M, int64_t N,
                           double beta, double lnZ) {
    int64_t R = (int64_t)E.size();
    int64_t SE = 0, SE2 = 0, SA = 0, SM2 = 0;
    std::vector<double> q(R);
    for (int64_t j = 0; j < R; ++j) {
        SE += E[j]; SE2 += (int64_t)E[j] * E[j];
        SA += M[j] < 0 ? -(int64_t)M[j] : (int64_t)M[j];
        SM2 += (int64_t)M[j] * M[j];
        double m = (double)M[j] / (double)N, mm = m * m;
        q[j] = mm * mm;
    }
    double SM4 = tree1024(q.data(), R);
    __int128 num = (__int128)R * (__int128)SE2 - (__int128)SE * (__int128)SE;   // exact
    obs_values v;
    v.e = (double)SE / ((double)R * (double)N);
    v.C = beta * beta * ((double)num / ((double)R * (double)R * (double)N));
    v.absm = (double)SA / ((double)R * (double)N);
    v.m2 = (double)SM2 / ((double)R * (double)N * (double)N);
    v.m4 = SM4 / (double)R;
    v.betaF_per_N = -lnZ / (double)N;
    v.S_per_N = beta * v.e + lnZ / (double)N;
    return v;
}

// O9, Eq. 9: fold the energy histogram at beta into the running sums.
// N here is the number of levels minus one, nlev: the number of sites in 2D (E = -2N + 4m), 3N/2 on the cubic lattice (O16).
void hist_fold_for(const std::vector<int32_t>& E, int N, double lnZ, double beta, int64_t* Hsum, double* lnD, int e0 = 0) {
    int64_t R = (int64_t)E.size();
    std::vector<int64_t> H(N + 1, 0);
    for (int64_t j = 0; j < R; ++j) H[(E[j] + 2 * N - e0) / 4] += 1;
    double lnR = std::log((double)R);
    for (int m = 0; m <= N; ++m) {
        Hsum[m] += H[m];
        double Em = (double)(-2 * N + 4 * m + e0);
        // R_i exp[beta_i F(beta_i) - beta_i E], with -beta_i F = lnZ (Eq. 4)
        lnD[m] = logaddexp(lnD[m], lnR - lnZ - beta * Em);
    }
}

// O12, Sec. 2.4: what Eq. 9 is for.  ln Omega(E_m) = ln Hsum[m] - lnD[m] where Hsum[m] > 0 (Eq. 9 in the log
// domain), and canonical averages at ANY beta follow from the density of states by the textbook sums
//   Z(beta) = sum_m Omega_m exp(-beta E_m),  <E^k> = sum_m E_m^k Omega_m exp(-beta E_m) / Z,
// evaluated with the largest exponent taken out; the variance is summed about the mean (two passes).
//   e = <E>/N,  C = beta^2 (<E^2> - <E>^2)/N  (Eq. 3),  ln Z = -beta F (Eq. 4).
// N = nlev (levels E_m = -2N + 4m + e0, m = 0..N); nsites = number of spins (the same number in 2D; 0 = take N).
void reweight_for(int N, const int64_t* Hsum, const double* lnD, double beta, double* lnZ, double* e, double* C, int e0 = 0, int nsites = 0) {
    if (nsites == 0) nsites = N;
    const double ninf = -std::numeric_limits<double>::infinity();
    double amax = ninf;
    for (int m = 0; m <= N; ++m) {
        if (Hsum[m] <= 0) continue;
        double a = (std::log((double)Hsum[m]) - lnD[m]) - beta * (double)(-2 * N + 4 * m + e0);
        if (a > amax) amax = a;
    }
    double S0 = 0.0, S1 = 0.0;
    for (int m = 0; m <= N; ++m) {
        if (Hsum[m] <= 0) continue;
        double Em = (double)(-2 * N + 4 * m + e0);
        double p = std::exp(((std::log((double)Hsum[m]) - lnD[m]) - beta * Em) - amax);
        S0 += p; S1 += Em * p;
    }
    double mean = S1 / S0, S2 = 0.0;
    for (int m = 0; m <= N; ++m) {
        if (Hsum[m] <= 0) continue;
        double Em = (double)(-2 * N + 4 * m + e0);
        double p = std::exp(((std::log((double)Hsum[m]) - lnD[m]) - beta * Em) - amax);
        S2 += (Em - mean) * (Em - mean) * p;
    }
    *lnZ = amax + std::log(S0);
    *e = mean / (double)nsites;
    *C = beta * beta * (S2 / S0) / (double)nsites;
}

// O14, L129 "Generalizations to other quantities such as magnetizations are possible": microcanonical magnetisation sums.
// At every fold, for every replica j with energy level m_j: A1[m_j] += |M_j|, A2[m_j] += M_j^2 (exact integers).  The mean of
// |M| (M^2) at fixed energy does not depend on beta, so the pooled ratio A[m]/Hsum[m] estimates it from all temperatures, and
//   <|m|>(beta) = sum_m p_m(beta) (A1[m]/Hsum[m]) / N,   <m^2>(beta) = sum_m p_m(beta) (A2[m]/Hsum[m]) / N^2,
// with p_m = Omega_m exp(-beta E_m) / Z from Eq. 9 exactly as in reweight_for.
void mag_fold_for(const std::vector<int32_t>& E, const std::vector<int32_t>& M, int N, int64_t* A1, int64_t* A2, int e0 = 0) {
    for (size_t j = 0; j < E.size(); ++j) {
        int m = (E[j] + 2 * N - e0) / 4;
        int64_t a = M[j] < 0 ? -(int64_t)M[j] : (int64_t)M[j];
        A1[m] += a; A2[m] += a * a;
    }
}
void reweight_mag_for(int N, const int64_t* Hsum, const double* lnD, const int64_t* A1, const int64_t* A2, double beta,
                      double* absm, double* m2, int e0 = 0, int nsites = 0) {
    if (nsites == 0) nsites = N;
    const double ninf = -std::numeric_limits<double>::infinity();
    double amax = ninf;
    for (int m = 0; m <= N; ++m) {
        if (Hsum[m] <= 0) continue;
        double a = (std::log((double)Hsum[m]) - lnD[m]) - beta * (double)(-2 * N + 4 * m + e0);
        if (a > amax) amax = a;
    }
    double S0 = 0.0, Sa = 0.0, Sq = 0.0;
    for (int m = 0; m <= N; ++m) {
        if (Hsum[m] <= 0) continue;
        double Em = (double)(-2 * N + 4 * m + e0);
        double p = std::exp(((std::log((double)Hsum[m]) - lnD[m]) - beta * Em) - amax);
        S0 += p;
        Sa += p * ((double)A1[m] / (double)Hsum[m]);
        Sq += p * ((double)A2[m] / (double)Hsum[m]);
    }
    *absm = (Sa / S0) / (double)nsites;
    *m2 = (Sq / S0) / ((double)nsites * (double)nsites);
}

}  // namespace

extern "C" {

typedef struct { double beta, e, C, absm, m2, m4, betaF_per_N, S_per_N, lnQ; int64_t R; } ora_obs_t;

enum { ORA_OK = 0, ORA_ERR_INVALID_ARG = -1, ORA_ERR_CAPACITY = -2, ORA_ERR_NOMEM = -3 };

// ---- stateless pieces (also used for the sampled parity checks at the large configs) --------

void ora_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], out);
}
uint32_t ora_threshold(double p) { return threshold(p); }
void ora_thresholds(double beta, uint32_t* T4, uint32_t* T8) {
    *T4 = threshold(std::exp(-4.0 * beta));
    *T8 = threshold(std::exp(-8.0 * beta));
}
double ora_tree1024(const double* a, int64_t n) { return tree1024(a, n); }
int64_t ora_capacity(int64_t R) { return capacity_for(R); }

// theta sweeps (O3) of nslots replicas given as spins[nslots][N], replica i living in population
// slot slot_ids[i]; the sweep counter runs t0, t0+1, ..., t0+theta-1.
int ora_sweep_slots_mode(int L, uint64_t seed, uint32_t t0, double beta, int theta,
                         int64_t nslots, const int64_t* slot_ids, uint8_t* spins, int rng_mode) {
    if (L < 4 || (L & 1) || theta < 0 || nslots < 0 || rng_mode < 0 || rng_mode > 1) return ORA_ERR_INVALID_ARG;
    uint32_t T4, T8; ora_thresholds(beta, &T4, &T8);
    int N = L * L;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nslots; ++i)
        for (int it = 0; it < theta; ++it)
            sweep_one_replica(spins + (size_t)i * N, L, seed, slot_ids[i], t0 + (uint32_t)it, T4, T8, rng_mode);
    return ORA_OK;
}
int ora_sweep_slots(int L, uint64_t seed, uint32_t t0, double beta, int theta,
                    int64_t nslots, const int64_t* slot_ids, uint8_t* spins) {
    return ora_sweep_slots_mode(L, seed, t0, beta, theta, nslots, slot_ids, spins, RNG_PHILOX);
}
uint32_t ora_lcg_next(uint32_t r) { return lcg_next(r); }

int ora_energies_of(int L, int64_t n, const uint8_t* spins, int32_t* E, int32_t* M) {
    if (L < 4 || (L & 1) || n < 0) return ORA_ERR_INVALID_ARG;
    int N = L * L;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) {
        int32_t e, m; energy_one_replica(spins + (size_t)j * N, L, &e, &m);
        E[j] = e; if (M) M[j] = m;
    }
    return ORA_OK;
}

// O5-O7 from an energy vector alone: weights, W, copy numbers, offsets, R_new, lnQ.
// Any output pointer may be NULL.  Eq. 1, Eq. 2 L67, L69 (tau_hat = (R/R_{i-1}) tau).
int ora_resample_plan(int64_t R_target, int64_t R_cur, const int32_t* E, uint64_t seed, uint32_t k,
                      double dbeta, double* W_out, double* w_out, uint32_t* r_out, uint32_t* o_out,
                      int64_t* R_new_out, double* lnQ_out) {
    if (R_cur < 1 || R_target < 1) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> Ev(E, E + R_cur);
    std::vector<double> w; double W; int32_t E_ref;
    weights_for(Ev, dbeta, &E_ref, w, &W);
    uint64_t run = 0;
    for (int64_t j = 0; j < R_cur; ++j) {
        double tau = ((double)R_target * w[j]) / W;          // one multiply, one divide (O6)
        double n = std::floor(tau);
        double f = tau - n;                                   // exact
        double u = (double)x_resample(seed, j, k) * (1.0 / 4294967296.0);   // exact, in [0,1)
        uint32_t r = (uint32_t)n + (u < f ? 1u : 0u);        // Eq. 2 with strict '<' (O6)
        if (r_out) r_out[j] = r;
        if (o_out) o_out[j] = (uint32_t)run;                  // exclusive prefix sum (O7, L165)
        if (w_out) w_out[j] = w[j];
        run += r;
    }
    if (W_out) *W_out = W;
    if (R_new_out) *R_new_out = (int64_t)run;
    if (lnQ_out) *lnQ_out = -dbeta * (double)E_ref + std::log(W / (double)R_cur);   // Eq. 1 shifted
    return ORA_OK;
}

double ora_overlap_of(int64_t R_target, int64_t R_cur, const int32_t* E, double dbeta) {
    std::vector<int32_t> Ev(E, E + R_cur);
    return overlap_for(Ev, R_target, dbeta);
}

// O10 from an energy vector alone (sampled parity checks at the large configs)
int ora_adapt_dbeta_of(int64_t R_target, int64_t R_cur, const int32_t* E, double target, double beta,
                       double beta_max, double* dbeta_out) {
    if (R_cur < 1 || !dbeta_out || !(target > 0.0 && target < 1.0) || !(beta_max > beta)) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> Ev(E, E + R_cur);
    *dbeta_out = adapt_for(Ev, R_target, target, beta_max - beta);
    return ORA_OK;
}

// O8 from the vectors E_j, M_j; lnZ and lnQ are the caller's running values (Eq. 4)
int ora_observables_of(int L, int64_t R_cur, const int32_t* E, const int32_t* M, double beta, double lnZ,
                       double lnQ, ora_obs_t* out);

// O9 from an energy vector: Hsum[N+1], lnD[N+1] are updated in place
int ora_hist_fold_of(int L, int64_t R_cur, const int32_t* E, double lnZ, double beta, int64_t* Hsum, double* lnD) {
    if (L < 4 || (L & 1) || R_cur < 1 || !Hsum || !lnD) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> Ev(E, E + R_cur);
    hist_fold_for(Ev, L * L, lnZ, beta, Hsum, lnD);
    return ORA_OK;
}

// O12 from the accumulated sums alone: lnZ, e, C at every beta of a grid
int ora_reweight_of(int L, const int64_t* Hsum, const double* lnD, int n, const double* betas,
                    double* lnZ, double* e, double* C) {
    if (L < 4 || (L & 1) || !Hsum || !lnD || n < 0) return ORA_ERR_INVALID_ARG;
    bool any = false;
    for (int m = 0; m <= L * L; ++m) any = any || Hsum[m] > 0;
    if (!any) return ORA_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) reweight_for(L * L, Hsum, lnD, betas[i], &lnZ[i], &e[i], &C[i]);
    return ORA_OK;
}

// O14 from the accumulated sums alone
int ora_reweight_mag_of(int L, const int64_t* Hsum, const double* lnD, const int64_t* A1, const int64_t* A2, int n,
                        const double* betas, double* absm, double* m2) {
    if (L < 4 || (L & 1) || !Hsum || !lnD || !A1 || !A2 || n < 0) return ORA_ERR_INVALID_ARG;
    bool any = false;
    for (int m = 0; m <= L * L; ++m) any = any || Hsum[m] > 0;
    if (!any) return ORA_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) reweight_mag_for(L * L, Hsum, lnD, A1, A2, betas[i], &absm[i], &m2[i]);
    return ORA_OK;
}
int ora_mag_fold_of(int L, int64_t R_cur, const int32_t* E, const int32_t* M, int64_t* A1, int64_t* A2) {
    if (L < 4 || (L & 1) || R_cur < 1 || !E || !M || !A1 || !A2) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> Ev(E, E + R_cur), Mv(M, M + R_cur);
    mag_fold_for(Ev, Mv, L * L, A1, A2);
    return ORA_OK;
}

// O13, Sec. 2.2 Eq. 6-7 (L99-L109): weighted average of M independent runs,
//   omega_m = exp(-beta F_m) / sum_m exp(-beta F_m) with -beta F_m = lnZ_m (Eq. 4), A~ = sum_m omega_m A_m,
// the largest lnZ_m taken out of the exponentials.  A is [M][nobs] row-major; omega_out may be NULL.
int ora_weighted_average(int M, const double* lnZ, const double* A, int nobs, double* A_out, double* omega_out) {
    if (M < 1 || nobs < 0 || !lnZ || (nobs > 0 && (!A || !A_out))) return ORA_ERR_INVALID_ARG;
    double zmax = lnZ[0];
    for (int m = 1; m < M; ++m) if (lnZ[m] > zmax) zmax = lnZ[m];
    std::vector<double> w(M);
    double S = 0.0;
    for (int m = 0; m < M; ++m) { w[m] = std::exp(lnZ[m] - zmax); S += w[m]; }
    for (int m = 0; m < M; ++m) { w[m] = w[m] / S; if (omega_out) omega_out[m] = w[m]; }
    for (int k = 0; k < nobs; ++k) {
        double acc = 0.0;
        for (int m = 0; m < M; ++m) acc += w[m] * A[(size_t)m * nobs + k];
        A_out[k] = acc;
    }
    return ORA_OK;
}

// ---- the population handle (the same calls as include/pa.h, prefixed ora_) -------------------

int ora_create(int L, int64_t R, uint64_t seed, Oracle** out) {
    if (!out || L < 4 || (L & 1) || R < 1) return ORA_ERR_INVALID_ARG;
    Oracle* o = new (std::nothrow) Oracle();
    if (!o) return ORA_ERR_NOMEM;
    o->L = L; o->N = L * L; o->R_target = R; o->R_cur = R; o->R_cap = capacity_for(R);
    o->D = 2; o->Lx = L; o->Ly = L; o->Lz = 1; o->nlev = o->N;
    o->seed = seed; o->t = 0; o->k = 0;
    o->lnZ = (double)o->N * std::log(2.0);                    // Z_{beta_0} = 2^N, L93
    try { o->spin.assign((size_t)o->R_cap * o->N, 0); } catch (...) { delete o; return ORA_ERR_NOMEM; }
    o->Hsum.assign(o->nlev + 1, 0);
    o->lnD.assign(o->nlev + 1, -std::numeric_limits<double>::infinity());
    o->A1sum.assign(o->nlev + 1, 0); o->A2sum.assign(o->nlev + 1, 0);
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < R; ++j)                           // step 1, L55, L65
        for (int s = 0; s < o->N; ++s) o->spin[(size_t)j * o->N + s] = x_init(seed, j, (uint32_t)s);
    *out = o;
    return ORA_OK;
}

// O16: the same population on a periodic simple-cubic box dims = (Lx, Ly, Lz), every edge even and >= 2; ndim must be 3
// (ndim = 2 with dims = (L, L) is ora_create).  ln Z starts at N ln 2 with N = Lx Ly Lz (L93).
int ora_create_box(int ndim, const int* dims, int64_t R, uint64_t seed, Oracle** out) {
    if (!out || !dims || R < 1) return ORA_ERR_INVALID_ARG;
    if (ndim == 2) { if (dims[0] != dims[1]) return ORA_ERR_INVALID_ARG; return ora_create(dims[0], R, seed, out); }
    if (ndim != 3) return ORA_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) if (dims[a] < 2 || (dims[a] & 1)) return ORA_ERR_INVALID_ARG;
    Oracle* o = new (std::nothrow) Oracle();
    if (!o) return ORA_ERR_NOMEM;
    o->D = 3; o->Lx = dims[0]; o->Ly = dims[1]; o->Lz = dims[2]; o->L = dims[0];
    o->N = o->Lx * o->Ly * o->Lz; o->nlev = 3 * o->N / 2;
    o->R_target = R; o->R_cur = R; o->R_cap = capacity_for(R);
    o->seed = seed; o->t = 0; o->k = 0;
    o->lnZ = (double)o->N * std::log(2.0);                    // Z_{beta_0} = 2^N, L93
    try { o->spin.assign((size_t)o->R_cap * o->N, 0); } catch (...) { delete o; return ORA_ERR_NOMEM; }
    o->Hsum.assign(o->nlev + 1, 0);
    o->lnD.assign(o->nlev + 1, -std::numeric_limits<double>::infinity());
    o->A1sum.assign(o->nlev + 1, 0); o->A2sum.assign(o->nlev + 1, 0);
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < R; ++j)                           // step 1, L55, L65: the INIT stream with the box's site index
        for (int s = 0; s < o->N; ++s) o->spin[(size_t)j * o->N + s] = x_init(seed, j, (uint32_t)s);
    *out = o;
    return ORA_OK;
}
int ora_num_levels(const Oracle* o) { return o ? o->nlev + 1 : 0; }

// stateless O16 pieces (pins, sampled parity checks)
void ora_thresholds3(double beta, uint32_t* T4, uint32_t* T8, uint32_t* T12) {
    *T4 = threshold(std::exp(-4.0 * beta));
    *T8 = threshold(std::exp(-8.0 * beta));
    *T12 = threshold(std::exp(-12.0 * beta));
}
int ora_sweep_slots_3d(const int* dims, uint64_t seed, uint32_t t0, double beta, int theta, int64_t nslots,
                       const int64_t* slot_ids, uint8_t* spins) {
    if (!dims || theta < 0 || nslots < 0) return ORA_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) if (dims[a] < 2 || (dims[a] & 1)) return ORA_ERR_INVALID_ARG;
    uint32_t T4, T8, T12; ora_thresholds3(beta, &T4, &T8, &T12);
    const int N = dims[0] * dims[1] * dims[2];
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nslots; ++i)
        for (int it = 0; it < theta; ++it)
            sweep_one_replica_3d(spins + (size_t)i * N, dims[0], dims[1], dims[2], seed, slot_ids[i], t0 + (uint32_t)it, T4, T8, T12);
    return ORA_OK;
}
int ora_energies_of_3d(const int* dims, int64_t n, const uint8_t* spins, int32_t* E, int32_t* M) {
    if (!dims || n < 0) return ORA_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) if (dims[a] < 2 || (dims[a] & 1)) return ORA_ERR_INVALID_ARG;
    const int N = dims[0] * dims[1] * dims[2];
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) {
        int32_t e, m; energy_one_replica_3d(spins + (size_t)j * N, dims[0], dims[1], dims[2], &e, &m);
        E[j] = e; if (M) M[j] = m;
    }
    return ORA_OK;
}

void ora_destroy(Oracle* o) { delete o; }

// O15: bimodal couplings, Jx[s] = bond (x,y)-(x+1,y), Jy[s] = bond (x,y)-(x,y+1), values +1 / -1, s = y*L + x.
// Both NULL: back to the ferromagnet.  Only before any histogram has been folded (the level offset e0 is part of the sums).
int ora_set_couplings(Oracle* o, const int8_t* Jx, const int8_t* Jy) {
    if (!o || ((Jx == nullptr) != (Jy == nullptr)) || (o->D == 3 && Jx)) return ORA_ERR_INVALID_ARG;   // O15 is a 2D workload
    for (int m = 0; m <= o->nlev; ++m) if (o->Hsum[m] != 0) return ORA_ERR_INVALID_ARG;
    if (!Jx) { o->Jx.clear(); o->Jy.clear(); o->e0 = 0; return ORA_OK; }
    int64_t n_af = 0;
    for (int s = 0; s < o->N; ++s) {
        if ((Jx[s] != 1 && Jx[s] != -1) || (Jy[s] != 1 && Jy[s] != -1)) return ORA_ERR_INVALID_ARG;
        n_af += (Jx[s] < 0) + (Jy[s] < 0);
    }
    o->Jx.assign(Jx, Jx + o->N); o->Jy.assign(Jy, Jy + o->N);
    // E = 2 (unsatisfied bonds) - 2N, and a spin flip changes the number of unsatisfied bonds by 4 - 2u (even), so its parity
    // is that of the all-up state, i.e. of the number of J = -1 bonds
    o->e0 = (int)((2 * n_af) % 4);
    return ORA_OK;
}
int ora_level_offset(const Oracle* o) { return o ? o->e0 : 0; }

// stateless O15 pieces for the pins
int ora_sweep_slots_j(int L, uint64_t seed, uint32_t t0, double beta, int theta, int64_t nslots, const int64_t* slot_ids,
                      uint8_t* spins, int rng_mode, const int8_t* Jx, const int8_t* Jy) {
    if (L < 4 || (L & 1) || theta < 0 || nslots < 0 || rng_mode < 0 || rng_mode > 1 || !Jx || !Jy) return ORA_ERR_INVALID_ARG;
    uint32_t T4, T8; ora_thresholds(beta, &T4, &T8);
    int N = L * L;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nslots; ++i)
        for (int it = 0; it < theta; ++it)
            sweep_one_replica(spins + (size_t)i * N, L, seed, slot_ids[i], t0 + (uint32_t)it, T4, T8, rng_mode, Jx, Jy);
    return ORA_OK;
}
int ora_energies_of_j(int L, int64_t n, const uint8_t* spins, const int8_t* Jx, const int8_t* Jy, int32_t* E, int32_t* M) {
    if (L < 4 || (L & 1) || n < 0 || !Jx || !Jy) return ORA_ERR_INVALID_ARG;
    int N = L * L;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) {
        int32_t e, m; energy_one_replica(spins + (size_t)j * N, L, &e, &m, Jx, Jy);
        E[j] = e; if (M) M[j] = m;
    }
    return ORA_OK;
}
// 0 = one Philox number per spin (O1), 1 = Philox-seeded LCG per word (O11, L236-L241)
int ora_set_rng_mode(Oracle* o, int mode) {
    if (!o || mode < 0 || mode > 1 || (o->D == 3 && mode != RNG_PHILOX)) return ORA_ERR_INVALID_ARG;   // O11 is keyed by 2D row quads
    o->rng_mode = mode;
    return ORA_OK;
}
int64_t ora_population(const Oracle* o) { return o->R_cur; }
int64_t ora_capacity_of(const Oracle* o) { return o->R_cap; }
uint32_t ora_sweep_counter(const Oracle* o) { return o->t; }
uint32_t ora_resample_counter(const Oracle* o) { return o->k; }
double ora_lnZ(const Oracle* o) { return o->lnZ; }

// step 3, L61: theta rounds of MCMC at inverse temperature beta.
int ora_sweep(Oracle* o, double beta, int theta) {
    if (!o || theta < 0) return ORA_ERR_INVALID_ARG;
    if (o->D == 3) {
        uint32_t T4, T8, T12; ora_thresholds3(beta, &T4, &T8, &T12);
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < o->R_cur; ++j)
            for (int it = 0; it < theta; ++it)
                sweep_one_replica_3d(&o->spin[(size_t)j * o->N], o->Lx, o->Ly, o->Lz, o->seed, j, o->t + (uint32_t)it, T4, T8, T12);
        o->t += (uint32_t)theta;
        return ORA_OK;
    }
    uint32_t T4, T8; ora_thresholds(beta, &T4, &T8);
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < o->R_cur; ++j)
        for (int it = 0; it < theta; ++it)
            sweep_one_replica(&o->spin[(size_t)j * o->N], o->L, o->seed, j, o->t + (uint32_t)it, T4, T8, o->rng_mode,
                              o->Jx.empty() ? nullptr : o->Jx.data(), o->Jy.empty() ? nullptr : o->Jy.data());
    o->t += (uint32_t)theta;
    return ORA_OK;
}

int ora_energies(Oracle* o, int32_t* E_out, int32_t* M_out) {
    if (!o || !E_out) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    std::memcpy(E_out, E.data(), sizeof(int32_t) * o->R_cur);
    if (M_out) std::memcpy(M_out, M.data(), sizeof(int32_t) * o->R_cur);
    return ORA_OK;
}

// step 2, L56-L58 and L65-L69: resample from beta to beta_new.
int ora_resample(Oracle* o, double beta, double beta_new, int64_t* R_new_out) {
    if (!o || !(beta_new >= beta)) return ORA_ERR_INVALID_ARG;
    double dbeta = beta_new - beta;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    std::vector<double> w(o->R_cur); std::vector<uint32_t> r(o->R_cur), off(o->R_cur);
    double W, lnQ; int64_t R_new;
    ora_resample_plan(o->R_target, o->R_cur, E.data(), o->seed, o->k, dbeta,
                      &W, w.data(), r.data(), off.data(), &R_new, &lnQ);
    if (R_new > o->R_cap) return ORA_ERR_CAPACITY;            // state unchanged (O7)
    if (R_new < 1) return ORA_ERR_CAPACITY;
    // new[o_j + c] = old[j], c = 0..r_j-1: slots keep parent order (O7, L165 "new population vector")
    std::vector<uint8_t> fresh((size_t)o->R_cap * o->N, 0);
    for (int64_t j = 0; j < o->R_cur; ++j)
        for (uint32_t c = 0; c < r[j]; ++c)
            std::memcpy(&fresh[((size_t)off[j] + c) * o->N], &o->spin[(size_t)j * o->N], o->N);
    o->spin.swap(fresh);
    o->R_cur = R_new; o->k += 1; o->lnZ += lnQ; o->lnQ_last = lnQ;   // Eq. 4
    o->W_last = W; o->w_last.swap(w); o->r_last.swap(r); o->o_last.swap(off);
    if (R_new_out) *R_new_out = R_new;
    return ORA_OK;
}

int ora_adapt_dbeta(Oracle* o, double target, double beta, double beta_max, double* dbeta_out) {
    if (!o || !dbeta_out || !(target > 0.0 && target < 1.0) || !(beta_max > beta)) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    *dbeta_out = adapt_for(E, o->R_target, target, beta_max - beta);
    return ORA_OK;
}

int ora_overlap(Oracle* o, double dbeta, double* alpha) {
    if (!o || !alpha) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    *alpha = overlap_for(E, o->R_target, dbeta);
    return ORA_OK;
}

// output fields of L179-L181
static void fill_obs(ora_obs_t* out, const obs_values& v, double beta, double lnQ, int64_t R) {
    out->beta = beta; out->e = v.e; out->C = v.C; out->absm = v.absm; out->m2 = v.m2; out->m4 = v.m4;
    out->betaF_per_N = v.betaF_per_N; out->S_per_N = v.S_per_N; out->lnQ = lnQ; out->R = R;
}

int ora_observables_of(int L, int64_t R_cur, const int32_t* E, const int32_t* M, double beta, double lnZ,
                       double lnQ, ora_obs_t* out) {
    if (L < 4 || (L & 1) || R_cur < 1 || !out) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> Ev(E, E + R_cur), Mv(M, M + R_cur);
    fill_obs(out, observables_for(Ev, Mv, (int64_t)L * L, beta, lnZ), beta, lnQ, R_cur);
    return ORA_OK;
}

int ora_observables(Oracle* o, double beta, ora_obs_t* out) {
    if (!o || !out) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    fill_obs(out, observables_for(E, M, o->N, beta, o->lnZ), beta, o->lnQ_last, o->R_cur);
    return ORA_OK;
}

int ora_hist_accumulate(Oracle* o, double beta) {
    if (!o) return ORA_ERR_INVALID_ARG;
    std::vector<int32_t> E, M; all_energies(o, E, M);
    hist_fold_for(E, o->nlev, o->lnZ, beta, o->Hsum.data(), o->lnD.data(), o->e0);
    mag_fold_for(E, M, o->nlev, o->A1sum.data(), o->A2sum.data(), o->e0);
    return ORA_OK;
}

int ora_get_mag_sums(const Oracle* o, int64_t* A1, int64_t* A2) {
    if (!o) return ORA_ERR_INVALID_ARG;
    if (A1) std::memcpy(A1, o->A1sum.data(), sizeof(int64_t) * (o->nlev + 1));
    if (A2) std::memcpy(A2, o->A2sum.data(), sizeof(int64_t) * (o->nlev + 1));
    return ORA_OK;
}
int ora_reweight_mag(const Oracle* o, int n, const double* betas, double* absm, double* m2) {
    if (!o || n < 0) return ORA_ERR_INVALID_ARG;
    bool any = false;
    for (int m = 0; m <= o->nlev; ++m) any = any || o->Hsum[m] > 0;
    if (!any) return ORA_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i)
        reweight_mag_for(o->nlev, o->Hsum.data(), o->lnD.data(), o->A1sum.data(), o->A2sum.data(), betas[i], &absm[i], &m2[i], o->e0, o->N);
    return ORA_OK;
}

int ora_get_histogram(const Oracle* o, int64_t* Hsum, double* lnD) {
    if (!o) return ORA_ERR_INVALID_ARG;
    if (Hsum) std::memcpy(Hsum, o->Hsum.data(), sizeof(int64_t) * (o->nlev + 1));
    if (lnD) std::memcpy(lnD, o->lnD.data(), sizeof(double) * (o->nlev + 1));
    return ORA_OK;
}

int ora_reweight(const Oracle* o, int n, const double* betas, double* lnZ, double* e, double* C) {
    if (!o || n < 0) return ORA_ERR_INVALID_ARG;
    bool any = false;
    for (int m = 0; m <= o->nlev; ++m) any = any || o->Hsum[m] > 0;
    if (!any) return ORA_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) reweight_for(o->nlev, o->Hsum.data(), o->lnD.data(), betas[i], &lnZ[i], &e[i], &C[i], o->e0, o->N);
    return ORA_OK;
}

// spins as +1/-1, [nrep][N], site = y*L + x
int ora_get_spins(const Oracle* o, int64_t j0, int64_t nrep, int8_t* out) {
    if (!o || j0 < 0 || nrep < 0 || j0 + nrep > o->R_cur) return ORA_ERR_INVALID_ARG;
    for (int64_t i = 0; i < nrep * o->N; ++i) out[i] = o->spin[(size_t)j0 * o->N + i] ? 1 : -1;
    return ORA_OK;
}
int ora_set_spins(Oracle* o, int64_t j0, int64_t nrep, const int8_t* in) {
    if (!o || j0 < 0 || nrep < 0 || j0 + nrep > o->R_cur) return ORA_ERR_INVALID_ARG;
    for (int64_t i = 0; i < nrep * o->N; ++i) o->spin[(size_t)j0 * o->N + i] = in[i] > 0 ? 1 : 0;
    return ORA_OK;
}

int ora_get_resample_debug(const Oracle* o, double* W, double* w, uint32_t* r, uint32_t* off) {
    if (!o) return ORA_ERR_INVALID_ARG;
    if (W) *W = o->W_last;
    if (w) std::memcpy(w, o->w_last.data(), sizeof(double) * o->w_last.size());
    if (r) std::memcpy(r, o->r_last.data(), sizeof(uint32_t) * o->r_last.size());
    if (off) std::memcpy(off, o->o_last.data(), sizeof(uint32_t) * o->o_last.size());
    return ORA_OK;
}

// thread count of the OpenMP loops over replicas (the results do not depend on it); n < 1 leaves it alone
void ora_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int ora_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}

}  // extern "C"
