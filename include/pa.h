/* pa.h -- C ABI of the B200 population-annealing (PA) hot path for the 2D Ising model.
 *
 * The calls follow the paper's statement of the algorithm (Sec. 2.1, steps
 * 1-5) and BASELINE.json's north_star: pa_create = step 1, pa_resample = step 2,
 * pa_sweep = step 3, pa_observables = step 4; the caller owns the loop and the beta schedule
 * (equal steps, L71, or pa_adapt_dbeta, Sec. 2.3).  "L<n>" below cites a line of
 * /root/reference/PAPER.md; "O<n>" cites the reading of that passage listed in DESIGN.md Sec. 3.
 *
 * One handle = one population of replicas of the L x L periodic ferromagnetic Ising model
 * (Eq. 10), resident in device memory, bit-packed 32 replicas per 32-bit word
 * (asynchronous multi-spin coding, L185).  All work is enqueued on the handle's CUDA stream.
 * Calls that return a host scalar synchronise that stream; the others are asynchronous.
 * A handle is not thread-safe; different handles are independent.  There is no global state.
 *
 * Pointers: every `out`/`in` buffer below may be a HOST pointer or a DEVICE pointer (of the
 * handle's device); the library asks the CUDA runtime which it is.  Buffers are caller-owned;
 * the library never keeps them after the call returns.
 *
 * Every function returning int returns PA_OK (0) or a negative PA_ERR_* code; on error the
 * population is unchanged unless stated otherwise.  There is no CPU fallback: without a CUDA
 * device pa_create / pa_create_ex return PA_ERR_CUDA.
 */
#ifndef PA_B200_PA_H
#define PA_B200_PA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pa_handle pa_t; /* opaque */

enum {
    PA_OK = 0,
    PA_ERR_INVALID_ARG = -1, /* L odd or < 4 or > 512, R < 1, theta < 0, beta' < beta, alpha* not in (0,1), NULL */
    PA_ERR_CAPACITY = -2,    /* resampling would exceed the capacity R_cap (or produce an empty population) */
    PA_ERR_CUDA = -3,        /* a CUDA call failed (sticky: see pa_last_cuda_error) */
    PA_ERR_WORKSPACE = -4,   /* caller-provided workspace too small or not 256-byte aligned */
    PA_ERR_NOMEM = -5,
    PA_ERR_STATIC_LIMIT = -6 /* pa_weighted_average_static: more runs than its fixed scratch array holds */
};

/* One output line of the paper's program (L179-L181): beta, energy per site, specific heat,
 * |m|, m^2, m^4 (Eq. 3), beta F / N (Eq. 4), S / N (Eq. 5), population size,
 * ln Q of the last resampling step (Eq. 1). */
typedef struct {
    double beta, e, C, absm, m2, m4, betaF_per_N, S_per_N, lnQ;
    int64_t R;
} pa_obs_t;

/* Capacity in replicas of a population with target size R (O7; the paper is silent):
 * R_cap = 32 * ceil((R + max(1024, ceil(8 sqrt R))) / 32).  sigma(R_i) <= sqrt(R)/2 by Eq. 2. */
int64_t pa_capacity(int64_t R);

/* Bytes of device workspace pa_create_ex needs for (L, R): two packed spin buffers of R_cap
 * replicas (the population and the "new population vector" of L165) plus per-replica vectors,
 * tables and scalars. */
int pa_workspace_bytes(int L, int64_t R, size_t* bytes);

/* Step 1 (L55, L65): R independent replicas with i.i.d. uniform +-1 spins (equilibrium at
 * beta_0 = 0), drawn from the INIT stream of the Philox4x32-10 generator keyed by `seed` (O1).
 * Sets ln Z = N ln 2 (L93), sweep counter t = 0, resample counter k = 0, empty histograms.
 * L even, 4 <= L <= 512, and such that L/C rows of one 32-replica group (L*L*4/C bytes) fit the shared memory of a CTA for a
 * cluster size C in {1,2,4,8} dividing L: every even L <= 338, the multiples of 4 up to 476, the multiples of 8 up to 512
 * (other L: PA_ERR_INVALID_ARG, also from pa_workspace_bytes); 1 <= R <= 2^31.
 * The handle belongs to the CUDA device that is current when it is created: its kernels, its stream and its memory live there.
 * Every later call on the handle makes that device current for the duration of the call and restores the caller's device before it
 * returns, so handles on several GPUs can be driven from one thread without cudaSetDevice between the calls; host / device
 * buffers passed to a call must be reachable from the handle's device.
 * pa_create allocates with cudaMalloc on the current device and uses its own stream.
 * pa_create_ex borrows `dev_ws` (device memory, >= pa_workspace_bytes, 256-byte aligned; e.g.
 * a torch tensor's data_ptr()) and enqueues on `cuda_stream` (a cudaStream_t; NULL = the
 * legacy default stream).  The handle must be destroyed before the workspace is freed. */
int pa_create(int L, int64_t R, uint64_t seed, pa_t** out);
int pa_create_ex(int L, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out);
void pa_destroy(pa_t* h);

/* The same population on another lattice (L313 "models on different lattices in various dimensions ... straightforward", L43
 * "3D Ising systems"; reading O16): ndim = 3, dims = {Lx, Ly, Lz} (HOST int[3]): a periodic simple-cubic box, every edge even and
 * >= 2, at most 2^18 sites, Lz/C planes of a group (4 Lx Ly Lz / C bytes) fitting a CTA's shared memory for a C in {1,2,4,8}
 * dividing Lz.  Site s = (z*Ly + y)*Lx + x in every per-site array of this header (spins, words).  A spin has six neighbour
 * slots x+-1, y+-1, z+-1 (an edge of length 2 holds the same site in both slots of its direction; it counts twice); with u
 * anti-parallel slots dE = 12 - 4u and pa_sweep flips iff u >= 3, or u = 2 and x < T4, or u = 1 and x < T8, or u = 0 and
 * x < T12 = floor(exp(-12 beta) 2^32); colour 0 = (x+y+z) even first; the random numbers are the SWEEP stream's with this s.
 * E_j = -sum_s s_s (s_{x+1} + s_{y+1} + s_{z+1}) lies on -3N + 4m, m = 0 .. 3N/2: the histogram arrays of pa_get_histogram /
 * pa_get_mag_sums have pa_num_levels(h) = 3N/2 + 1 entries (N + 1 on the square lattice).  Every other call is unchanged;
 * PA_RNG_LCG and pa_set_couplings are readings of the square lattice and return PA_ERR_INVALID_ARG on a box.
 * ndim = 2 with dims = {L, L} is pa_create_ex.  dev_ws = NULL: cudaMalloc and a private stream, as pa_create. */
int pa_workspace_bytes_box(int ndim, const int* dims, int64_t R, size_t* bytes);
int pa_create_box(int ndim, const int* dims, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out);
int pa_dims(const pa_t* h, int* ndim, int* dims);      /* dims: int[3] (dims[2] = 1 on the square lattice); either may be NULL */
int64_t pa_num_levels(const pa_t* h);                  /* number of energy levels = length of the histogram arrays */

/* Step 3 (L61; L151-L157): theta checkerboard Metropolis sweeps of every replica at inverse
 * temperature beta.  One sweep = colour 0 ((x+y) even), then colour 1.  A spin with u
 * anti-parallel neighbours (dE = 8 - 4u) flips iff u >= 2, or u = 1 and x < T4, or u = 0 and
 * x < T8, with x = the SWEEP-stream uint32 of (slot j, site s, sweep t, colour c) (O1, O3) and
 * T4, T8 = floor(exp(-4 beta) 2^32), floor(exp(-8 beta) 2^32) clamped to 2^32-1, computed on
 * the host (O2; L163).  Advances t by theta.  Asynchronous. */
int pa_sweep(pa_t* h, double beta, int theta);

/* Source of the SWEEP-stream numbers x (the resampling always uses Philox directly, L241):
 *   PA_RNG_PHILOX (default; O1): one Philox4x32-10 output word per spin, x(j,s,t,c) =
 *     philox(s, j>>2, 2t+c, TAG_SWEEP)[j&3]  (Table 1's n_RNG = p rows, L193-L196);
 *   PA_RNG_LCG (O11; Sec. 4, Table 1's last section): the paper's fast variant.  The word
 *     of group g at site s = (x,y) is seeded at every visit (sweep t, colour c) with
 *     r_0 = philox((y>>2)*(L/2) + (x>>1), g, 2t+c, TAG_LCG)[y&3] and its 32 replicas take the next 32
 *     outputs of r_{n+1} = 1664525 r_n + 1013904223 mod 2^32 (L236), most significant lane first:
 *     x(32g+b) = r_{32-b}.
 * Both are functions of (slot, site, sweep) only, so trajectories do not depend on the launch
 * geometry.  Takes effect from the next pa_sweep.  mode outside {0,1}: PA_ERR_INVALID_ARG. */
enum { PA_RNG_PHILOX = 0, PA_RNG_LCG = 1 };
int pa_set_rng_mode(pa_t* h, int mode);
int pa_get_rng_mode(const pa_t* h);

/* A second workload (L313: "the case of different couplings including spin glasses"; O15): bimodal couplings J = +-1 on
 * the bonds, shared by all replicas of the population, H = -sum_<ab> J_ab s_a s_b.  Jx[s] couples site s = y*L+x to
 * (x+1, y), Jy[s] couples it to (x, y+1) (periodic); int8[N] each, values +1 / -1, host or device.  Both NULL: back to
 * the ferromagnet of Eq. 10 (the default).  The acceptance rule is unchanged with u = the number of UNSATISFIED bonds of
 * the spin (dE = 8 - 4u); energies lie on -2N + 4m + e0 with e0 = pa_level_offset = 2 (number of J = -1 bonds) mod 4,
 * which the histogram (Eq. 9) and reweighting calls use for E_m.  Must be called before the first pa_hist_accumulate
 * (PA_ERR_INVALID_ARG afterwards, or if a value is not +-1).  Sweeps and energies run on the same kernels as the
 * ferromagnet, instantiated with one bond-mask byte per word.  Synchronous. */
int pa_set_couplings(pa_t* h, const int8_t* Jx, const int8_t* Jy);
int pa_level_offset(const pa_t* h);

/* Configurational energies E_j = -sum_<ab> s_a s_b and magnetisations M_j = sum_a s_a of the
 * current replicas j = 0..R_cur-1 (Eq. 10; L173).  E_out, M_out: int32[>= R_cur], host or
 * device; M_out may be NULL.  Synchronises if an output is a host pointer. */
int pa_energies(pa_t* h, int32_t* E_out, int32_t* M_out);

/* Step 2 (L56-L58, L65-L69): resample from beta to beta_new >= beta.
 *   w_j = exp(-(beta_new - beta)(E_j - E_min))          (Eq. 1 with the common factor taken out, O5)
 *   W = sum_j w_j in the fixed TREE1024 order (O5; L165: deterministic),  ln Q = -dbeta E_min + ln(W / R_cur)
 *   tau_j = R w_j / W,  r_j = floor(tau_j) + [u_j < frac(tau_j)],  u_j = RESAMPLE-stream uniform (Eq. 2, O6)
 *   o_j = sum_{i<j} r_i,  R_new = sum_j r_j,  new[o_j + c] = old[j] for c < r_j   (L165, O7)
 * Then R_cur = R_new, k += 1, ln Z += ln Q (Eq. 4).  R_new is also written to *R_new (may be NULL).
 * PA_ERR_CAPACITY if R_new > R_cap or R_new = 0: population, k and ln Z unchanged.  Synchronises. */
int pa_resample(pa_t* h, double beta, double beta_new, int64_t* R_new);

/* Sec. 2.3 (L113-L118), Eq. 8: the overlap alpha(dbeta) = (1/R_cur) sum_j min(1, tau_j(dbeta)),
 * summed in the TREE1024 order.  0 < target_overlap < 1, beta_max > beta.
 * Returns in *dbeta: beta_max - beta if alpha(beta_max - beta) >= target; otherwise the lower end
 * of the bracket after exactly 40 bisection steps starting from [0, beta_max - beta] (O10), so
 * that alpha(*dbeta) >= target.  Does not change the population.  Synchronises. */
int pa_adapt_dbeta(pa_t* h, double target_overlap, double beta, double beta_max, double* dbeta);
/* How the last pa_adapt_dbeta reached its 41 decisions (diagnostics): most are taken inside one kernel on the energy histogram,
 * whose sum differs from the TREE1024 sum by a bounded rounding error; a decision closer to the target than four times that
 * bound is taken by an exact evaluation (weight table, two fixed-order reductions, one host round trip) -- *exact_evaluations
 * of them, typically 2-4 instead of 41; *filter_launches = launches of the histogram kernel.  The result is the one O10
 * defines either way.  Environment PA_ADAPT_EXACT=1 forces all 41 exact evaluations.  Either pointer may be NULL. */
int pa_adapt_stats(const pa_t* h, int* exact_evaluations, int* filter_launches);
/* A tripwire for that rounding bound (first-order, with a factor 4 on top).  *min_margin: over the decisions
 * the kernel took itself in the last pa_adapt_dbeta, the smallest |alpha' - alpha*| in units of the decision threshold (> 1 by
 * construction; +inf if it took none).  *max_error: over the whole life of the handle, the largest |alpha' - alpha| seen at an
 * iteration that was handed to the exact evaluation, in units of the first-order bound (2 R_cur + 2 dmax + 32) 2^-53; the decision
 * threshold is 4 of these units, so the results are safe while this stays below 4 (0 if no iteration was handed back yet). */
int pa_adapt_margins(const pa_t* h, double* min_margin, double* max_error);
/* alpha(dbeta) of Eq. 8 for one dbeta >= 0 (the function pa_adapt_dbeta bisects on). */
int pa_overlap(pa_t* h, double dbeta, double* alpha);

/* Step 4 (L62): population averages of the current population at `beta` (Eq. 3-5; field list
 * L179-L181).  Integer sums are exact; the m^4 sum uses the TREE1024 order (O8).  No side
 * effects.  Synchronises. */
int pa_observables(pa_t* h, double beta, pa_obs_t* out);

/* Sec. 2.4, Eq. 9 (L124-L129): fold the energy histogram of the current population at `beta`
 * into the running sums  Hsum[m] += #{j : E_j = -2N + 4m}  and
 * lnD[m] = logaddexp(lnD[m], ln R_cur - ln Z - beta (-2N + 4m))   (O9).
 * Call once per temperature, after the sweeps.  Asynchronous. */
int pa_hist_accumulate(pa_t* h, double beta);
/* Hsum: int64[pa_num_levels], lnD: double[pa_num_levels] (N + 1 on the square lattice; either may be NULL);
 * ln Omega(E_m) = ln Hsum[m] - lnD[m]. */
int pa_get_histogram(pa_t* h, int64_t* Hsum, double* lnD);

/* n temperature steps in one call (steps 2-4 of L56-L62, n times): for i = 1..n, resample betas[i-1] -> betas[i], theta
 * sweeps at betas[i], measure; obs_out[i-1] = the output line of betas[i] (L179-L181).  betas: double[n+1], HOST, non-decreasing,
 * betas[0] = the current temperature; obs_out: pa_obs_t[n], HOST, or NULL.  Computes exactly what the same sequence of
 * pa_resample / pa_sweep / pa_observables calls computes (same spins, copy numbers, ln Z, observables), but the population
 * size and E_min stay on the device and nothing inside a chunk of steps waits for the host: the launch-bound small
 * configurations run at the speed of their kernels.  The Eq. 9 histogram is not folded (call pa_hist_accumulate between
 * calls for that).  Errors: PA_ERR_INVALID_ARG as for the single calls; PA_ERR_CAPACITY if a step left [1, R_cap]: as after a
 * failed pa_resample the population is then the one BEFORE that step (the kernels of the later steps see the device-side error
 * flag and do nothing), the steps before it have been applied (pa_resample_counter tells how many; their obs_out entries are
 * valid), and the handle stays usable.  Synchronises. */
int pa_anneal(pa_t* h, int n, const double* betas, int theta, pa_obs_t* obs_out);

/* Multi-histogram reweighting (Sec. 2.4; O12, O14): from the sums accumulated so far, the density of
 * states ln Omega(E_m) = ln Hsum[m] - lnD[m] (Eq. 9) and, for each of the n inverse temperatures betas[i]
 * (any values, not only simulated ones), lnZ[i] = ln sum_m Omega_m exp(-beta E_m) (= -beta F, Eq. 4),
 * e[i] = <E>/N and C[i] = beta^2 (<E^2> - <E>^2)/N (Eq. 3), and -- the generalisation to magnetisations of L129 --
 * absm[i] = <|m|>, m2[i] = <m^2> from the microcanonical sums that pa_hist_accumulate keeps per energy level
 * (A1[m] = sum |M_j|, A2[m] = sum M_j^2 over all folded replicas with E_j = E_m): <|m|> = sum_m p_m A1[m]/Hsum[m] / N.
 * betas and the outputs: double[n], host or device (all of the same kind); outputs may be NULL.  1 <= n <= 2^20.
 * PA_ERR_INVALID_ARG if no histogram has been accumulated.  Does not change the population.  Synchronises if the
 * buffers are host pointers. */
int pa_reweight(pa_t* h, int n, const double* betas, double* lnZ, double* e, double* C, double* absm, double* m2);

/* The microcanonical magnetisation sums (O14): A1, A2: int64[pa_num_levels], host or device, either may be NULL. */
int pa_get_mag_sums(pa_t* h, int64_t* A1, int64_t* A2);

/* Weighted average of M independent runs (Sec. 2.2, Eq. 6-7; O13): omega_m = exp(lnZ_m) /
 * sum_m exp(lnZ_m) with lnZ_m = -beta F_m(beta) = pa_lnZ of run m at this temperature, A_out[k] =
 * sum_m omega_m A[m*nobs + k].  HOST pointers; lnZ: double[M], A: double[M*nobs], A_out: double[nobs],
 * omega_out: double[M] or NULL.  Runs on the current CUDA device (no handle needed); synchronous. */
int pa_weighted_average(int M, const double* lnZ, const double* A, int nobs, double* A_out, double* omega_out);

/* The same weighted average (Eq. 6-7; O13) for callers that must not allocate device memory.
 * pa_weighted_average above stages its host arguments through a cudaMalloc / cudaFree pair.  Three kinds of caller cannot
 * live with that: one that has already given all of the GPU's memory away (populations sized to fill the HBM, or a host
 * framework whose pool owns the rest), where an allocation late in a run may fail; one that combines its runs at every
 * temperature while other populations are sweeping on other streams, because cudaMalloc and cudaFree make the whole device
 * wait; and one running where a blocking driver call is not allowed (a stream callback, a latency-bounded loop).
 * This entry point calls no cudaMalloc, no cudaFree and nothing else that allocates.  The caller passes DEVICE pointers (of the
 * current device) for everything: d_lnZ: double[M], d_A: double[M*nobs] (run-major, A[m*nobs + k]), d_A_out: double[nobs];
 * d_A and d_A_out may be NULL if nobs = 0.  The weights omega_m, which the kernel has to write and read back, live in a
 * fixed array inside the library: PA_WAVG_STATIC_MAX_RUNS doubles = 32 KiB of device memory that every GPU which loads the
 * library keeps until the process ends.  M > PA_WAVG_STATIC_MAX_RUNS: PA_ERR_STATIC_LIMIT, nothing launched (use
 * pa_weighted_average).  A pointer the CUDA runtime does not know as device (or managed) memory: PA_ERR_INVALID_ARG.
 * The kernel is enqueued on `cuda_stream` (a cudaStream_t; NULL = the legacy default stream) and the call returns without
 * waiting: d_A_out is valid once that stream has reached this point.  The result equals pa_weighted_average's.
 * Sharing: all calls on one GPU use the same array and find in it whatever the previous call left.  No entry has to start at
 * zero -- each call writes omega_0..omega_{M-1} before reading them -- so nothing is cleared; but two calls that can run on the
 * GPU at the same time (two streams) race on the array and both results are undefined: order them on one stream or with an event.
 * Set-up: the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device current;
 * this may load the library's device code) and remembers it; make that first call during start-up, before any stream capture
 * is begun on that device.  Thread-safe as far as the set-up goes; the sharing rule above still applies.
 * pa_weighted_average_static_max_runs() returns PA_WAVG_STATIC_MAX_RUNS for callers that load the library dynamically. */
#define PA_WAVG_STATIC_MAX_RUNS 4096
int pa_weighted_average_static(int M, const double* d_lnZ, const double* d_A, int nobs, double* d_A_out, void* cuda_stream);
int pa_weighted_average_static_max_runs(void);

/* State export / import (parity tests, checkpoints, the end-to-end benchmark).
 * Spins are +1 / -1, one int8 per spin, out[i][s] with site s = y*L + x.
 * pa_get_spins: replicas j0 .. j0+nrep-1.  pa_get_spins_at: replicas slots[0..n-1] (host int64).
 * pa_set_spins overwrites replicas j0 .. j0+nrep-1 (j0 + nrep <= R_cur).
 * pa_get_words / pa_set_words move the packed population, uint32 words[ceil(R_cur/32)][N] with
 * word (g, s) holding replica 32g+b at site s = y*L + x in bit b (the interchange layout; the
 * resident layout is colour-split); bits of slots >= R_cur in the last group read as 0.  pa_set_words also sets R_cur = R
 * (1 <= R <= R_cap) and leaves t, k, ln Z untouched. */
int pa_get_spins(pa_t* h, int64_t j0, int64_t nrep, int8_t* out);
int pa_get_spins_at(pa_t* h, const int64_t* slots, int64_t n, int8_t* out);
int pa_set_spins(pa_t* h, int64_t j0, int64_t nrep, const int8_t* in);
int pa_get_words(pa_t* h, uint32_t* words);
int pa_set_words(pa_t* h, int64_t R, const uint32_t* words);

/* One temperature step of the paper's loop (steps 2-4) for a population that lives in HOST memory between
 * steps: the same results, bit for bit, as pa_set_words(R_in, words_in); pa_resample(beta, beta_new); pa_sweep(beta_new, theta);
 * pa_observables(beta_new); pa_energies; pa_get_words(words_out) -- but the sweeps run in chunks of groups and every finished
 * chunk travels to the host on a second stream while the following chunks are swept.
 * words_in: HOST uint32 [ceil(R_in/32)][N] (interchange layout, above); words_out: HOST uint32 [ceil(R_cap/32)][N], of which the
 * first ceil(R_new/32) groups are written (pinned memory for the overlap; pageable memory works, serially).  E_out / M_out: host or
 * device int32[R_new] or NULL; obs_out, R_new_out: host or NULL.  words_out may be the same buffer as words_in (the upload has
 * completed before the first chunk is copied back).  Synchronous: on every return path, errors included, no copy into words_out is
 * still in flight.  Errors as the single calls; after
 * PA_ERR_CAPACITY the handle holds the uploaded population unchanged and words_out is untouched. */
int pa_step_host(pa_t* h, int64_t R_in, const uint32_t* words_in, double beta, double beta_new, int theta,
                 uint32_t* words_out, int32_t* E_out, int32_t* M_out, pa_obs_t* obs_out, int64_t* R_new_out);

/* Vectors of the last resampling step (pa_resample, or the last step of pa_anneal), indexed by the parent slot
 * j < R_prev = pa_prev_population(h), the population size before that step; any pointer may be NULL.  A step that fails with
 * PA_ERR_CAPACITY has already overwritten them: from then until the next successful step (and before the first one)
 * pa_prev_population is 0 and this call returns PA_ERR_INVALID_ARG.
 * W (one double), w[R_prev] double, r[R_prev] uint32 copy numbers, o[R_prev] uint32 offsets. */
int pa_get_resample_debug(pa_t* h, double* W, double* w, uint32_t* r, uint32_t* o);
int64_t pa_prev_population(const pa_t* h);

/* Scalars of the handle. */
int64_t pa_population(const pa_t* h);       /* R_cur */
int64_t pa_capacity_of(const pa_t* h);      /* R_cap */
uint32_t pa_sweep_counter(const pa_t* h);   /* t */
uint32_t pa_resample_counter(const pa_t* h);/* k */
double pa_lnZ(const pa_t* h);               /* = -beta F(beta), Eq. 4 */
/* Overwrite the counters (restart from a checkpoint; sampled parity checks at the large configs). */
int pa_set_counters(pa_t* h, uint32_t t, uint32_t k, double lnZ);

/* Tests and tuning: the library's switches (PA_SWEEP_C, PA_SWEEP_T, PA_SWEEP_KIND, PA_LCG_P64, PA_ADAPT_EXACT,
 * PA_STEP_HOST_CHUNK, ...; every value gives the same bytes) are environment variables that are read ONCE, when a handle is
 * created; no later call reads the environment.  pa_set_switch changes one on a live handle: `name` = the variable's name,
 * is_set = 0 returns it to "not set" (the default behaviour), otherwise it takes `value`.  The sweep launch geometry is re-planned.
 * PA_ERR_INVALID_ARG for an unknown name or a value that leaves no valid geometry (the switch then keeps its old state). */
int pa_set_switch(pa_t* h, const char* name, int is_set, int64_t value);
/* Which sweep kernel the last pa_sweep launched (diagnostics; the results do not depend on it): bit 0 = column-walk kernel,
 * bit 1 = lane-split CTAs present, bit 2 = the p = 64 (uint2) variant of the LCG-assisted kernel, bit 3 = mixed launch.  0 before
 * the first sweep. */
enum { PA_SWEEP_RAN_COL = 1, PA_SWEEP_RAN_SPLIT = 2, PA_SWEEP_RAN_P64 = 4, PA_SWEEP_RAN_MIXED = 8 };
int pa_last_sweep_kind(const pa_t* h);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
int64_t pa_launch_count(const pa_t* h);
/* Device time in milliseconds of the last pa_sweep / the last pa_resample on this handle,
 * measured with CUDA events on the handle's stream; the kernel that dominates each is the
 * sweep kernel / the replica-copy kernel (time of that kernel alone in *kernel_ms).
 * pa_last_measure_ms: the last launch of the energy / magnetisation / observable-sums kernel (row a3 + a8),
 * which runs inside the first of pa_energies / pa_observables / pa_resample / pa_adapt_dbeta /
 * pa_hist_accumulate that follows a change of the population.
 * Synchronises.  Either pointer may be NULL.  PA_ERR_INVALID_ARG if no such operation has run yet with its
 * phase timed.  Timing events are not free on a stream of small kernels (about 3 us each; measured: 8 events per step
 * cost 4 % of a cfg2 step and 36 % of a cfg1 step), so only the sweep is timed by default:
 * pa_set_timing(h, PA_TIME_SWEEP | PA_TIME_RESAMPLE | PA_TIME_MEASURE) turns the others on, 0 turns all off. */
enum { PA_TIME_SWEEP = 1, PA_TIME_RESAMPLE = 2, PA_TIME_MEASURE = 4 };
int pa_set_timing(pa_t* h, int mask);
int pa_last_sweep_ms(pa_t* h, float* kernel_ms);
int pa_last_resample_ms(pa_t* h, float* total_ms, float* copy_kernel_ms);
int pa_last_measure_ms(pa_t* h, float* kernel_ms);

/* Integer-pipe calibration for the roofline denominator: runs a dependent
 * chain of `kind` = 0: LOP3, 1: IMAD.WIDE.U32, 2: the Philox round's mix (2 IMAD.WIDE + 2 LOP3),
 * on every SM and returns the achieved thread-instructions per nanosecond of the whole GPU in
 * *ginstr_per_ns and the SM clock it ran at in *sm_mhz (from the cycle counter).  Uses the
 * current device and the default stream; synchronises. */
int pa_calibrate(int kind, double* ginstr_per_ns, double* sm_mhz);

/* Text for a PA_ERR_* code (static storage); the message of the last failed CUDA call on this handle (owned by the
 * handle, valid until the next call on it; "" if none); the library's version string (static storage). */
const char* pa_strerror(int code);
const char* pa_last_cuda_error(const pa_t* h);
const char* pa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PA_B200_PA_H */
