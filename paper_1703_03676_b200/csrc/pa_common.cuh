// pa_common.cuh -- shared declarations of the CUDA library (handle, layout, Philox, error macros).
// Product code: shares nothing with oracle/.  Citations "L<n>" = /root/reference/PAPER.md line n,
// "O<n>" = reading n of DESIGN.md Sec. 3.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/pa.h"

// ------------------------------------------------------------------------------------------------
// Resident layout.  One "group" = 32 replica slots = one uint32 per site
// (asynchronous multi-spin coding with p = 32, L185); bit b of a word of group g = replica 32g+b.
// Inside a group the N = L*L words are split by checkerboard colour c = (x+y)&1 (the paper stores
// the two sub-lattices separately too, L157):   index(c, y, xh) = c*(N/2) + y*(L/2) + xh,
// xh = x >> 1.   Site (x,y) of colour c in row y has x = 2*xh + ((y+c)&1).
// ------------------------------------------------------------------------------------------------
// A simple-cubic box Lx x Ly x Lz (O16) uses the same scheme with the "row" r = z*Ly + y:
//   index(c, r, xh) = c*(N/2) + r*(Lx/2) + xh,  x = 2*xh + ((y+z+c)&1),  site s = r*Lx + x;
// Lz = 1 is the square lattice.
struct PaGeom { int Lx, Ly, Lz; };
#ifdef __CUDACC__
// site index s = (z*Ly + y)*Lx + x of the word at resident index idx
__host__ __device__ __forceinline__ int pa_site_of_index(int idx, PaGeom g) {
    const int Lh = g.Lx >> 1, half = (g.Lx * g.Ly * g.Lz) >> 1;
    const int c = idx >= half ? 1 : 0;
    const int rem = idx - c * half;
    const int r = rem / Lh, xh = rem - r * Lh;
    const int z = r / g.Ly, y = r - z * g.Ly;
    return r * g.Lx + 2 * xh + ((y + z + c) & 1);
}
__host__ __device__ __forceinline__ int pa_index_of_site(int s, PaGeom g) {
    const int r = s / g.Lx, x = s - r * g.Lx;
    const int z = r / g.Ly, y = r - z * g.Ly;
    const int c = (x + y + z) & 1;
    return c * ((g.Lx * g.Ly * g.Lz) >> 1) + r * (g.Lx >> 1) + (x >> 1);
}
#endif

#define PA_TAG_INIT 0u
#define PA_TAG_SWEEP 1u
#define PA_TAG_RESAMPLE 2u
#define PA_TAG_LCG 3u

#define PA_LCG_A 1664525u      // L236, ref. [43]
#define PA_LCG_C 1013904223u

#define PA_PHILOX_M0 0xD2511F53u
#define PA_PHILOX_M1 0xCD9E8D57u
#define PA_PHILOX_W0 0x9E3779B9u
#define PA_PHILOX_W1 0xBB67AE85u

#define PA_TILE 1024  // elements per reduction / scan tile (TREE1024, O5)

struct PhiloxKeys {  // the 10 round keys of Philox4x32-10 for one 64-bit seed (uniform per launch)
    uint32_t k0[10], k1[10];
};

static inline PhiloxKeys pa_make_keys(uint64_t seed) {
    PhiloxKeys k;
    uint32_t a = (uint32_t)(seed & 0xffffffffull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { k.k0[r] = a; k.k1[r] = b; a += PA_PHILOX_W0; b += PA_PHILOX_W1; }
    return k;
}

#ifdef __CUDACC__
__device__ __forceinline__ void pa_mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
    unsigned long long p = (unsigned long long)a * (unsigned long long)b;   // IMAD.WIDE.U32
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
}
// Plain Philox4x32-10 (ref. [33], L368; L163), used where the call is not the bottleneck.
__device__ __forceinline__ uint4 pa_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& K) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0, lo0, hi1, lo1;
        pa_mulhilo(PA_PHILOX_M0, c0, hi0, lo0);
        pa_mulhilo(PA_PHILOX_M1, c2, hi1, lo1);
        uint32_t n0 = hi1 ^ c1 ^ K.k0[r], n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}
#endif

// device-resident scalars (one block, also mirrored in pinned host memory for small D2H reads)
struct PaScalars {
    // --- written by pa_measure_kernel; zeroed (cudaMemsetAsync up to R_new) before it runs
    uint32_t mmin_inv, mmax;     // 2^32-1 - min_j m_j and max_j m_j, m = (E + 2N)/4
    uint32_t done_counter;       // ticket of the measure kernel's last-CTA stage
    uint32_t pad0;
    long long SE, SE2, SA, SM2;  // exact integer sums (O8)
    double m4sum;                // TREE1024 of (M_j/N)^4
    // --- written by the resample kernels
    uint32_t R_new;              // sum of the copy numbers (pa_plan_kernel)
    uint32_t tile_counter;       // scan tile tickets (reset by pa_tree_kernel<0>)
    uint32_t tree_ticket;        // ticket of pa_tree_kernel's last-CTA stage (self-resetting)
    uint32_t pad1;
    double W;                    // normaliser of the last weight table, TREE1024 order (pa_tree_kernel<0>)
    double sum;                  // TREE1024 of min(1, tau_j) (pa_tree_kernel<1>)
    // --- device-resident loop (pa_anneal): the population size lives on the device between host reads
    uint32_t R_dev;              // current population size (copy kernel, pa_anneal)
    uint32_t err;                // 1 = a resampling step left [1, R_cap]
};

// Kernels take the population size and E_min either from the host (the step-by-step calls) or, inside pa_anneal, from
// the device scalars: R < 0 / Emin == PA_EMIN_DEV select the device copy.
#define PA_EMIN_DEV (-2147483647 - 1)
#ifdef __CUDACC__
// Once a resampling step of pa_anneal has left [1, R_cap] (sc->err) the population counts as empty for every later kernel of the
// call: they all exit without touching the spins or E, M, so the population stays the one before the failing step (O7).
__device__ __forceinline__ long long pa_live_R(long long R, const PaScalars* sc) { return R >= 0 ? R : (sc->err ? 0ll : (long long)sc->R_dev); }
// nlev = (number of bonds)/2: energies lie on -2 nlev + 4m + e0, m = 0..nlev (nlev = N on the square lattice, 3N/2 on the cubic one)
__device__ __forceinline__ int pa_live_Emin(int Emin, const PaScalars* sc, int nlev, int e0) {
    return Emin != PA_EMIN_DEV ? Emin : -2 * nlev + 4 * (int)(0xffffffffu - sc->mmin_inv) + e0;
}
#endif

// State of the bisection of pa_adapt_dbeta between launches of pa_adapt_kernel (pa_adapt.cu)
#define PA_ADAPT_BINS 8192          // energy levels the kernel's shared-memory table holds (wider populations: exact path)
enum { PA_ADAPT_DONE = 0, PA_ADAPT_AMBIG = 1, PA_ADAPT_AMBIG_FIRST = 2, PA_ADAPT_RETURN_HI = 3 };
struct PaAdaptState {
    double lo, hi;   // bracket
    int it;          // next bisection iteration (0..40); -1: the test alpha(hi) >= alpha* comes first
    int status;      // PA_ADAPT_*: done / iteration `it` (or the first test) is too close to alpha* for the histogram sum
    double margin;   // diagnostics: min over the decisions the kernel took itself of |alpha' - alpha*| / bound (> 1 by construction)
    double a_last;   // diagnostics: alpha' of the iteration handed back (status AMBIG*), to be set against the exact alpha
};

// Environment switches (tests and tuning, every value gives the same bytes).  The environment is read ONCE, in
// pa_create*, into the handle (pa_switches_read, the only getenv of the library); pa_set_switch changes one on a live handle.
enum {
    PA_SW_PDL, PA_SW_SNAP_HOST, PA_SW_ADAPT_EXACT, PA_SW_ANNEAL_CHUNK, PA_SW_FUSE_COPY, PA_SW_STEP_HOST_CHUNK, PA_SW_MEASURE_GENERIC,
    PA_SW_SMALL_PLAN, PA_SW_SWEEP_C, PA_SW_SWEEP_T, PA_SW_SWEEP_SMEM_KB, PA_SW_SWEEP_KIND, PA_SW_SWEEP_CMP, PA_SW_SWEEP_MIXED,
    PA_SW_LCG_P64, PA_SW_LCG_NOR, PA_SW_SWEEP_SPLIT, PA_SW_COUNT
};
struct PaSwitches { bool set[PA_SW_COUNT]; long long val[PA_SW_COUNT]; };
void pa_switches_read(PaSwitches* sw);                 // pa_api.cu
int pa_switch_index(const char* name);                 // "PA_SWEEP_C" -> PA_SW_SWEEP_C, -1 if unknown

struct pa_handle {
    int device;              // the CUDA device the handle was created on; every entry point makes it current for the call (PaDeviceGuard)
    PaSwitches sw;
    int L, N;                // N = number of sites; L = Lx
    int D; PaGeom geom;      // dimension (2 / 3, O16) and edges; D = 2: geom = {L, L, 1}
    int nlev;                // energy levels m = 0..nlev, E_m = -2 nlev + 4m + e0: N (2D), 3N/2 (3D)
    int64_t R_target, R_cur, R_cap;
    int64_t G_cap;           // groups at capacity
    uint64_t seed;
    uint32_t t, k;
    int rng_mode;            // PA_RNG_PHILOX / PA_RNG_LCG (O11)
    bool has_j;              // O15: bimodal couplings set
    int e0;                  // O15: every energy is -2N + 4m + e0, e0 = 2 (number of J = -1 bonds) mod 4
    uint16_t* jm16;          // [N/8] O15 bond masks in the order of the quad-column measure kernel (16 bond words per row and quad)
    uint8_t* jmask;          // [N] resident order: bits 0-3 = bond to (same-cell, x, up, down) neighbour has J = -1; bit 4 = right bond
    double lnZ, lnQ_last;
    PhiloxKeys keys;

    cudaStream_t stream;
    bool owns_stream, owns_ws;
    void* ws; size_t ws_bytes;

    uint32_t* spins[2]; int cur;        // two packed populations [G_cap][N] (L165 "new population vector")
    int32_t *E, *M; bool em_valid;      // per-replica energy / magnetisation of the current population (+ sums in d_scal)
    bool host_scal_valid;               // h_scal mirrors d_scal's measure block for the current population
    int Emin, Emax;                     // range of E_j of the current population (valid with host_scal_valid)
    double* runsum;                     // [G_cap] run-of-32 sums of the measure kernel
    double* w;                          // weights of the last resample (debug export)
    uint32_t *r, *o, *parent;           // copy numbers, exclusive offsets, parent map
    double* partials;                   // per-tile partial sums (TREE1024)
    double* wtab;                       // weight table, device, N+1 entries
    const double* wtab_cur;             // pa_anneal: this step's full-range table (NULL = wtab)
    unsigned long long* scan_state;     // decoupled look-back tile states
    unsigned long long* Hsum;           // [N+1]
    uint32_t* Hcur;                     // [N+1] histogram of the current temperature
    uint32_t* Hd;                       // [N+1] count-only histogram of the current population for pa_adapt_dbeta
    PaAdaptState *d_adapt, *h_adapt;    // bisection state, device / pinned host (mapped: the kernel writes it there)
    PaAdaptState* h_adapt_dev;          // device address of h_adapt
    int adapt_exact_evals, adapt_filter_launches;   // of the last pa_adapt_dbeta (diagnostics)
    double adapt_min_margin;            // of the last pa_adapt_dbeta: smallest |alpha' - alpha*| / bound at a decision of the filter
    double adapt_max_err;               // over the handle's life: largest |alpha' - alpha_exact| / first-order bound seen at a hand-back
    double* lnD;                        // [N+1]
    unsigned long long *A1, *A2;        // [N+1] sums of |M_j| and M_j^2 per energy level over all folded replicas (O14)
    int64_t* d_slots;                   // slot list for pa_get_spins_at
    int8_t* stage;                      // staging for unpacked spin export/import
    size_t stage_bytes;
    PaScalars* d_scal;
    int64_t n_tiles_cap;

    PaScalars* h_scal;                  // pinned
    PaScalars *h_snap, *h_snap_dev;     // pinned and mapped: the measure kernel's last CTA leaves the scalars there itself (single calls)
    bool snap_on_host;                  // ... and has done so for the current population
    PaScalars* mail_out;                // pa_resample: where the plan kernel leaves R_new and W for the host (mapped memory), or NULL
    double* h_wtab;                     // pinned, N+1
    int64_t R_prev; double W_last;      // of the last resample

    cudaEvent_t ev[9];                  // sweep begin/end, resample begin/end, copy begin/end, plan scalars on the host, measure begin/end
    bool sweep_timed, resample_timed, measure_timed;
    int timing;                         // PA_TIME_* mask: which phases record CUDA timing events (pa_set_timing)
    bool hist_any;                      // pa_hist_accumulate has run at least once
    bool scal_zeroed;                   // the copy kernel has cleared the measure accumulators (pa_anneal): no memset needed
    PaScalars* snap_out;                // pa_anneal: where the measure kernel leaves a copy of the device scalars (or NULL)
    bool dev_R;                         // inside pa_anneal: kernels read R and E_min from d_scal, grids cover the capacity
    cudaEvent_t ev_chunk[2];            // pa_anneal: completion of the chunk staged in buffer 0 / 1
    cudaStream_t xfer_stream; cudaEvent_t ev_xfer;   // pa_step_host: device-to-host copies of finished chunks run beside the sweeps
    double* h_tabs; size_t h_tabs_bytes; // pinned staging for pa_anneal's weight tables and snapshots
    int pdl;                            // 1: the step's kernels are launched with programmatic stream serialization
    int n_sm;                           // streaming multiprocessors of the device (148 on B200): launch plans count rounds of them
    int64_t launches;
    bool sweep_C_forced;
    uint32_t T12;            // third threshold of the cubic lattice (dE = 12), set by pa_sweep
    int last_sweep_kind;     // PA_SWEEP_RAN_* bits of the last sweep launch (pa_last_sweep_kind)
    int sweep_C, sweep_T, sweep_cmp, sweep_kind;   // sweep launch geometry (cluster size, threads), compare variant, kernel kind
    char cuda_err[256];
};

// value of a switch on this handle, `dflt` if it was not set
static inline long long pa_sw(const pa_handle* h, int key, long long dflt) { return h->sw.set[key] ? h->sw.val[key] : dflt; }

// Makes the handle's device current for the duration of a call and restores the caller's afterwards (handles on several GPUs in
// one process: pa_weighted_average over runs "or over GPUs").  cudaGetDevice is a thread-local read.
struct PaDeviceGuard {
    int prev; bool switched;
    explicit PaDeviceGuard(const pa_handle* h) : prev(-1), switched(false) {
        if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->device) switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~PaDeviceGuard() { if (switched) cudaSetDevice(prev); }
    PaDeviceGuard(const PaDeviceGuard&) = delete;
    PaDeviceGuard& operator=(const PaDeviceGuard&) = delete;
};

#define PA_CUDA(h, call)                                                                      \
    do {                                                                                      \
        cudaError_t e__ = (call);                                                             \
        if (e__ != cudaSuccess) { pa_note_cuda_error((h), e__, #call, __FILE__, __LINE__); return PA_ERR_CUDA; } \
    } while (0)

void pa_note_cuda_error(pa_handle* h, cudaError_t e, const char* what, const char* file, int line);

// ------------------------------------------------------------------------------------------------
// Programmatic dependent launch (sm_90+): the kernels of a temperature step form a chain tree -> plan -> copy -> sweep -> measure
// in which every kernel needs its predecessor's output.  Launched with cudaLaunchAttributeProgrammaticStreamSerialization, a kernel
// may be scheduled while its predecessor is still draining; it must then execute pa_pdl_wait() (griddepcontrol.wait: returns when
// the predecessor grid has completed and its memory is visible) before it touches anything, and it lets ITS successor be scheduled
// early with pa_pdl_launch().  On the launch-bound small populations this hides the launch latency between the five kernels.
// Without the attribute both instructions do nothing.  h->pdl = 0 (environment PA_PDL=0) launches everything the classic way.
// ------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pa_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pa_pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static inline cudaError_t pa_launch(const pa_handle* h, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = h->pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}
#endif

// kernels' host launchers (each returns PA_OK / PA_ERR_CUDA and counts its launches in h->launches)
int pa_launch_init(pa_handle* h);
int pa_launch_sweep(pa_handle* h, uint32_t T4, uint32_t T8, int theta);
int pa_sweep_configure(pa_handle* h);
int pa_launch_sweep_range(pa_handle* h, uint32_t T4, uint32_t T8, int theta, int64_t g0, int64_t ng);   // groups g0 .. g0+ng-1 (column-walk kernels)
int pa_launch_words_out_range(pa_handle* h, uint32_t* d_words, int64_t g0, int64_t ng);              // interchange words of those groups -> d_words[g0*N ...]
int pa_launch_measure(pa_handle* h);                                   // E, M, integer sums, m range, m^4 sum
int pa_launch_weights(pa_handle* h, int Emin, double* w_out);          // w_j, W = TREE1024(w) -> d_scal->W
int pa_launch_overlap(pa_handle* h, int Emin);                         // TREE1024(min(1, tau_j)) -> d_scal->sum
int pa_launch_plan(pa_handle* h, int Emin);                            // tau, r, scan, parent map, R_new
int pa_launch_weights_plan(pa_handle* h, int Emin, double* w_out, bool commit);   // both; one fused launch for populations of a few tiles
bool pa_small_plan_ok(const pa_handle* h);                             // ... which this says
bool pa_sweep_gathers(const pa_handle* h, int theta);                  // pa_anneal: the next sweep launch can do the replica copy while staging
int pa_launch_sweep_gather(pa_handle* h, uint32_t T4, uint32_t T8, int theta);   // sweep of spins[cur] := resampled spins[1-cur]
int pa_launch_copy(pa_handle* h);                                      // new[d] = old[parent(d)], d < R_new (read on the device); pa_anneal: + commit
int pa_launch_hist(pa_handle* h, double beta);
int pa_launch_ehist(pa_handle* h);                                     // count-only energy histogram -> Hd
int pa_run_adapt_filter(pa_handle* h, double target, double bound);   // bisection on the histogram from *h_adapt; synchronises
int pa_launch_reweight(pa_handle* h, int n, double* d_io);              // O12, O14: d_io = [betas | lnZ | e | C | absm | m2], n each
cudaError_t pa_run_wavg(int M, const double* d_lnZ, const double* d_A, int nobs, double* d_out, double* d_omega, cudaStream_t st);
int pa_launch_unpack(pa_handle* h, const int64_t* d_slots, int64_t j0, int64_t n, int8_t* d_out);
int pa_launch_pack(pa_handle* h, int64_t j0, int64_t n, const int8_t* d_in);
int pa_launch_words_out(pa_handle* h, uint32_t* d_words);
int pa_launch_words_in(pa_handle* h, int64_t R, const uint32_t* d_words);
int pa_run_calibrate(int kind, double* ginstr_per_ns, double* sm_mhz);
