// pa_api.cu -- the C ABI of include/pa.h: handle, workspace layout, host-side step logic
// (threshold and weight tables, bisection, observables from exact integer sums).
// All arithmetic that decides an integer (thresholds, weight table) is computed here on the host in
// fp64 with libm and handed to the kernels as data (O2, O5); the device never calls exp for a decision.
#include "pa_common.cuh"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>

#define PA_ALIGN 256
#define PA_STAGE_BYTES ((size_t)32 << 20)
#define PA_SLOTS_CAP 65536

static size_t pa_align_up(size_t v) { return (v + PA_ALIGN - 1) / PA_ALIGN * PA_ALIGN; }

void pa_note_cuda_error(pa_handle* h, cudaError_t e, const char* what, const char* file, int line) {
    if (h) snprintf(h->cuda_err, sizeof(h->cuda_err), "%s: %s (%s:%d)", cudaGetErrorString(e), what, file, line);
}

struct PaLayout {
    size_t spins0, spins1, E, M, w, r, o, parent, partials, runsum, wtab, scan, Hsum, Hcur, Hd, adapt, lnD, A1, A2, jmask, jm16, scal, slots, stage, total;
    size_t stage_bytes;
    int64_t R_cap, G_cap, tiles;
};

// N = number of sites, nlev + 1 = number of energy levels (tables, histograms)
static PaLayout pa_layout_n(size_t N, size_t nlev, int64_t R) {
    PaLayout y;
    y.R_cap = pa_capacity(R);
    y.G_cap = y.R_cap / 32;
    y.tiles = (y.R_cap + PA_TILE - 1) / PA_TILE;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t at = off; off = pa_align_up(off + bytes); return at; };
    y.spins0 = take((size_t)y.G_cap * N * 4);
    y.spins1 = take((size_t)y.G_cap * N * 4);
    y.E = take((size_t)y.R_cap * 4);
    y.M = take((size_t)y.R_cap * 4);
    y.w = take((size_t)y.R_cap * 8);
    y.r = take((size_t)y.R_cap * 4);
    y.o = take((size_t)y.R_cap * 4);
    y.parent = take((size_t)y.R_cap * 4);
    y.partials = take((size_t)y.tiles * 8);
    y.runsum = take((size_t)y.G_cap * 8);
    y.wtab = take((nlev + 1) * 8);
    y.scan = take((size_t)y.tiles * 8);
    y.Hsum = take((nlev + 1) * 8);
    y.Hcur = take((nlev + 1) * 4);
    y.Hd = take((nlev + 1) * 4);
    y.adapt = take(sizeof(PaAdaptState));
    y.lnD = take((nlev + 1) * 8);
    y.A1 = take((nlev + 1) * 8);
    y.A2 = take((nlev + 1) * 8);
    y.jmask = take(N);
    y.jm16 = take(N / 8 * 2 + 2);
    y.scal = take(sizeof(PaScalars));
    y.slots = take((size_t)PA_SLOTS_CAP * 8);
    y.stage_bytes = (size_t)y.R_cap * N < PA_STAGE_BYTES ? pa_align_up((size_t)y.R_cap * N) : PA_STAGE_BYTES;
    if (y.stage_bytes < (size_t)N * 4 * 4) y.stage_bytes = pa_align_up((size_t)N * 4 * 4);
    y.stage = take(y.stage_bytes);
    y.total = off;
    return y;
}
static PaLayout pa_layout(int L, int64_t R) { return pa_layout_n((size_t)L * L, (size_t)L * L, R); }

// O16: a periodic simple-cubic box, every edge even and >= 2, at most 2^18 sites, and Lz/C whole planes of one group
// (N*4/C bytes) must fit the shared memory of a CTA for a cluster size C in {1,2,4,8} dividing Lz.
static bool pa_box_ok(const int* d, int64_t R) {
    if (!d || R < 1 || R > (int64_t)1 << 31) return false;
    for (int a = 0; a < 3; ++a) if (d[a] < 2 || (d[a] & 1) || d[a] > 512) return false;
    const long long N = (long long)d[0] * d[1] * d[2];
    if (N > (1 << 18)) return false;
    for (int C = 1; C <= 8; C *= 2)
        if (d[2] % C == 0 && (size_t)N * 4 / C <= (size_t)224 * 1024) return true;
    return false;
}

// L even, 4 <= L <= 512, and the sweep kernel's strip of L/C rows of a group (L*L*4/C bytes) must fit the shared memory of a CTA
// for some cluster size C in {1,2,4,8} dividing L: every even L <= 338, and above that the multiples of 4 up to 476 and the
// multiples of 8 (pa_sweep_configure picks C).
static bool pa_args_ok(int L, int64_t R) {
    if (!(L >= 4 && L <= 512 && (L & 1) == 0 && R >= 1 && R <= (int64_t)1 << 31)) return false;
    for (int C = 1; C <= 8; C *= 2)
        if (L % C == 0 && (size_t)L * L * 4 / C <= (size_t)224 * 1024) return true;
    return false;
}

// O2: T(p) = (uint32) min(floor(p * 2^32), 2^32 - 1)
static uint32_t pa_threshold(double p) {
    double v = floor(p * 4294967296.0);
    if (v > 4294967295.0) v = 4294967295.0;
    if (v < 0.0) v = 0.0;
    return (uint32_t)v;
}

static bool pa_is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

static int pa_copy_out(pa_handle* h, void* dst, const void* dev_src, size_t bytes, bool* synced) {
    if (bytes == 0) return PA_OK;
    if (pa_is_device_ptr(dst)) {
        PA_CUDA(h, cudaMemcpyAsync(dst, dev_src, bytes, cudaMemcpyDeviceToDevice, h->stream));
    } else {
        PA_CUDA(h, cudaMemcpyAsync(dst, dev_src, bytes, cudaMemcpyDeviceToHost, h->stream));
        PA_CUDA(h, cudaStreamSynchronize(h->stream));
        if (synced) *synced = true;
    }
    return PA_OK;
}

static int pa_read_scalars(pa_handle* h) {
    PA_CUDA(h, cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(PaScalars), cudaMemcpyDeviceToHost, h->stream));
    PA_CUDA(h, cudaStreamSynchronize(h->stream));
    return PA_OK;
}
// The scalars of the measure kernel: its last CTA has written them into mapped host memory itself (no copy operation between
// the kernel and the host's wake-up: a few microseconds per call on the launch-bound populations); else the copy above.
static int pa_read_measure_scalars(pa_handle* h) {
    if (!h->snap_on_host) return pa_read_scalars(h);
    PA_CUDA(h, cudaStreamSynchronize(h->stream));
    *h->h_scal = *h->h_snap;
    return PA_OK;
}

static int pa_ensure_energies(pa_handle* h) { return h->em_valid ? PA_OK : pa_launch_measure(h); }

// E, M, the integer sums and the range of m = (E + 2N)/4 of the current population, mirrored on the host:
// one measure launch (if the population changed) and one small device-to-host read (if not read yet).
static int pa_ensure_host_scalars(pa_handle* h) {
    int rc = pa_ensure_energies(h);
    if (rc != PA_OK) return rc;
    if (h->host_scal_valid) return PA_OK;
    if ((rc = pa_read_measure_scalars(h)) != PA_OK) return rc;
    h->host_scal_valid = true;
    h->Emin = -2 * h->nlev + 4 * (int)(0xffffffffu - h->h_scal->mmin_inv) + h->e0;
    h->Emax = -2 * h->nlev + 4 * (int)h->h_scal->mmax + h->e0;
    return PA_OK;
}

// O5: wtab[d] = exp(-(dbeta * (double)(4 d))), d = 0..dmax, uploaded to the device table
static int pa_upload_wtab(pa_handle* h, double dbeta, int dmax) {
    for (int d = 0; d <= dmax; ++d) h->h_wtab[d] = exp(-(dbeta * (double)(4 * d)));
    PA_CUDA(h, cudaMemcpyAsync(h->wtab, h->h_wtab, sizeof(double) * (size_t)(dmax + 1), cudaMemcpyHostToDevice, h->stream));
    return PA_OK;
}

extern "C" {

int64_t pa_capacity(int64_t R) {
    int64_t slack = (int64_t)ceil(8.0 * sqrt((double)R));
    if (slack < 1024) slack = 1024;
    return 32 * ((R + slack + 31) / 32);
}

int pa_workspace_bytes(int L, int64_t R, size_t* bytes) {
    if (!bytes || !pa_args_ok(L, R)) return PA_ERR_INVALID_ARG;
    *bytes = pa_layout(L, R).total;
    return PA_OK;
}

int pa_workspace_bytes_box(int ndim, const int* dims, int64_t R, size_t* bytes) {
    if (!bytes || !dims) return PA_ERR_INVALID_ARG;
    if (ndim == 2) return dims[0] == dims[1] ? pa_workspace_bytes(dims[0], R, bytes) : PA_ERR_INVALID_ARG;
    if (ndim != 3 || !pa_box_ok(dims, R)) return PA_ERR_INVALID_ARG;
    const size_t N = (size_t)dims[0] * dims[1] * dims[2];
    *bytes = pa_layout_n(N, 3 * N / 2, R).total;
    return PA_OK;
}

static int pa_create_impl(int D, PaGeom geom, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out);

int pa_create_ex(int L, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out) {
    if (!out || !pa_args_ok(L, R)) return PA_ERR_INVALID_ARG;
    const PaGeom g = {L, L, 1};
    return pa_create_impl(2, g, R, seed, dev_ws, ws_bytes, cuda_stream, out);
}

int pa_create_box(int ndim, const int* dims, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out) {
    if (!out || !dims) return PA_ERR_INVALID_ARG;
    if (ndim == 2) return dims[0] == dims[1] ? pa_create_ex(dims[0], R, seed, dev_ws, ws_bytes, cuda_stream, out) : PA_ERR_INVALID_ARG;
    if (ndim != 3 || !pa_box_ok(dims, R)) return PA_ERR_INVALID_ARG;
    const PaGeom g = {dims[0], dims[1], dims[2]};
    return pa_create_impl(3, g, R, seed, dev_ws, ws_bytes, cuda_stream, out);
}

int pa_dims(const pa_t* h, int* ndim, int* dims) {
    if (!h) return PA_ERR_INVALID_ARG;
    if (ndim) *ndim = h->D;
    if (dims) { dims[0] = h->geom.Lx; dims[1] = h->geom.Ly; dims[2] = h->D == 3 ? h->geom.Lz : 1; }
    return PA_OK;
}
int64_t pa_num_levels(const pa_t* h) { return h ? (int64_t)h->nlev + 1 : 0; }

static int pa_create_impl(int D, PaGeom geom, int64_t R, uint64_t seed, void* dev_ws, size_t ws_bytes, void* cuda_stream, pa_t** out) {
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return PA_ERR_CUDA; }
    const int L = geom.Lx;
    const size_t Nsites = (size_t)geom.Lx * geom.Ly * geom.Lz, nlev_ = D == 3 ? 3 * Nsites / 2 : Nsites;
    const PaLayout y = pa_layout_n(Nsites, nlev_, R);
    pa_handle* h = new (std::nothrow) pa_handle();
    if (!h) return PA_ERR_NOMEM;
    memset(h, 0, sizeof(*h));
    h->L = L; h->N = (int)Nsites; h->D = D; h->geom = geom; h->nlev = (int)nlev_;
    h->R_target = R; h->R_cur = R; h->R_cap = y.R_cap; h->G_cap = y.G_cap;
    h->seed = seed; h->keys = pa_make_keys(seed); h->rng_mode = PA_RNG_PHILOX; h->timing = PA_TIME_SWEEP;
    pa_switches_read(&h->sw);                                         // the environment is read here and nowhere else
    h->pdl = pa_sw(h, PA_SW_PDL, 1) == 0 ? 0 : 1;
    { int dev = 0, nsm = 0;                                           // launch plans count rounds of the SMs (148 on B200)
      if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); delete h; return PA_ERR_CUDA; }
      h->device = dev;                                                // the handle lives on the device current at creation
      h->n_sm = (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0) ? nsm : 148; }
    h->lnZ = (double)h->N * log(2.0);           // Z_{beta_0} = 2^N (L93)
    h->n_tiles_cap = y.tiles;
    int rc = PA_OK;
    if (dev_ws) {
        if (ws_bytes < y.total || ((uintptr_t)dev_ws % PA_ALIGN) != 0) { delete h; return PA_ERR_WORKSPACE; }
        h->ws = dev_ws; h->owns_ws = false; h->stream = (cudaStream_t)cuda_stream; h->owns_stream = false;
    } else {
        cudaError_t e = cudaMalloc(&h->ws, y.total);
        if (e != cudaSuccess) { cudaGetLastError(); delete h; return e == cudaErrorMemoryAllocation ? PA_ERR_NOMEM : PA_ERR_CUDA; }
        h->owns_ws = true;
        if (cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(h->ws); delete h; return PA_ERR_CUDA; }
        h->owns_stream = true;
    }
    h->ws_bytes = y.total;
    char* b = (char*)h->ws;
    h->spins[0] = (uint32_t*)(b + y.spins0); h->spins[1] = (uint32_t*)(b + y.spins1); h->cur = 0;
    h->E = (int32_t*)(b + y.E); h->M = (int32_t*)(b + y.M);
    h->w = (double*)(b + y.w); h->r = (uint32_t*)(b + y.r); h->o = (uint32_t*)(b + y.o); h->parent = (uint32_t*)(b + y.parent);
    h->partials = (double*)(b + y.partials); h->runsum = (double*)(b + y.runsum); h->wtab = (double*)(b + y.wtab);
    h->scan_state = (unsigned long long*)(b + y.scan);
    h->Hsum = (unsigned long long*)(b + y.Hsum); h->Hcur = (uint32_t*)(b + y.Hcur); h->lnD = (double*)(b + y.lnD);
    h->Hd = (uint32_t*)(b + y.Hd); h->d_adapt = (PaAdaptState*)(b + y.adapt);
    h->A1 = (unsigned long long*)(b + y.A1); h->A2 = (unsigned long long*)(b + y.A2);
    h->jmask = (uint8_t*)(b + y.jmask); h->jm16 = (uint16_t*)(b + y.jm16); h->has_j = false; h->e0 = 0;
    h->d_scal = (PaScalars*)(b + y.scal);
    h->d_slots = (int64_t*)(b + y.slots);
    h->stage = (int8_t*)(b + y.stage); h->stage_bytes = y.stage_bytes;
    // pinned host mirrors
    if (cudaHostAlloc(&h->h_snap, sizeof(PaScalars), cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer(&h->h_snap_dev, h->h_snap, 0) != cudaSuccess ||
        cudaMallocHost(&h->h_scal, sizeof(PaScalars)) != cudaSuccess ||
        cudaMallocHost(&h->h_wtab, sizeof(double) * ((size_t)h->nlev + 1)) != cudaSuccess ||
        cudaHostAlloc(&h->h_adapt, sizeof(PaAdaptState), cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer(&h->h_adapt_dev, h->h_adapt, 0) != cudaSuccess) { rc = PA_ERR_CUDA; }
    for (int i = 0; i < 9 && rc == PA_OK; ++i)
        if (cudaEventCreateWithFlags(&h->ev[i], i == 6 ? cudaEventDisableTiming : cudaEventDefault) != cudaSuccess) rc = PA_ERR_CUDA;
    if (rc == PA_OK) rc = pa_sweep_configure(h);
    if (rc == PA_OK) {
        // empty histograms: Hsum = 0, Hcur = 0, lnD = -inf
        cudaMemsetAsync(h->d_scal, 0, sizeof(PaScalars), h->stream);
        cudaMemsetAsync(h->Hsum, 0, ((size_t)h->nlev + 1) * 8, h->stream);
        cudaMemsetAsync(h->Hcur, 0, ((size_t)h->nlev + 1) * 4, h->stream);
        cudaMemsetAsync(h->A1, 0, ((size_t)h->nlev + 1) * 8, h->stream);
        cudaMemsetAsync(h->A2, 0, ((size_t)h->nlev + 1) * 8, h->stream);
        for (int m = 0; m <= h->nlev; ++m) h->h_wtab[m] = -INFINITY;
        if (cudaMemcpyAsync(h->lnD, h->h_wtab, ((size_t)h->nlev + 1) * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess) rc = PA_ERR_CUDA;
        if (rc == PA_OK) rc = pa_launch_init(h);
        if (rc == PA_OK && cudaStreamSynchronize(h->stream) != cudaSuccess) rc = PA_ERR_CUDA;
    }
    if (rc != PA_OK) { pa_destroy(h); return rc; }
    *out = h;
    return PA_OK;
}

int pa_create(int L, int64_t R, uint64_t seed, pa_t** out) { return pa_create_ex(L, R, seed, nullptr, 0, nullptr, out); }

void pa_destroy(pa_t* h) {
    PaDeviceGuard dg__(h);
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    for (int i = 0; i < 9; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->h_snap) cudaFreeHost(h->h_snap);
    if (h->h_wtab) cudaFreeHost(h->h_wtab);
    if (h->h_adapt) cudaFreeHost(h->h_adapt);
    if (h->h_tabs) cudaFreeHost(h->h_tabs);
    for (int b = 0; b < 2; ++b) if (h->ev_chunk[b]) cudaEventDestroy(h->ev_chunk[b]);
    if (h->ev_xfer) cudaEventDestroy(h->ev_xfer);
    if (h->xfer_stream) cudaStreamDestroy(h->xfer_stream);
    if (h->owns_stream && h->stream) cudaStreamDestroy(h->stream);
    if (h->owns_ws && h->ws) cudaFree(h->ws);
    delete h;
}

int pa_sweep(pa_t* h, double beta, int theta) {
    PaDeviceGuard dg__(h);
    if (!h || theta < 0 || !(beta == beta)) return PA_ERR_INVALID_ARG;
    if (theta == 0) return PA_OK;
    const uint32_t T4 = pa_threshold(exp(-4.0 * beta)), T8 = pa_threshold(exp(-8.0 * beta));
    h->T12 = pa_threshold(exp(-12.0 * beta));                                    // O16: dE = 12 exists on the cubic lattice only
    const bool timed = (h->timing & PA_TIME_SWEEP) != 0;
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[0], h->stream));
    int rc = pa_launch_sweep(h, T4, T8, theta);
    if (rc != PA_OK) return rc;
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[1], h->stream));
    h->sweep_timed = timed;
    h->t += (uint32_t)theta;
    h->em_valid = false; h->host_scal_valid = false;
    return PA_OK;
}

int pa_set_rng_mode(pa_t* h, int mode) {
    PaDeviceGuard dg__(h);
    if (!h || (mode != PA_RNG_PHILOX && mode != PA_RNG_LCG)) return PA_ERR_INVALID_ARG;
    if (h->D == 3 && mode != PA_RNG_PHILOX) return PA_ERR_INVALID_ARG;        // O11 is keyed by quads of rows of the square lattice
    h->rng_mode = mode;
    return PA_OK;
}
int pa_get_rng_mode(const pa_t* h) { return h ? h->rng_mode : PA_ERR_INVALID_ARG; }

// O15 (L313): bimodal couplings shared by all replicas.  Builds the per-word bond mask in the resident (colour-split) order.
int pa_set_couplings(pa_t* h, const int8_t* Jx, const int8_t* Jy) {
    PaDeviceGuard dg__(h);
    if (!h || ((Jx == nullptr) != (Jy == nullptr)) || h->hist_any || (h->D == 3 && Jx)) return PA_ERR_INVALID_ARG;   // O15 is a 2D workload
    h->em_valid = false; h->host_scal_valid = false;
    if (!Jx) { h->has_j = false; h->e0 = 0; return PA_OK; }
    const int L = h->L, N = h->N, Lh = L / 2;
    int8_t* hx = (int8_t*)malloc((size_t)N * 2);
    uint8_t* jm = (uint8_t*)malloc((size_t)N);
    if (!hx || !jm) { free(hx); free(jm); return PA_ERR_NOMEM; }
    int8_t* hy = hx + N;
    cudaError_t err = cudaMemcpy(hx, Jx, (size_t)N, cudaMemcpyDefault);
    if (err == cudaSuccess) err = cudaMemcpy(hy, Jy, (size_t)N, cudaMemcpyDefault);
    if (err != cudaSuccess) { free(hx); free(jm); pa_note_cuda_error(h, err, "cudaMemcpy(couplings)", __FILE__, __LINE__); return PA_ERR_CUDA; }
    long long n_af = 0;
    for (int s = 0; s < N; ++s) {
        if ((hx[s] != 1 && hx[s] != -1) || (hy[s] != 1 && hy[s] != -1)) { free(hx); free(jm); return PA_ERR_INVALID_ARG; }
        n_af += (hx[s] < 0) + (hy[s] < 0);
    }
    for (int c = 0; c < 2; ++c)
        for (int y = 0; y < L; ++y)
            for (int xh = 0; xh < Lh; ++xh) {
                const int p = (y + c) & 1, x = 2 * xh + p;
                const int xl = x == 0 ? L - 1 : x - 1, yu = y == 0 ? L - 1 : y - 1;
                const bool right = hx[y * L + x] < 0, left = hx[y * L + xl] < 0, down = hy[y * L + x] < 0, up = hy[yu * L + x] < 0;
                // neighbour "same cell" of the other colour is x+1 for p = 0 and x-1 for p = 1; the "x" neighbour is the other one
                const bool same = p ? left : right, other = p ? right : left;
                jm[c * (N / 2) + y * Lh + xh] = (uint8_t)((same ? 1 : 0) | (other ? 2 : 0) | (up ? 4 : 0) | (down ? 8 : 0) | (right ? 16 : 0));
            }
    err = cudaMemcpyAsync(h->jmask, jm, (size_t)N, cudaMemcpyHostToDevice, h->stream);
    // the same bonds in the order of the quad-column measure kernel (L a multiple of 8): per row y and quad q of four cells
    // xh = 4q+k: bit k = bond inside cell (x = 2xh), 4+k = bond to the next cell (x = 2xh+1), 8+k / 12+k = down bonds of the
    // colour-0 / colour-1 site of the cell (x = 2xh + (y&1) / 2xh + ((y+1)&1))
    uint16_t* j16 = nullptr;
    if (err == cudaSuccess && L % 8 == 0) {
        const int QPR = L / 8;
        j16 = (uint16_t*)malloc((size_t)L * QPR * 2);
        if (!j16) { free(hx); free(jm); return PA_ERR_NOMEM; }
        for (int y = 0; y < L; ++y)
            for (int q = 0; q < QPR; ++q) {
                unsigned m = 0;
                for (int k = 0; k < 4; ++k) {
                    const int xh = 4 * q + k;
                    if (hx[y * L + 2 * xh] < 0) m |= 1u << k;
                    if (hx[y * L + 2 * xh + 1] < 0) m |= 1u << (4 + k);
                    if (hy[y * L + 2 * xh + (y & 1)] < 0) m |= 1u << (8 + k);
                    if (hy[y * L + 2 * xh + ((y + 1) & 1)] < 0) m |= 1u << (12 + k);
                }
                j16[y * QPR + q] = (uint16_t)m;
            }
        err = cudaMemcpyAsync(h->jm16, j16, (size_t)L * QPR * 2, cudaMemcpyHostToDevice, h->stream);
    }
    if (err == cudaSuccess) err = cudaStreamSynchronize(h->stream);
    free(hx); free(jm); free(j16);
    if (err != cudaSuccess) { pa_note_cuda_error(h, err, "upload couplings", __FILE__, __LINE__); return PA_ERR_CUDA; }
    h->has_j = true;
    h->e0 = (int)((2 * n_af) % 4);
    return PA_OK;
}
int pa_level_offset(const pa_t* h) { return h ? h->e0 : 0; }

int pa_energies(pa_t* h, int32_t* E_out, int32_t* M_out) {
    PaDeviceGuard dg__(h);
    if (!h || !E_out) return PA_ERR_INVALID_ARG;
    int rc = pa_ensure_energies(h);
    if (rc != PA_OK) return rc;
    rc = pa_copy_out(h, E_out, h->E, sizeof(int32_t) * (size_t)h->R_cur, nullptr);
    if (rc == PA_OK && M_out) rc = pa_copy_out(h, M_out, h->M, sizeof(int32_t) * (size_t)h->R_cur, nullptr);
    return rc;
}

int pa_resample(pa_t* h, double beta, double beta_new, int64_t* R_new_out) {
    PaDeviceGuard dg__(h);
    if (!h || !(beta_new >= beta)) return PA_ERR_INVALID_ARG;
    const double dbeta = beta_new - beta;
    int rc;
    const bool timed = (h->timing & PA_TIME_RESAMPLE) != 0;
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[2], h->stream));
    // E_min / E_max: already on the host if pa_observables ran on this population (the usual loop, L62);
    // otherwise one measure launch and one read
    if ((rc = pa_ensure_host_scalars(h)) != PA_OK) return rc;
    const int Emin = h->Emin, Emax = h->Emax;
    if ((rc = pa_upload_wtab(h, dbeta, (Emax - Emin) / 4)) != PA_OK) return rc;
    // weights + W, plan (tau, r, scan, parents, R_new), copy: queued back to back; the copy reads R_new on
    // the device, so the host waits once, at the end
    // R_new and W travel to the host right after the plan kernel -- written by the kernel itself into mapped host memory
    // (PA_SNAP_HOST=0: by a copy operation) --; the copy kernel is queued behind and runs while the host wakes up, so the stream
    // never idles on this call's one synchronisation
    const bool mailed = h->h_snap_dev && pa_sw(h, PA_SW_SNAP_HOST, 1) != 0;
    h->mail_out = mailed ? h->h_snap_dev : nullptr;
    rc = pa_launch_weights_plan(h, Emin, h->w, false);
    h->mail_out = nullptr;
    if (rc != PA_OK) return rc;
    if (!mailed) PA_CUDA(h, cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(PaScalars), cudaMemcpyDeviceToHost, h->stream));
    PA_CUDA(h, cudaEventRecord(h->ev[6], h->stream));                // the host waits on this one (created without timing)
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[4], h->stream));
    if ((rc = pa_launch_copy(h)) != PA_OK) return rc;
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[5], h->stream));
    if (timed) PA_CUDA(h, cudaEventRecord(h->ev[3], h->stream));
    PA_CUDA(h, cudaEventSynchronize(h->ev[6]));
    h->resample_timed = timed;
    if (mailed) { h->h_scal->R_new = h->h_snap->R_new; h->h_scal->W = h->h_snap->W; }
    const int64_t R_new = (int64_t)h->h_scal->R_new;
    const double W = h->h_scal->W;
    if (R_new > h->R_cap || R_new < 1) { h->R_prev = 0; return PA_ERR_CAPACITY; }   // population, k, lnZ unchanged (O7): only the spare buffer was
                                                                                     // written -- and w, r, o: no resample vectors to export now
    h->R_prev = h->R_cur; h->W_last = W;
    const double lnQ = -dbeta * (double)Emin + log(W / (double)h->R_cur);   // Eq. 1 with the shift (O5)
    h->cur ^= 1;
    h->R_cur = R_new;
    h->k += 1;
    h->lnZ += lnQ;                                                    // Eq. 4 (L90)
    h->lnQ_last = lnQ;
    h->em_valid = false; h->host_scal_valid = false;
    if (R_new_out) *R_new_out = R_new;
    return PA_OK;
}

// alpha(dbeta) of Eq. 8 given Emin/Emax already on the host: two launches, one read
static int pa_eval_overlap(pa_handle* h, double dbeta, int Emin, int Emax, double* alpha) {
    int rc;
    if ((rc = pa_upload_wtab(h, dbeta, (Emax - Emin) / 4)) != PA_OK) return rc;
    if ((rc = pa_launch_weights(h, Emin, nullptr)) != PA_OK) return rc;
    const bool mailed = h->h_snap_dev && pa_sw(h, PA_SW_SNAP_HOST, 1) != 0;   // the kernel writes the sum into mapped host memory itself
    h->mail_out = mailed ? h->h_snap_dev : nullptr;
    rc = pa_launch_overlap(h, Emin);
    h->mail_out = nullptr;
    if (rc != PA_OK) return rc;
    if (mailed) { PA_CUDA(h, cudaStreamSynchronize(h->stream)); h->h_scal->sum = h->h_snap->sum; }
    else if ((rc = pa_read_scalars(h)) != PA_OK) return rc;
    *alpha = h->h_scal->sum / (double)h->R_cur;
    return PA_OK;
}

static int pa_overlap_prepare(pa_handle* h, int* Emin, int* Emax) {
    int rc;
    if ((rc = pa_ensure_host_scalars(h)) != PA_OK) return rc;
    *Emin = h->Emin; *Emax = h->Emax;
    return PA_OK;
}

int pa_overlap(pa_t* h, double dbeta, double* alpha) {
    PaDeviceGuard dg__(h);
    if (!h || !alpha || !(dbeta >= 0.0)) return PA_ERR_INVALID_ARG;
    int Emin, Emax, rc;
    if ((rc = pa_overlap_prepare(h, &Emin, &Emax)) != PA_OK) return rc;
    return pa_eval_overlap(h, dbeta, Emin, Emax, alpha);
}

// O10 with every alpha evaluated exactly (41 host round trips): the definition, kept as the reference path
// (PA_ADAPT_EXACT=1) and for populations whose energy range exceeds the filter's table.
static int pa_adapt_exact(pa_handle* h, double target, double hi, int Emin, int Emax, double* dbeta_out) {
    int rc; double a;
    if ((rc = pa_eval_overlap(h, hi, Emin, Emax, &a)) != PA_OK) return rc;
    h->adapt_exact_evals = 1;
    if (a >= target) { *dbeta_out = hi; return PA_OK; }
    double lo = 0.0;
    for (int it = 0; it < 40; ++it) {                                // O10: exactly 40 bisection steps
        const double mid = 0.5 * (lo + hi);
        if ((rc = pa_eval_overlap(h, mid, Emin, Emax, &a)) != PA_OK) return rc;
        h->adapt_exact_evals += 1;
        if (a >= target) lo = mid; else hi = mid;
    }
    *dbeta_out = lo;
    return PA_OK;
}

int pa_adapt_dbeta(pa_t* h, double target, double beta, double beta_max, double* dbeta_out) {
    PaDeviceGuard dg__(h);
    if (!h || !dbeta_out || !(target > 0.0 && target < 1.0) || !(beta_max > beta)) return PA_ERR_INVALID_ARG;
    int Emin, Emax, rc;
    if ((rc = pa_overlap_prepare(h, &Emin, &Emax)) != PA_OK) return rc;
    const double hi0 = beta_max - beta;
    const int dmax = (Emax - Emin) / 4;
    h->adapt_exact_evals = 0; h->adapt_filter_launches = 0; h->adapt_min_margin = INFINITY;
    if (pa_sw(h, PA_SW_ADAPT_EXACT, 0) != 0 || dmax + 1 > PA_ADAPT_BINS) return pa_adapt_exact(h, target, hi0, Emin, Emax, dbeta_out);
    // The same 41 decisions, most of them taken on the energy histogram inside one kernel (pa_adapt.cu): an iteration comes back
    // to the host only when the histogram sum is within `bound` of the target, and is then decided by the exact evaluation.
    // |alpha_hist - alpha_TREE1024| <= (2 R_cur + 2 dmax + 32) 2^-53 to first order; bound = 4 x that.
    const double bound = 4.0 * (2.0 * (double)h->R_cur + 2.0 * (double)dmax + 32.0) * 1.1102230246251565e-16;
    if ((rc = pa_launch_ehist(h)) != PA_OK) return rc;
    PaAdaptState* st = h->h_adapt;
    st->lo = 0.0; st->hi = hi0; st->it = -1; st->status = PA_ADAPT_DONE; st->margin = INFINITY; st->a_last = 0.0;
    for (;;) {
        if ((rc = pa_run_adapt_filter(h, target, bound)) != PA_OK) return rc;
        h->adapt_filter_launches += 1;
        h->adapt_min_margin = st->margin;
        if (st->status == PA_ADAPT_RETURN_HI) { *dbeta_out = hi0; return PA_OK; }
        if (st->status == PA_ADAPT_DONE) { *dbeta_out = st->lo; return PA_OK; }
        double a;
        if (st->status == PA_ADAPT_AMBIG_FIRST) {
            if ((rc = pa_eval_overlap(h, hi0, Emin, Emax, &a)) != PA_OK) return rc;
            h->adapt_exact_evals += 1;
            h->adapt_max_err = fmax(h->adapt_max_err, fabs(st->a_last - a) / (0.25 * bound));
            if (a >= target) { *dbeta_out = hi0; return PA_OK; }
            st->it = 0;
        } else {                                                     // PA_ADAPT_AMBIG: iteration st->it of the bracket [lo, hi]
            const double mid = 0.5 * (st->lo + st->hi);
            if ((rc = pa_eval_overlap(h, mid, Emin, Emax, &a)) != PA_OK) return rc;
            h->adapt_exact_evals += 1;
            h->adapt_max_err = fmax(h->adapt_max_err, fabs(st->a_last - a) / (0.25 * bound));   // the filter's alpha' against the exact alpha
            if (a >= target) st->lo = mid; else st->hi = mid;
            st->it += 1;
        }
        if (st->it >= 40) { *dbeta_out = st->lo; return PA_OK; }
    }
}

int pa_adapt_stats(const pa_t* h, int* exact_evaluations, int* filter_launches) {
    if (!h) return PA_ERR_INVALID_ARG;
    if (exact_evaluations) *exact_evaluations = h->adapt_exact_evals;
    if (filter_launches) *filter_launches = h->adapt_filter_launches;
    return PA_OK;
}

int pa_adapt_margins(const pa_t* h, double* min_margin, double* max_error) {
    if (!h) return PA_ERR_INVALID_ARG;
    if (min_margin) *min_margin = h->adapt_min_margin;
    if (max_error) *max_error = h->adapt_max_err;
    return PA_OK;
}

// Eq. 3-5 (O8) from the exact integer sums of a measured population
static void pa_fill_obs(const pa_handle* h, const PaScalars& s, double beta, int64_t R_cur, double lnZ, double lnQ, pa_obs_t* out) {
    const double R = (double)R_cur, N = (double)h->N;
    const __int128 num = (__int128)R_cur * (__int128)s.SE2 - (__int128)s.SE * (__int128)s.SE;   // exact (O8)
    out->beta = beta;
    out->e = (double)s.SE / (R * N);
    out->C = beta * beta * ((double)num / (R * R * N));
    out->absm = (double)s.SA / (R * N);
    out->m2 = (double)s.SM2 / (R * N * N);
    out->m4 = s.m4sum / R;
    out->betaF_per_N = -lnZ / N;
    out->S_per_N = beta * out->e + lnZ / N;
    out->lnQ = lnQ;
    out->R = R_cur;
}

int pa_observables(pa_t* h, double beta, pa_obs_t* out) {
    PaDeviceGuard dg__(h);
    if (!h || !out) return PA_ERR_INVALID_ARG;
    int rc;
    if ((rc = pa_ensure_host_scalars(h)) != PA_OK) return rc;
    pa_fill_obs(h, *h->h_scal, beta, h->R_cur, h->lnZ, h->lnQ_last, out);
    return PA_OK;
}

// ------------------------------------------------------------------------------------------------
// pa_anneal: n temperature steps (resample -> theta sweeps -> measure) enqueued back to back, with NO host round trip inside:
// the population size and E_min stay on the device (PaScalars::R_dev, mmin_inv), the weight tables of all steps of a chunk are
// built on the host beforehand for the full level range and uploaded once, and a snapshot of the device scalars is kept per
// step.  The host reads the snapshots at the end of the chunk and does exactly the arithmetic of pa_resample / pa_observables
// on them (ln Q, ln Z, Eq. 3-5), so every number equals the step-by-step calls'.
// ------------------------------------------------------------------------------------------------
struct PaAnnealCtx {            // host bookkeeping that runs along the snapshots, in step order
    int Emin_prev; int64_t R_prev;
    int done;                   // steps digested without error
};

// the arithmetic of pa_resample / pa_observables on the snapshots of one finished chunk
static int pa_anneal_digest(pa_handle* h, PaAnnealCtx& cx, const char* h_snaps, size_t snap, int s0, int cs, int n,
                            const double* betas, pa_obs_t* obs_out) {
    for (int i = 0; i < cs; ++i) {
        const PaScalars& S = *(const PaScalars*)(h_snaps + (size_t)i * snap);
        const double beta_old = betas[s0 + i], beta = betas[s0 + i + 1], dbeta = beta - beta_old;
        const int64_t R_new = (int64_t)S.R_new;
        if (S.err != 0u || R_new > h->R_cap || R_new < 1) { h->R_prev = 0; return PA_ERR_CAPACITY; }   // the failing step overwrote w, r, o
        const double lnQ = -dbeta * (double)cx.Emin_prev + log(S.W / (double)cx.R_prev);   // Eq. 1 with the shift (O5)
        h->lnZ += lnQ; h->lnQ_last = lnQ;                                                  // Eq. 4 (L90)
        h->R_prev = cx.R_prev; h->W_last = S.W;
        h->R_cur = R_new;
        if (obs_out) pa_fill_obs(h, S, beta, R_new, h->lnZ, lnQ, &obs_out[s0 + i]);
        cx.Emin_prev = -2 * h->nlev + 4 * (int)(0xffffffffu - S.mmin_inv) + h->e0;
        cx.R_prev = R_new;
        cx.done += 1;
        if (s0 + i == n - 1) {
            *h->h_scal = S;
            h->host_scal_valid = true; h->em_valid = true;
            h->Emin = cx.Emin_prev; h->Emax = -2 * h->nlev + 4 * (int)S.mmax + h->e0;
        }
    }
    return PA_OK;
}

int pa_anneal(pa_t* h, int n, const double* betas, int theta, pa_obs_t* obs_out) {
    PaDeviceGuard dg__(h);
    if (!h || !betas || n < 1 || theta < 0 || pa_is_device_ptr(betas) || (obs_out && pa_is_device_ptr(obs_out))) return PA_ERR_INVALID_ARG;
    for (int i = 0; i <= n; ++i) if (!(betas[i] == betas[i]) || (i > 0 && !(betas[i] >= betas[i - 1]))) return PA_ERR_INVALID_ARG;
    int rc;
    if ((rc = pa_ensure_host_scalars(h)) != PA_OK) return rc;
    // Steps go in chunks with two staging buffers: while the device runs chunk c the host builds the weight tables of chunk
    // c+1 (N+1 exponentials per step) and digests the snapshots of chunk c-1.
    const size_t tab = (size_t)h->nlev + 1, snap = (sizeof(PaScalars) + 15) / 16 * 16;
    const size_t per_step = tab * 8 + snap;
    int chunk_cap = (int)(h->stage_bytes / 2 / per_step);
    if (chunk_cap > 16) chunk_cap = 16;
    { const long long ec = pa_sw(h, PA_SW_ANNEAL_CHUNK, 0);         // tests: force other chunk sizes
      if (ec >= 1 && ec < chunk_cap) chunk_cap = (int)ec; }
    if (chunk_cap < 1) return PA_ERR_WORKSPACE;
    if (chunk_cap > n) chunk_cap = n;
    const size_t buf_bytes = ((size_t)chunk_cap * per_step + 255) / 256 * 256;
    const size_t need = 2 * buf_bytes + 16;
    if (h->h_tabs_bytes < need) {
        if (h->h_tabs) cudaFreeHost(h->h_tabs);                      // (the chunk events live until pa_destroy)
        h->h_tabs = nullptr; h->h_tabs_bytes = 0;
        PA_CUDA(h, cudaMallocHost(&h->h_tabs, need));
        h->h_tabs_bytes = need;
    }
    for (int b = 0; b < 2; ++b)
        if (!h->ev_chunk[b]) PA_CUDA(h, cudaEventCreateWithFlags(&h->ev_chunk[b], cudaEventDisableTiming));
    // the device copy of the population size
    uint32_t* h_init = (uint32_t*)((char*)h->h_tabs + 2 * buf_bytes);
    h_init[0] = (uint32_t)h->R_cur; h_init[1] = 0u;
    PA_CUDA(h, cudaMemcpyAsync(&h->d_scal->R_dev, h_init, 8, cudaMemcpyHostToDevice, h->stream));
    PaAnnealCtx cx = {h->Emin, h->R_cur, 0};
    const int cur0 = h->cur; const uint32_t k0 = h->k, t0 = h->t;   // to put the bookkeeping back if a step fails (below)
    int pend_s0[2] = {-1, -1}, pend_cs[2] = {0, 0};
    rc = PA_OK;
    int c = 0;
    int cs = 0;
    for (int s0 = 0; s0 < n && rc == PA_OK; s0 += cs, ++c) {
        const int b = c & 1;
        // chunk sizes 1, 2, 4, ... up to the capacity: the device starts after one table, and the host stays ahead of it
        cs = c < 30 && (1 << c) < chunk_cap ? (1 << c) : chunk_cap;
        if (cs > n - s0) cs = n - s0;
        char* hb = (char*)h->h_tabs + (size_t)b * buf_bytes;
        char* db = (char*)h->stage + (size_t)b * buf_bytes;
        double *h_t = (double*)hb, *d_t = (double*)db;
        char *h_snaps = hb + (size_t)chunk_cap * tab * 8, *d_snaps = db + (size_t)chunk_cap * tab * 8;
        if (pend_s0[b] >= 0) {                                       // chunk c-2 used this buffer: wait for it and digest it
            if (cudaEventSynchronize(h->ev_chunk[b]) != cudaSuccess) { rc = PA_ERR_CUDA; break; }
            rc = pa_anneal_digest(h, cx, h_snaps, snap, pend_s0[b], pend_cs[b], n, betas, obs_out);
            pend_s0[b] = -1;
            if (rc != PA_OK) break;
        }
        for (int i = 0; i < cs; ++i) {                               // O5: wtab[d] = exp(-(dbeta * (double)(4 d))), full level range
            const double dbeta = betas[s0 + i + 1] - betas[s0 + i];
            double* t = h_t + (size_t)i * tab;
            // the first step of the call is on the critical path (nothing is running yet) and its population is known on the
            // host: only the levels it occupies are read; the later tables are built while the device works
            const int dlast = (s0 + i == 0) ? (h->Emax - h->Emin) / 4 : h->nlev;
            for (int d = 0; d <= dlast; ++d) t[d] = exp(-(dbeta * (double)(4 * d)));
        }
        if (cudaMemcpyAsync(d_t, h_t, (size_t)cs * tab * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess) { rc = PA_ERR_CUDA; break; }
        h->dev_R = true;
        const bool fuse_copy = pa_sw(h, PA_SW_FUSE_COPY, 1) != 0;
        for (int i = 0; i < cs && rc == PA_OK; ++i) {
            const double beta = betas[s0 + i + 1];
            h->wtab_cur = d_t + (size_t)i * tab;
            if (h->timing & PA_TIME_RESAMPLE) cudaEventRecord(h->ev[2], h->stream);
            // small populations on the lane-split sweep kernel: the sweep launch gathers the new population while it stages its
            // strip, so the step is three launches (plan, sweep, measure) instead of four
            const bool gather = fuse_copy && pa_sweep_gathers(h, theta);
            if ((rc = pa_launch_weights_plan(h, 0, h->w, gather)) != PA_OK) break;
            if (h->timing & PA_TIME_RESAMPLE) cudaEventRecord(h->ev[4], h->stream);
            if (!gather && (rc = pa_launch_copy(h)) != PA_OK) break;
            if (h->timing & PA_TIME_RESAMPLE) cudaEventRecord(h->ev[5], h->stream);
            if (h->timing & PA_TIME_RESAMPLE) cudaEventRecord(h->ev[3], h->stream);
            h->cur ^= 1; h->k += 1;
            const uint32_t T4 = pa_threshold(exp(-4.0 * beta)), T8 = pa_threshold(exp(-8.0 * beta));
            h->T12 = pa_threshold(exp(-12.0 * beta));
            if (h->timing & PA_TIME_SWEEP) cudaEventRecord(h->ev[0], h->stream);
            if ((rc = gather ? pa_launch_sweep_gather(h, T4, T8, theta) : pa_launch_sweep(h, T4, T8, theta)) != PA_OK) break;
            if (h->timing & PA_TIME_SWEEP) cudaEventRecord(h->ev[1], h->stream);
            h->t += (uint32_t)theta;
            h->snap_out = (PaScalars*)(d_snaps + (size_t)i * snap);   // the measure kernel's last CTA leaves the snapshot there
            rc = pa_launch_measure(h);
            h->snap_out = nullptr;
        }
        h->dev_R = false; h->wtab_cur = nullptr; h->scal_zeroed = false;
        if (rc != PA_OK) break;
        if (cudaMemcpyAsync(h_snaps, d_snaps, (size_t)cs * snap, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
            cudaEventRecord(h->ev_chunk[b], h->stream) != cudaSuccess) { rc = PA_ERR_CUDA; break; }
        pend_s0[b] = s0; pend_cs[b] = cs;
        h->sweep_timed = theta > 0 && (h->timing & PA_TIME_SWEEP); h->resample_timed = (h->timing & PA_TIME_RESAMPLE) != 0;
    }
    // drain: the chunks still in flight, oldest first
    cudaError_t se = cudaStreamSynchronize(h->stream);
    if (rc == PA_OK && se != cudaSuccess) { pa_note_cuda_error(h, se, "pa_anneal drain", __FILE__, __LINE__); rc = PA_ERR_CUDA; }
    for (int k = 0; k < 2 && rc == PA_OK; ++k) {
        const int b = pend_s0[0] >= 0 && (pend_s0[1] < 0 || pend_s0[0] < pend_s0[1]) ? 0 : 1;
        if (pend_s0[b] < 0) break;
        const char* h_snaps = (const char*)h->h_tabs + (size_t)b * buf_bytes + (size_t)chunk_cap * tab * 8;
        rc = pa_anneal_digest(h, cx, h_snaps, snap, pend_s0[b], pend_cs[b], n, betas, obs_out);
        pend_s0[b] = -1;
    }
    if (rc == PA_ERR_CAPACITY) {
        // Step f = k - k0 + 1 (1-based) left [1, R_cap].  Its copy went to the spare buffer, the device raised sc->err, and every
        // later kernel of the call saw an empty population (pa_live_R) and exited: the population is the one before that step,
        // exactly as after a failed pa_resample (O7).  The digest stopped there too (R_cur, ln Z, obs_out[0..f-2] are those of the
        // steps that succeeded); the counters follow.
        h->cur = cur0 ^ (cx.done & 1); h->k = k0 + (uint32_t)cx.done; h->t = t0 + (uint32_t)cx.done * (uint32_t)theta;
    }
    if (rc != PA_OK) { h->em_valid = false; h->host_scal_valid = false; }
    return rc;
}

int pa_hist_accumulate(pa_t* h, double beta) {
    PaDeviceGuard dg__(h);
    if (!h) return PA_ERR_INVALID_ARG;
    int rc;
    if ((rc = pa_ensure_energies(h)) != PA_OK) return rc;
    h->hist_any = true;
    return pa_launch_hist(h, beta);
}

int pa_get_histogram(pa_t* h, int64_t* Hsum, double* lnD) {
    PaDeviceGuard dg__(h);
    if (!h) return PA_ERR_INVALID_ARG;
    int rc = PA_OK;
    if (Hsum) rc = pa_copy_out(h, Hsum, h->Hsum, ((size_t)h->nlev + 1) * 8, nullptr);
    if (rc == PA_OK && lnD) rc = pa_copy_out(h, lnD, h->lnD, ((size_t)h->nlev + 1) * 8, nullptr);
    return rc;
}

int pa_reweight(pa_t* h, int n, const double* betas, double* lnZ, double* e, double* C, double* absm, double* m2) {
    PaDeviceGuard dg__(h);
    if (!h || !betas || n < 1 || n > (1 << 20)) return PA_ERR_INVALID_ARG;
    if ((size_t)n * 48 > h->stage_bytes) return PA_ERR_INVALID_ARG;
    // any histogram yet?  (Hsum is all zero until the first pa_hist_accumulate)
    if (!h->hist_any) return PA_ERR_INVALID_ARG;
    double* d_io = (double*)h->stage;
    const bool dev = pa_is_device_ptr(betas);
    PA_CUDA(h, cudaMemcpyAsync(d_io, betas, (size_t)n * 8, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    int rc = pa_launch_reweight(h, n, d_io);
    if (rc != PA_OK) return rc;
    double* outs[5] = {lnZ, e, C, absm, m2};
    for (int i = 0; i < 5 && rc == PA_OK; ++i)
        if (outs[i]) rc = pa_copy_out(h, outs[i], d_io + (size_t)(i + 1) * n, (size_t)n * 8, nullptr);
    return rc;
}

int pa_get_mag_sums(pa_t* h, int64_t* A1, int64_t* A2) {
    PaDeviceGuard dg__(h);
    if (!h) return PA_ERR_INVALID_ARG;
    int rc = PA_OK;
    if (A1) rc = pa_copy_out(h, A1, h->A1, ((size_t)h->nlev + 1) * 8, nullptr);
    if (rc == PA_OK && A2) rc = pa_copy_out(h, A2, h->A2, ((size_t)h->nlev + 1) * 8, nullptr);
    return rc;
}

int pa_weighted_average(int M, const double* lnZ, const double* A, int nobs, double* A_out, double* omega_out) {
    if (M < 1 || nobs < 0 || !lnZ || (nobs > 0 && (!A || !A_out))) return PA_ERR_INVALID_ARG;
    double* d = nullptr;
    const size_t nA = (size_t)M * nobs, total = (size_t)M * 2 + nA + (size_t)nobs;
    if (cudaMalloc(&d, (total ? total : 1) * 8) != cudaSuccess) { cudaGetLastError(); return PA_ERR_CUDA; }
    double *d_lnZ = d, *d_om = d + M, *d_A = d + 2 * (size_t)M, *d_out = d_A + nA;
    cudaError_t err = cudaMemcpy(d_lnZ, lnZ, (size_t)M * 8, cudaMemcpyHostToDevice);
    if (err == cudaSuccess && nA) err = cudaMemcpy(d_A, A, nA * 8, cudaMemcpyHostToDevice);
    if (err == cudaSuccess) err = pa_run_wavg(M, d_lnZ, d_A, nobs, d_out, d_om, 0);
    if (err == cudaSuccess && nobs) err = cudaMemcpy(A_out, d_out, (size_t)nobs * 8, cudaMemcpyDeviceToHost);
    if (err == cudaSuccess && omega_out) err = cudaMemcpy(omega_out, d_om, (size_t)M * 8, cudaMemcpyDeviceToHost);
    if (err == cudaSuccess) err = cudaDeviceSynchronize();
    cudaFree(d);
    if (err != cudaSuccess) { cudaGetLastError(); return PA_ERR_CUDA; }
    return PA_OK;
}

static int pa_get_spins_impl(pa_handle* h, const int64_t* slots, int64_t j0, int64_t n, int8_t* out) {
    const bool dev_out = pa_is_device_ptr(out);
    const size_t N = (size_t)h->N;
    int64_t chunk = (int64_t)(h->stage_bytes / N);
    if (chunk > PA_SLOTS_CAP) chunk = PA_SLOTS_CAP;
    if (chunk < 1) return PA_ERR_WORKSPACE;
    int64_t* d_slots = h->d_slots;
    for (int64_t a = 0; a < n; a += chunk) {
        const int64_t m = n - a < chunk ? n - a : chunk;
        if (slots) PA_CUDA(h, cudaMemcpyAsync(d_slots, slots + a, sizeof(int64_t) * (size_t)m, cudaMemcpyHostToDevice, h->stream));
        int8_t* target = dev_out ? out + (size_t)a * N : h->stage;
        int rc = pa_launch_unpack(h, slots ? d_slots : nullptr, j0 + a, m, target);
        if (rc != PA_OK) return rc;
        if (!dev_out) {
            PA_CUDA(h, cudaMemcpyAsync(out + (size_t)a * N, h->stage, (size_t)m * N, cudaMemcpyDeviceToHost, h->stream));
            PA_CUDA(h, cudaStreamSynchronize(h->stream));
        } else if (slots) {
            PA_CUDA(h, cudaStreamSynchronize(h->stream));
        }
    }
    return PA_OK;
}

int pa_get_spins(pa_t* h, int64_t j0, int64_t nrep, int8_t* out) {
    PaDeviceGuard dg__(h);
    if (!h || !out || j0 < 0 || nrep < 0 || j0 + nrep > h->R_cur) return PA_ERR_INVALID_ARG;
    return pa_get_spins_impl(h, nullptr, j0, nrep, out);
}

int pa_get_spins_at(pa_t* h, const int64_t* slots, int64_t n, int8_t* out) {
    PaDeviceGuard dg__(h);
    if (!h || !out || !slots || n < 0) return PA_ERR_INVALID_ARG;
    for (int64_t i = 0; i < n; ++i) if (slots[i] < 0 || slots[i] >= h->R_cur) return PA_ERR_INVALID_ARG;
    return pa_get_spins_impl(h, slots, 0, n, out);
}

int pa_set_spins(pa_t* h, int64_t j0, int64_t nrep, const int8_t* in) {
    PaDeviceGuard dg__(h);
    if (!h || !in || j0 < 0 || nrep < 0 || j0 + nrep > h->R_cur) return PA_ERR_INVALID_ARG;
    const bool dev_in = pa_is_device_ptr(in);
    const size_t N = (size_t)h->N;
    const int64_t chunk = (int64_t)(h->stage_bytes / N);
    for (int64_t a = 0; a < nrep; a += chunk) {
        const int64_t m = nrep - a < chunk ? nrep - a : chunk;
        const int8_t* src = in + (size_t)a * N;
        if (!dev_in) {
            PA_CUDA(h, cudaMemcpyAsync(h->stage, src, (size_t)m * N, cudaMemcpyHostToDevice, h->stream));
            src = h->stage;
        }
        int rc = pa_launch_pack(h, j0 + a, m, src);
        if (rc != PA_OK) return rc;
        PA_CUDA(h, cudaStreamSynchronize(h->stream));
    }
    h->em_valid = false; h->host_scal_valid = false;
    return PA_OK;
}

int pa_get_words(pa_t* h, uint32_t* words) {
    PaDeviceGuard dg__(h);
    if (!h || !words) return PA_ERR_INVALID_ARG;
    const size_t bytes = (size_t)((h->R_cur + 31) / 32) * h->N * 4;
    if (pa_is_device_ptr(words)) return pa_launch_words_out(h, words);
    // host destination: convert into the spare population buffer, then copy out
    int rc = pa_launch_words_out(h, h->spins[1 - h->cur]);
    if (rc != PA_OK) return rc;
    PA_CUDA(h, cudaMemcpyAsync(words, h->spins[1 - h->cur], bytes, cudaMemcpyDeviceToHost, h->stream));
    PA_CUDA(h, cudaStreamSynchronize(h->stream));
    return PA_OK;
}

int pa_set_words(pa_t* h, int64_t R, const uint32_t* words) {
    PaDeviceGuard dg__(h);
    if (!h || !words || R < 1 || R > h->R_cap) return PA_ERR_INVALID_ARG;
    const size_t bytes = (size_t)((R + 31) / 32) * h->N * 4;
    const uint32_t* src = words;
    if (!pa_is_device_ptr(words)) {
        PA_CUDA(h, cudaMemcpyAsync(h->spins[1 - h->cur], words, bytes, cudaMemcpyHostToDevice, h->stream));
        src = h->spins[1 - h->cur];
    }
    int rc = pa_launch_words_in(h, R, src);
    if (rc != PA_OK) return rc;
    h->R_cur = R;
    h->em_valid = false; h->host_scal_valid = false;
    return PA_OK;
}

// One temperature step with the population living in HOST memory between steps (the end-to-end shape of bench.py): exactly
// pa_set_words, pa_resample, pa_sweep, pa_observables, pa_energies, pa_get_words in this order, with the same results -- but the
// sweeps run in chunks of groups (whole rounds of the 148 SMs), and a finished chunk is converted to the interchange layout and
// copied to the host on a second stream while the next chunks are swept: the 8.2 GB that cfg5 sends back per step hide behind
// 0.39 s of sweeps, and only the upload (which the resampling plan needs complete) and the last chunk stay exposed.
int pa_step_host(pa_t* h, int64_t R_in, const uint32_t* words_in, double beta, double beta_new, int theta,
                 uint32_t* words_out, int32_t* E_out, int32_t* M_out, pa_obs_t* obs_out, int64_t* R_new_out) {
    PaDeviceGuard dg__(h);
    if (!h || !words_in || !words_out || theta < 0 || !(beta_new >= beta) || pa_is_device_ptr(words_in) || pa_is_device_ptr(words_out))
        return PA_ERR_INVALID_ARG;
    int rc;
    if ((rc = pa_set_words(h, R_in, words_in)) != PA_OK) return rc;
    int64_t R_new = 0;
    if ((rc = pa_resample(h, beta, beta_new, &R_new)) != PA_OK) return rc;
    if (R_new_out) *R_new_out = R_new;
    const int64_t G = (R_new + 31) / 32;
    // chunks of whole rounds: multiples of 148 groups, about 16 per step; small populations go in one piece
    int64_t chunk = G / 16 / h->n_sm * h->n_sm;
    chunk = pa_sw(h, PA_SW_STEP_HOST_CHUNK, chunk);                  // tests: force a chunk size (groups), 0 = one piece
    bool piped = chunk >= 1 && chunk < G && theta > 0;
    bool copies_in_flight = false;
    rc = PA_OK;
    if (piped) {
        if (!h->xfer_stream) PA_CUDA(h, cudaStreamCreateWithFlags(&h->xfer_stream, cudaStreamNonBlocking));   // (nothing in flight yet)
        if (!h->ev_xfer) PA_CUDA(h, cudaEventCreateWithFlags(&h->ev_xfer, cudaEventDisableTiming));
        const uint32_t T4 = pa_threshold(exp(-4.0 * beta_new)), T8 = pa_threshold(exp(-8.0 * beta_new));
        uint32_t* stage = h->spins[1 - h->cur];                      // the population before resampling: no longer needed
        for (int64_t g0 = 0; g0 < G; g0 += chunk) {
            const int64_t ng = g0 + chunk <= G ? chunk : G - g0;
            rc = pa_launch_sweep_range(h, T4, T8, theta, g0, ng);
            if (rc == PA_ERR_INVALID_ARG && g0 == 0) { piped = false; rc = PA_OK; break; }     // this geometry has no range launch: one piece
            if (rc != PA_OK) break;
            if ((rc = pa_launch_words_out_range(h, stage, g0, ng)) != PA_OK) break;
            cudaError_t ce = cudaEventRecord(h->ev_xfer, h->stream);
            if (ce == cudaSuccess) ce = cudaStreamWaitEvent(h->xfer_stream, h->ev_xfer, 0);
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(words_out + g0 * (size_t)h->N, stage + g0 * (size_t)h->N, (size_t)ng * h->N * 4,
                                                        cudaMemcpyDeviceToHost, h->xfer_stream);
            if (ce != cudaSuccess) { pa_note_cuda_error(h, ce, "pa_step_host: copy of a finished chunk", __FILE__, __LINE__); rc = PA_ERR_CUDA; break; }
            copies_in_flight = true;
        }
        if (piped && rc == PA_OK) { h->t += (uint32_t)theta; h->em_valid = false; h->host_scal_valid = false; h->sweep_timed = false; }
    }
    if (rc == PA_OK && !piped) rc = pa_sweep(h, beta_new, theta);
    if (rc == PA_OK && obs_out) rc = pa_observables(h, beta_new, obs_out);
    if (rc == PA_OK && E_out) rc = pa_energies(h, E_out, M_out);
    if (rc == PA_OK && !piped) rc = pa_get_words(h, words_out);
    if (copies_in_flight) {
        // every exit, errors included: no copy into the caller's words_out is left running, and the staging buffer (the spare
        // population) is free for the next call
        const cudaError_t c1 = cudaStreamSynchronize(h->xfer_stream), c2 = cudaStreamSynchronize(h->stream);
        if (rc == PA_OK && (c1 != cudaSuccess || c2 != cudaSuccess)) {
            pa_note_cuda_error(h, c1 != cudaSuccess ? c1 : c2, "pa_step_host: drain", __FILE__, __LINE__);
            rc = PA_ERR_CUDA;
        }
    }
    return rc;
}

int pa_get_resample_debug(pa_t* h, double* W, double* w, uint32_t* r, uint32_t* o) {
    PaDeviceGuard dg__(h);
    if (!h) return PA_ERR_INVALID_ARG;
    int rc = PA_OK;
    if (h->R_prev == 0) return PA_ERR_INVALID_ARG;                   // no resampling step yet, or the last one failed
    const size_t n = (size_t)h->R_prev;
    if (W) *W = h->W_last;
    if (w) rc = pa_copy_out(h, w, h->w, n * 8, nullptr);
    if (rc == PA_OK && r) rc = pa_copy_out(h, r, h->r, n * 4, nullptr);
    if (rc == PA_OK && o) rc = pa_copy_out(h, o, h->o, n * 4, nullptr);
    return rc;
}

int64_t pa_population(const pa_t* h) { return h ? h->R_cur : 0; }
int64_t pa_prev_population(const pa_t* h) { return h ? h->R_prev : 0; }
int64_t pa_capacity_of(const pa_t* h) { return h ? h->R_cap : 0; }
uint32_t pa_sweep_counter(const pa_t* h) { return h ? h->t : 0; }
uint32_t pa_resample_counter(const pa_t* h) { return h ? h->k : 0; }
double pa_lnZ(const pa_t* h) { return h ? h->lnZ : 0.0; }
int pa_set_counters(pa_t* h, uint32_t t, uint32_t k, double lnZ) {
    if (!h) return PA_ERR_INVALID_ARG;
    h->t = t; h->k = k; h->lnZ = lnZ;
    return PA_OK;
}
int64_t pa_launch_count(const pa_t* h) { return h ? h->launches : 0; }
int pa_last_sweep_kind(const pa_t* h) { return h ? h->last_sweep_kind : 0; }

int pa_set_timing(pa_t* h, int mask) {
    if (!h || mask < 0 || mask > (PA_TIME_SWEEP | PA_TIME_RESAMPLE | PA_TIME_MEASURE)) return PA_ERR_INVALID_ARG;
    h->timing = mask;
    return PA_OK;
}

int pa_last_sweep_ms(pa_t* h, float* kernel_ms) {
    PaDeviceGuard dg__(h);
    if (!h || !h->sweep_timed) return PA_ERR_INVALID_ARG;
    PA_CUDA(h, cudaEventSynchronize(h->ev[1]));
    float ms = 0.f;
    PA_CUDA(h, cudaEventElapsedTime(&ms, h->ev[0], h->ev[1]));
    if (kernel_ms) *kernel_ms = ms;
    return PA_OK;
}
int pa_last_resample_ms(pa_t* h, float* total_ms, float* copy_kernel_ms) {
    PaDeviceGuard dg__(h);
    if (!h || !h->resample_timed) return PA_ERR_INVALID_ARG;
    PA_CUDA(h, cudaEventSynchronize(h->ev[3]));
    float a = 0.f, b = 0.f;
    PA_CUDA(h, cudaEventElapsedTime(&a, h->ev[2], h->ev[3]));
    PA_CUDA(h, cudaEventElapsedTime(&b, h->ev[4], h->ev[5]));
    if (total_ms) *total_ms = a;
    if (copy_kernel_ms) *copy_kernel_ms = b;
    return PA_OK;
}

int pa_last_measure_ms(pa_t* h, float* kernel_ms) {
    PaDeviceGuard dg__(h);
    if (!h || !h->measure_timed) return PA_ERR_INVALID_ARG;
    PA_CUDA(h, cudaEventSynchronize(h->ev[8]));
    float ms = 0.f;
    PA_CUDA(h, cudaEventElapsedTime(&ms, h->ev[7], h->ev[8]));
    if (kernel_ms) *kernel_ms = ms;
    return PA_OK;
}

int pa_calibrate(int kind, double* ginstr_per_ns, double* sm_mhz) { return pa_run_calibrate(kind, ginstr_per_ns, sm_mhz); }

static const char* const pa_switch_names[PA_SW_COUNT] = {
    "PA_PDL", "PA_SNAP_HOST", "PA_ADAPT_EXACT", "PA_ANNEAL_CHUNK", "PA_FUSE_COPY", "PA_STEP_HOST_CHUNK", "PA_MEASURE_GENERIC",
    "PA_SMALL_PLAN", "PA_SWEEP_C", "PA_SWEEP_T", "PA_SWEEP_SMEM_KB", "PA_SWEEP_KIND", "PA_SWEEP_CMP", "PA_SWEEP_MIXED",
    "PA_LCG_P64", "PA_LCG_NOR", "PA_SWEEP_SPLIT"};

int pa_set_switch(pa_t* h, const char* name, int is_set, int64_t value) {
    const int k = name ? pa_switch_index(name) : -1;
    if (!h || k < 0) return PA_ERR_INVALID_ARG;
    PaDeviceGuard dg__(h);
    const PaSwitches saved = h->sw;
    const int pdl = h->pdl;
    h->sw.set[k] = is_set != 0; h->sw.val[k] = value;
    h->pdl = pa_sw(h, PA_SW_PDL, 1) == 0 ? 0 : 1;
    const int rc = pa_sweep_configure(h);                 // the sweep geometry follows its switches
    if (rc != PA_OK) { h->sw = saved; h->pdl = pdl; pa_sweep_configure(h); }
    return rc;
}

const char* pa_strerror(int code) {
    switch (code) {
        case PA_OK: return "ok";
        case PA_ERR_INVALID_ARG: return "invalid argument";
        case PA_ERR_CAPACITY: return "resampled population would exceed the capacity (or be empty)";
        case PA_ERR_CUDA: return "CUDA error";
        case PA_ERR_WORKSPACE: return "workspace too small or misaligned";
        case PA_ERR_NOMEM: return "out of memory";
        case PA_ERR_STATIC_LIMIT: return "more runs than the fixed scratch array of pa_weighted_average_static holds (PA_WAVG_STATIC_MAX_RUNS)";
        default: return "unknown error";
    }
}
const char* pa_last_cuda_error(const pa_t* h) { return h ? h->cuda_err : ""; }
const char* pa_version(void) { return "pa-b200 0.1 (sm_100a)"; }

}  // extern "C"

void pa_switches_read(PaSwitches* sw) {
    for (int k = 0; k < PA_SW_COUNT; ++k) {
        const char* v = getenv(pa_switch_names[k]);
        sw->set[k] = v != nullptr;
        sw->val[k] = v ? atoll(v) : 0;
    }
}
int pa_switch_index(const char* name) {
    for (int k = 0; k < PA_SW_COUNT; ++k)
        if (strcmp(name, pa_switch_names[k]) == 0) return k;
    return -1;
}
