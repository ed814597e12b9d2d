// pa_resample.cu -- the resampling chain:
//   weights + TREE1024 normaliser, tau / copy numbers / decoupled look-back exclusive scan / parent map,
//   and the bit-lane gather copy into the new population.  Three launches per resampling step, no host
//   round trip between them (E_min comes from the measure kernel of the previous step's observables).
#include "pa_common.cuh"
#include <stdlib.h>

// ------------------------------------------------------------------------------------------------
// TREE1024 (O5; L165 "sum the per-block partial results in a subsequent kernel call"): one CTA of
// 1024 threads per aligned block of 1024 values.  __shfl_down trees give, in lane 0, exactly
// a[i] += a[i+off] (off = 16,8,4,2,1); the 32 run sums are combined by the same tree; the block
// sums are then added sequentially in ascending block order -- by the last CTA to finish (atomic
// ticket), which replaces the paper's second kernel call and keeps the fixed order.
//   MODE 0: v_j = w_j = wtab[(E_j - E_min)/4]  (stored to w_out if given)   -> sc->W
//           also clears this tile's look-back state and the tile ticket for the plan kernel
//   MODE 1: v_j = min(1, R_target * w_j / W)    (Eq. 8 summand)             -> sc->sum
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(PA_TILE)
pa_tree_kernel(const int32_t* __restrict__ E, const double* __restrict__ wtab, PaScalars* __restrict__ sc,
               long long R, double R_target, int Emin, double* __restrict__ w_out, double* __restrict__ partials,
               unsigned long long* __restrict__ scan_state, int N, int e0, PaScalars* __restrict__ mail) {
    __shared__ double run[32];
    __shared__ bool s_last;
    pa_pdl_wait(); pa_pdl_launch();
    R = pa_live_R(R, sc);
    Emin = pa_live_Emin(Emin, sc, N, e0);
    const long long j = (long long)blockIdx.x * PA_TILE + threadIdx.x;
    double v = 0.0;
    if (j < R) {
        const double w = wtab[(E[j] - Emin) >> 2];
        if (MODE == 0) { v = w; if (w_out) w_out[j] = w; }
        else { const double tau = __ddiv_rn(__dmul_rn(R_target, w), sc->W); v = tau < 1.0 ? tau : 1.0; }
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));
    if ((threadIdx.x & 31) == 0) run[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = run[threadIdx.x];
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));
        if (threadIdx.x == 0) {
            partials[blockIdx.x] = v;
            if (MODE == 0) { scan_state[blockIdx.x] = 0ull; if (blockIdx.x == 0) sc->tile_counter = 0u; }
            __threadfence();
            s_last = atomicAdd(&sc->tree_ticket, 1u) == gridDim.x - 1;
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // last CTA: block sums in ascending order, staged through shared memory 1024 at a time
    __shared__ double stage[PA_TILE];
    double total = 0.0;
    const int n = gridDim.x;
    for (int base = 0; base < n; base += PA_TILE) {
        const int i = base + threadIdx.x;
        stage[threadIdx.x] = i < n ? __ldcg(partials + i) : 0.0;
        __syncthreads();
        if (threadIdx.x == 0) {
            const int m = min(PA_TILE, n - base);
            for (int q = 0; q < m; ++q) total = __dadd_rn(total, stage[q]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (MODE == 0) sc->W = total; else { sc->sum = total; if (mail) mail->sum = total; }    // mail: mapped host memory (pa_eval_overlap)
        sc->tree_ticket = 0u;
    }
}

int pa_launch_weights(pa_handle* h, int Emin, double* w_out) {
    const int n = (int)(((h->dev_R ? h->R_cap : h->R_cur) + PA_TILE - 1) / PA_TILE);
    PA_CUDA(h, pa_launch(h, pa_tree_kernel<0>, dim3(n), dim3(PA_TILE), 0, (const int32_t*)h->E, h->wtab_cur ? h->wtab_cur : (const double*)h->wtab,
                         h->d_scal, (long long)(h->dev_R ? -1 : h->R_cur), (double)h->R_target, h->dev_R ? PA_EMIN_DEV : Emin, w_out,
                         h->partials, h->scan_state, h->nlev, h->e0, (PaScalars*)nullptr));
    h->launches += 1;
    return PA_OK;
}

int pa_launch_overlap(pa_handle* h, int Emin) {
    const int n = (int)((h->R_cur + PA_TILE - 1) / PA_TILE);
    PA_CUDA(h, pa_launch(h, pa_tree_kernel<1>, dim3(n), dim3(PA_TILE), 0, (const int32_t*)h->E, (const double*)h->wtab, h->d_scal,
                         (long long)h->R_cur, (double)h->R_target, Emin, (double*)nullptr, h->partials, h->scan_state, h->nlev, h->e0, h->mail_out));
    h->launches += 1;
    return PA_OK;
}

// ------------------------------------------------------------------------------------------------
// Plan: tau_j = R w_j / W (one multiply, one divide, O6), r_j = floor(tau_j) + [u_j < frac tau_j]
// (Eq. 2 L67 with strict '<'), o_j = exclusive prefix sum (L165 CalcParSum), parent[o_j + c] = j.
// Single-pass decoupled look-back scan over tiles of 1024 (256 threads x 4), no library.
// Tile ids are handed out by an atomic counter so that a tile's predecessors have always started.
// ------------------------------------------------------------------------------------------------
#define PA_FLAG_AGG (1ull << 32)
#define PA_FLAG_PREFIX (2ull << 32)

__global__ void __launch_bounds__(256)
pa_plan_kernel(const int32_t* __restrict__ E, const double* __restrict__ wtab, PaScalars* sc,
               long long R, double R_target, int Emin, PhiloxKeys K, uint32_t kcount, long long R_cap,
               uint32_t* __restrict__ r_out, uint32_t* __restrict__ o_out, uint32_t* __restrict__ parent,
               unsigned long long* __restrict__ state, int n_tiles, int N, int e0, PaScalars* __restrict__ mail) {
    __shared__ uint32_t s_tile, s_warp[8], s_excl;
    pa_pdl_wait(); pa_pdl_launch();
    R = pa_live_R(R, sc);
    Emin = pa_live_Emin(Emin, sc, N, e0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(&sc->tile_counter, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long j0 = (long long)tile * PA_TILE + tid * 4;

    uint32_t r[4] = {0, 0, 0, 0};
    if (j0 < R) {
        const double W = sc->W;
        // x(j,k) = philox(j>>2, 0, k, TAG_RESAMPLE)[j&3]   (O1)
        uint4 x = pa_philox((uint32_t)(j0 >> 2), 0u, kcount, PA_TAG_RESAMPLE, K);
        const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (j0 + q < R) {
                double w = wtab[(E[j0 + q] - Emin) >> 2];
                double tau = __ddiv_rn(__dmul_rn(R_target, w), W);
                double n = floor(tau);
                double f = __dsub_rn(tau, n);
                double u = __dmul_rn((double)xs[q], 1.0 / 4294967296.0);
                r[q] = (uint32_t)n + (u < f ? 1u : 0u);
            }
        }
    }
    const uint32_t tsum = r[0] + r[1] + r[2] + r[3];
    // block-wide exclusive scan of tsum
    uint32_t inc = tsum;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t wbase = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { uint32_t v = s_warp[w]; if (w < warp) wbase += v; btotal += v; }
    const uint32_t local_excl = wbase + inc - tsum;

    // decoupled look-back: publish this tile's aggregate, then walk the predecessors
    if (warp == 0) {
        uint32_t excl = 0;
        if (tile == 0) {
            if (lane == 0) atomicExch(&state[0], PA_FLAG_PREFIX | (unsigned long long)btotal);
        } else {
            if (lane == 0) atomicExch(&state[tile], PA_FLAG_AGG | (unsigned long long)btotal);
            long long idx = (long long)tile - 1;
            while (true) {
                long long my = idx - lane;
                unsigned long long s;
                if (my >= 0) {
                    do { s = *((volatile unsigned long long*)&state[my]); } while ((s >> 32) == 0ull);
                } else {
                    s = PA_FLAG_PREFIX;   // before tile 0: prefix 0
                }
                const unsigned pref = __ballot_sync(0xffffffffu, (s >> 32) == 2ull);
                uint32_t val = (uint32_t)s;
                if (pref) {
                    const int first = __ffs(pref) - 1;           // nearest predecessor holding a full prefix
                    val = lane <= first ? val : 0u;
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) val += __shfl_xor_sync(0xffffffffu, val, off);
                excl += val;
                if (pref) break;
                idx -= 32;
            }
            if (lane == 0) atomicExch(&state[tile], PA_FLAG_PREFIX | (unsigned long long)(excl + btotal));
        }
        if (lane == 0) {
            s_excl = excl;
            if ((int)tile == n_tiles - 1) {
                sc->R_new = excl + btotal;
                if (mail) { mail->R_new = excl + btotal; mail->W = sc->W; }     // single calls: straight into mapped host memory
            }
        }
    }
    __syncthreads();
    uint32_t o = s_excl + local_excl;
    if (j0 < R) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (j0 + q < R) {
                r_out[j0 + q] = r[q];
                o_out[j0 + q] = o;
                for (uint32_t c = 0; c < r[q]; ++c)
                    if ((long long)o + c < R_cap) parent[o + c] = (uint32_t)(j0 + q);
                o += r[q];
            }
        }
    }
}

int pa_launch_plan(pa_handle* h, int Emin) {
    const int n = (int)(((h->dev_R ? h->R_cap : h->R_cur) + PA_TILE - 1) / PA_TILE);
    PA_CUDA(h, pa_launch(h, pa_plan_kernel, dim3(n), dim3(256), 0, (const int32_t*)h->E, h->wtab_cur ? h->wtab_cur : (const double*)h->wtab,
                         h->d_scal, (long long)(h->dev_R ? -1 : h->R_cur), (double)h->R_target, h->dev_R ? PA_EMIN_DEV : Emin, h->keys, h->k,
                         (long long)h->R_cap, h->r, h->o, h->parent, h->scan_state, n, h->nlev, h->e0, h->mail_out));
    h->launches += 1;
    return PA_OK;
}

// ------------------------------------------------------------------------------------------------
// Small populations (at most PA_SMALL_TILES tiles of 1024, e.g. configs[0]): weights, W, tau, copy numbers, scan and parent map in
// ONE CTA and one launch.  The same arithmetic in the same order as pa_tree_kernel<0> + pa_plan_kernel -- per-tile TREE1024 trees,
// tile sums added in ascending order from 0.0, tau = (R w)/W with one multiply and one divide, the scan as plain integer
// sums -- but without the ticket, the fences and the look-back: what costs two launches of 6 us each on a launch-bound population
// (eight dependent trips to global memory) becomes one of about 4 us.
// ------------------------------------------------------------------------------------------------
#define PA_SMALL_TILES 4
__global__ void __launch_bounds__(PA_TILE)
pa_tree_plan_small_kernel(const int32_t* __restrict__ E, const double* __restrict__ wtab, PaScalars* sc,
                          long long R, double R_target, int Emin, PhiloxKeys K, uint32_t kcount, long long R_cap,
                          double* __restrict__ w_out, uint32_t* __restrict__ r_out, uint32_t* __restrict__ o_out,
                          uint32_t* __restrict__ parent, int n_tiles, int N, int e0, int commit, PaScalars* __restrict__ mail) {
    __shared__ double run[32];
    __shared__ double s_W;
    __shared__ uint32_t s_wsum[32];
    pa_pdl_wait(); pa_pdl_launch();
    R = pa_live_R(R, sc);
    Emin = pa_live_Emin(Emin, sc, N, e0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double wv[PA_SMALL_TILES];
    double total = 0.0;
#pragma unroll
    for (int t = 0; t < PA_SMALL_TILES; ++t) {
        wv[t] = 0.0;
        if (t < n_tiles) {
            const long long j = (long long)t * PA_TILE + tid;
            if (j < R) { wv[t] = wtab[(E[j] - Emin) >> 2]; if (w_out) w_out[j] = wv[t]; }
            double v = wv[t];
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));
            if (lane == 0) run[warp] = v;
            __syncthreads();
            if (warp == 0) {
                v = run[lane];
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) v = __dadd_rn(v, __shfl_down_sync(0xffffffffu, v, off));
                if (lane == 0) total = __dadd_rn(total, v);              // tile sums in ascending order (O5)
            }
            __syncthreads();
        }
    }
    if (tid == 0) { s_W = total; sc->W = total; }
    __syncthreads();
    const double W = s_W;
    uint32_t base = 0;
#pragma unroll
    for (int t = 0; t < PA_SMALL_TILES; ++t) {
        if (t < n_tiles) {
            const long long j = (long long)t * PA_TILE + tid;
            uint32_t r = 0;
            if (j < R) {
                const uint4 x = pa_philox((uint32_t)(j >> 2), 0u, kcount, PA_TAG_RESAMPLE, K);     // x(j,k), O1
                const uint32_t xq = (j & 3) == 0 ? x.x : (j & 3) == 1 ? x.y : (j & 3) == 2 ? x.z : x.w;
                const double tau = __ddiv_rn(__dmul_rn(R_target, wv[t]), W);
                const double n = floor(tau);
                const double f = __dsub_rn(tau, n);
                const double u = __dmul_rn((double)xq, 1.0 / 4294967296.0);
                r = (uint32_t)n + (u < f ? 1u : 0u);
            }
            uint32_t inc = r;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const uint32_t v = __shfl_up_sync(0xffffffffu, inc, off);
                if (lane >= off) inc += v;
            }
            if (lane == 31) s_wsum[warp] = inc;
            __syncthreads();
            uint32_t wbase = 0, btotal = 0;
#pragma unroll
            for (int w = 0; w < 32; ++w) { const uint32_t v = s_wsum[w]; if (w < warp) wbase += v; btotal += v; }
            uint32_t o = base + wbase + inc - r;
            if (j < R) {
                r_out[j] = r;
                o_out[j] = o;
                for (uint32_t c = 0; c < r; ++c)
                    if ((long long)o + c < R_cap) parent[o + c] = (uint32_t)j;
            }
            base += btotal;
            __syncthreads();
        }
    }
    if (tid == 0) {
        sc->R_new = base;
        if (mail) { mail->R_new = base; mail->W = W; }
        if (commit) {
            // pa_anneal with the copy fused into the sweep kernel's staging (pa_sweep_split_kernel<S, true>): what pa_copy_kernel's
            // first thread does there -- the new population size becomes current on the device (or the error flag is raised) and the
            // next measure launch's accumulators are cleared.  Every thread of this CTA has read R_dev / E_min long before.
            if (base >= 1u && (long long)base <= R_cap) sc->R_dev = base; else sc->err = 1u;
            sc->mmin_inv = 0u; sc->mmax = 0u; sc->done_counter = 0u; sc->pad0 = 0u;
            sc->SE = 0; sc->SE2 = 0; sc->SA = 0; sc->SM2 = 0; sc->m4sum = 0.0;
        }
    }
}

// a population of at most PA_SMALL_TILES tiles takes the fused kernel (PA_SMALL_PLAN=0: never)
bool pa_small_plan_ok(const pa_handle* h) {
    const int n = (int)(((h->dev_R ? h->R_cap : h->R_cur) + PA_TILE - 1) / PA_TILE);
    return n <= PA_SMALL_TILES && pa_sw(h, PA_SW_SMALL_PLAN, 1) != 0;
}

// weights + W, then the plan: two launches, or the fused kernel for a small population.  commit (pa_anneal, small populations
// only): the kernel also makes R_new the device's current population size, as the copy kernel would.
int pa_launch_weights_plan(pa_handle* h, int Emin, double* w_out, bool commit) {
    const int n = (int)(((h->dev_R ? h->R_cap : h->R_cur) + PA_TILE - 1) / PA_TILE);
    if (!pa_small_plan_ok(h)) {
        if (commit) return PA_ERR_INVALID_ARG;
        const int rc = pa_launch_weights(h, Emin, w_out);
        return rc != PA_OK ? rc : pa_launch_plan(h, Emin);
    }
    PA_CUDA(h, pa_launch(h, pa_tree_plan_small_kernel, dim3(1), dim3(PA_TILE), 0, (const int32_t*)h->E,
                         h->wtab_cur ? h->wtab_cur : (const double*)h->wtab, h->d_scal, (long long)(h->dev_R ? -1 : h->R_cur),
                         (double)h->R_target, h->dev_R ? PA_EMIN_DEV : Emin, h->keys, h->k, (long long)h->R_cap, w_out,
                         h->r, h->o, h->parent, n, h->nlev, h->e0, commit ? 1 : 0, h->mail_out));
    h->launches += 1;
    if (commit) h->scal_zeroed = true;
    return PA_OK;
}

// ------------------------------------------------------------------------------------------------
// Copy (L165-L171 resampleKer; O7): new[d] = old[parent(d)].  The parents of the 32 slots of a
// destination group are non-decreasing, so lane d reads global source bit parent(d) = s_d + d with an
// offset s_d = parent(d) - d that changes only where a copy number differs from 1.  All lanes with the
// same offset are served by one funnel shift of the two neighbouring source words (a 32-bit window at
// bit s of the concatenated source groups) and one mask: a destination word costs two instructions per
// DISTINCT offset, however the lanes interleave.  One warp builds the (shift, mask) classes of the
// group with __match_any_sync, sorted by offset and grouped into source windows so that every source
// word is loaded once; all threads then stream the group's N words with 128-bit loads and stores.
// ------------------------------------------------------------------------------------------------
struct __align__(8) PaSeg { uint32_t shift, mask; };              // one offset class: dst |= (window >> shift) & mask
struct __align__(16) PaWin {                                      // one source window = two neighbouring source groups
    uint32_t lo_g, hi_g;     // group indices of the low / high word, clamped into the buffer (a clamped word is never selected)
    int seg_end;             // classes [previous seg_end, seg_end) read this window
    int consecutive;         // the low word is the previous window's high word
};

// NCH chunks of 4 words per thread and pass: the class list is walked once for NCH chunks, and NCH x 2 loads are in flight.
template <int NCH>
__device__ __forceinline__ void pa_copy_chunks(const uint4* __restrict__ src4, uint4* __restrict__ out, const PaWin* wins, int nw,
                                               const PaSeg* segs, int chunks, int i, int stride) {
    uint4 acc[NCH], lo[NCH], hi[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) { acc[c] = make_uint4(0, 0, 0, 0); lo[c] = acc[c]; hi[c] = acc[c]; }
    int k = 0;
    for (int w = 0; w < nw; ++w) {
        const PaWin W = wins[w];
        const uint4* plo = src4 + (size_t)W.lo_g * chunks + i;
        const uint4* phi = src4 + (size_t)W.hi_g * chunks + i;
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            if (W.consecutive) lo[c] = hi[c]; else lo[c] = __ldg(plo + c * stride);
            hi[c] = __ldg(phi + c * stride);
        }
        for (; k < W.seg_end; ++k) {
            const PaSeg e = segs[k];
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                acc[c].x |= __funnelshift_r(lo[c].x, hi[c].x, e.shift) & e.mask;
                acc[c].y |= __funnelshift_r(lo[c].y, hi[c].y, e.shift) & e.mask;
                acc[c].z |= __funnelshift_r(lo[c].z, hi[c].z, e.shift) & e.mask;
                acc[c].w |= __funnelshift_r(lo[c].w, hi[c].w, e.shift) & e.mask;
            }
        }
    }
#pragma unroll
    for (int c = 0; c < NCH; ++c) out[i + c * stride] = acc[c];
}

#ifndef PA_COPY_MINB
#define PA_COPY_MINB 8
#endif
#ifndef PA_COPY_NCH
#define PA_COPY_NCH 4
#endif
__global__ void __launch_bounds__(128, PA_COPY_MINB)
pa_copy_kernel(const uint32_t* __restrict__ src, uint32_t* __restrict__ dst, const uint32_t* __restrict__ parent,
               PaScalars* sc, long long R_cap, int N, int commit) {
    __shared__ PaSeg segs[32];
    __shared__ PaWin wins[32];
    __shared__ int sq[32];
    __shared__ int nwin;
    const long long g = blockIdx.x;
    const int tid = threadIdx.x;
    pa_pdl_wait(); pa_pdl_launch();
    // R_new is read on the device: the launch does not wait for the host to see it, the grid covers the
    // capacity and groups past the new population exit.  R_new > R_cap is the PA_ERR_CAPACITY case: nothing
    // of the live population is touched (dst is the spare buffer) and the host discards the copy.
    if (commit && blockIdx.x == 0 && blockIdx.y == 0 && tid == 0) {
        // pa_anneal: the resampled population becomes the current one on the device (the host does the same bookkeeping later
        // from the per-step snapshots; outside [1, R_cap] the size is left alone and the error flag is raised), and the
        // accumulators of the next measure launch are cleared here instead of by a memset of their own.  No CTA of this
        // kernel reads R_dev or the measure block.
        const long long Rn = sc->R_new;
        if (Rn >= 1 && Rn <= R_cap) sc->R_dev = (uint32_t)Rn; else sc->err = 1u;
        sc->mmin_inv = 0u; sc->mmax = 0u; sc->done_counter = 0u; sc->pad0 = 0u;
        sc->SE = 0; sc->SE2 = 0; sc->SA = 0; sc->SM2 = 0; sc->m4sum = 0.0;
    }
    const long long R_new = min((long long)sc->R_new, R_cap);
    if (g * 32 >= R_new) return;
    if (tid < 32) {
        const long long d = g * 32 + tid;
        const bool valid = d < R_new;
        // offset of this lane; invalid lanes get private keys that sort last and carry no class
        const long long s = valid ? (long long)parent[d] - tid : (1ll << 40) + tid;
        const unsigned same = __match_any_sync(0xffffffffu, (unsigned long long)s);
        const bool leader = valid && (__ffs(same) - 1) == tid;
        const unsigned leaders = __ballot_sync(0xffffffffu, leader);
        int rank = 0;
        for (int l = 0; l < 32; ++l) {
            const long long sl = __shfl_sync(0xffffffffu, s, l);
            rank += (int)(((leaders >> l) & 1u) != 0u && sl < s);
        }
        if (leader) {
            PaSeg e;
            e.shift = (uint32_t)(s & 31);
            e.mask = same;
            segs[rank] = e;
            sq[rank] = (int)(s >> 5);               // arithmetic shift: floor, s may be negative (down to -31)
        }
        __syncwarp();
        // classes are sorted by offset, hence by source window q; consecutive classes with the same q share the loads
        const int ns = __popc(leaders);
        const long long Gmax = (R_cap + 31) >> 5;
        const int q = tid < ns ? sq[tid] : 0;
        const bool wstart = tid < ns && (tid == 0 || q != sq[tid - 1]);
        const unsigned wstarts = __ballot_sync(0xffffffffu, wstart);
        if (wstart) {
            const unsigned later = tid == 31 ? 0u : wstarts & ~((2u << tid) - 1u);
            PaWin W;
            const long long ql = q, qh = (long long)q + 1;
            W.lo_g = (uint32_t)(ql < 0 ? 0 : (ql >= Gmax ? Gmax - 1 : ql));
            W.hi_g = (uint32_t)(qh < 0 ? 0 : (qh >= Gmax ? Gmax - 1 : qh));
            W.seg_end = later ? (__ffs(later) - 1) : ns;
            W.consecutive = (tid > 0 && q == sq[tid - 1] + 1) ? 1 : 0;
            wins[__popc(wstarts & ((1u << tid) - 1u))] = W;
        }
        if (tid == 0) nwin = __popc(wstarts);
    }
    __syncthreads();
    const int nw = nwin;
    const int chunks = N >> 2;
    const uint4* src4 = reinterpret_cast<const uint4*>(src);
    uint4* out = reinterpret_cast<uint4*>(dst + g * (long long)N);
    const int stride = gridDim.y * blockDim.x;
    int i = blockIdx.y * blockDim.x + tid;
    for (; i + (PA_COPY_NCH - 1) * stride < chunks; i += PA_COPY_NCH * stride) pa_copy_chunks<PA_COPY_NCH>(src4, out, wins, nw, segs, chunks, i, stride);
    for (; i + stride < chunks; i += 2 * stride) pa_copy_chunks<2>(src4, out, wins, nw, segs, chunks, i, stride);
    if (i < chunks) pa_copy_chunks<1>(src4, out, wins, nw, segs, chunks, i, stride);
}

int pa_launch_copy(pa_handle* h) {
    const int64_t G = h->G_cap;
    const int chunks = h->N / 4;
    int gy = 1;
    // small populations: split a group's words over several CTAs to fill the GPU
    while (G * gy < 4 * h->n_sm && gy * 128 * 2 <= chunks) gy *= 2;
    dim3 grid((unsigned)G, (unsigned)gy, 1);
    PA_CUDA(h, pa_launch(h, pa_copy_kernel, grid, dim3(128), 0, (const uint32_t*)h->spins[h->cur], h->spins[1 - h->cur],
                         (const uint32_t*)h->parent, h->d_scal, (long long)h->R_cap, h->N, h->dev_R ? 1 : 0));
    h->scal_zeroed = h->dev_R;
    h->launches += 1;
    return PA_OK;
}
