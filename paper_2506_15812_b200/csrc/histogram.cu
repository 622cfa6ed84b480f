// a5: binning + Faraday-cup histogram (PAPER.md L330 segment geometry with optional non-uniform
// size and gaps; L344-350 segment ID or error indicator per ion, atomically summed counters;
// L352 only the compact counter array goes back to the host).
//
// One thread per ion.  Segment search: uniform-pitch guess verified against the real edges
// (half-open [lo,hi), reading A11), binary search otherwise.  Counting: block-private shared
// histogram flushed once when the whole matrix fits (<= 8192 counters), else warp-aggregated
// global atomics (__match_any_sync: one atomic per distinct counter per warp).
#include "taiga_internal.h"

#define HIST_SMEM_BINS 8192
#define TG_GRAZE 1e-9

struct HistParams {
    const double *hit_u, *hit_w;
    int32_t* cell;
    uint8_t* flags;
    const unsigned short* group;
    unsigned long long n;
    const double *u_lo, *u_hi, *w_lo, *w_hi;
    int nu, nw, n_hist;
    double inv_pu, inv_pw;            // 1/pitch when the axis is uniform with zero gaps, else 0
    unsigned long long *counts, *summary;
};

// index of the segment containing v, or -1; sets `graze` when v is within 1e-9 of an edge
__device__ __forceinline__ int find_segment(const double* __restrict__ lo, const double* __restrict__ hi, int n,
                                            double inv_pitch, double v, bool& graze) {
    int k;
    if (inv_pitch > 0.0) {                      // guess, then verify against the stored edges
        double g = floor((v - __ldg(lo)) * inv_pitch);
        k = (g < 0.0) ? -1 : (g >= (double)n ? n - 1 : (int)g);
        while (k >= 0 && v < __ldg(lo + k)) --k;
        while (k + 1 < n && v >= __ldg(lo + k + 1)) ++k;
    } else {                                    // last k with lo[k] <= v
        int a = -1, b = n;
        while (b - a > 1) { int m = (a + b) >> 1; if (__ldg(lo + m) <= v) a = m; else b = m; }
        k = a;
    }
    // nearest edges: lo[k], hi[k], lo[k+1] (segments are ordered and non-overlapping)
    if (k >= 0 && (fabs(v - __ldg(lo + k)) < TG_GRAZE || fabs(v - __ldg(hi + k)) < TG_GRAZE)) graze = true;
    if (k + 1 < n && fabs(v - __ldg(lo + k + 1)) < TG_GRAZE) graze = true;
    return (k >= 0 && v < __ldg(hi + k)) ? k : -1;
}

template <bool SMEM>
__global__ void __launch_bounds__(256) k_histogram(HistParams P) {
    __shared__ unsigned int sh[SMEM ? HIST_SMEM_BINS : 1];
    const int nbins = P.n_hist * P.nw * P.nu;
    if (SMEM) {
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) sh[b] = 0u;
        __syncthreads();
    }
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    int g = 0, cat = -1, bin = -1;
    bool flagged = false;
    if (i < P.n) {
        g = P.group ? (int)P.group[i] : 0;
        if (g < P.n_hist) {
            int st = P.cell[i];
            uint8_t fl = P.flags[i];
            if (st >= TAIGA_CELL_MISS) {        // crossed the plane
                bool gz = false;
                int iu = find_segment(P.u_lo, P.u_hi, P.nu, P.inv_pu, P.hit_u[i], gz);
                int iw = find_segment(P.w_lo, P.w_hi, P.nw, P.inv_pw, P.hit_w[i], gz);
                if (gz) { fl |= TAIGA_FLAG_EDGE; P.flags[i] = fl; }
                if (iu >= 0 && iw >= 0) { int c = iw * P.nu + iu; P.cell[i] = c; bin = (g * P.nw + iw) * P.nu + iu; cat = 0; }
                else { P.cell[i] = TAIGA_CELL_MISS; cat = 1; }
            } else cat = (st == TAIGA_CELL_MAXSTEPS) ? 2 : (st == TAIGA_CELL_OUT ? 3 : 4);
            flagged = fl != 0;
        }
    }
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    // per-segment counters
    if (SMEM) {
        if (bin >= 0) atomicAdd(&sh[bin], 1u);
    } else {
        unsigned m = __match_any_sync(FULL, bin);
        if (bin >= 0 && lane == __ffs(m) - 1) atomicAdd(&P.counts[bin], (unsigned long long)__popc(m));
    }
    // summary counters {hit, miss, maxsteps, out, badstart, flagged} per histogram
    int key = (cat >= 0) ? g * 8 + cat : -1;
    unsigned m1 = __match_any_sync(FULL, key);
    if (key >= 0 && lane == __ffs(m1) - 1) atomicAdd(&P.summary[(size_t)g * 6 + cat], (unsigned long long)__popc(m1));
    int key2 = (flagged && cat >= 0) ? g : -1;
    unsigned m2 = __match_any_sync(FULL, key2);
    if (key2 >= 0 && lane == __ffs(m2) - 1) atomicAdd(&P.summary[(size_t)g * 6 + 5], (unsigned long long)__popc(m2));
    if (SMEM) {
        __syncthreads();
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) {
            unsigned v = sh[b];
            if (v) atomicAdd(&P.counts[b], (unsigned long long)v);
        }
    }
}

static double uniform_inv_pitch(const double* lo, const double* hi, int n) {
    double pitch = hi[0] - lo[0];
    for (int k = 0; k < n; ++k) {
        if (fabs((hi[k] - lo[k]) - pitch) > 1e-12 * fabs(pitch)) return 0.0;
        if (k + 1 < n && hi[k] != lo[k + 1]) return 0.0;
    }
    return 1.0 / pitch;
}

int tg_histogram(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                 unsigned long long* counts, unsigned long long* summary) {
    size_t ne = 2 * ((size_t)det->nu + det->nw), cap = ctx->cap_edges;
    int rc = tg_reserve(ctx, &ctx->edges, &cap, ne);
    ctx->cap_edges = (int)cap;
    if (rc) return rc;
    cudaStream_t st = ctx->stream;
    double* e = ctx->edges;
    {   // edges staged through the context's pinned buffer: the caller's arrays are read during the call only
        rc = tg_stage(ctx, ne * sizeof(double));
        if (rc) return rc;
        double* h = (double*)ctx->stage;
        memcpy(h, det->u_lo, det->nu * sizeof(double)); memcpy(h + det->nu, det->u_hi, det->nu * sizeof(double));
        memcpy(h + 2 * det->nu, det->w_lo, det->nw * sizeof(double)); memcpy(h + 2 * det->nu + det->nw, det->w_hi, det->nw * sizeof(double));
        TG_CUDA(ctx, cudaMemcpyAsync(e, h, ne * sizeof(double), cudaMemcpyHostToDevice, st));
        TG_CUDA(ctx, cudaEventRecord(ctx->stage_done, st));
    }
    HistParams P;
    P.hit_u = ions->hit_u; P.hit_w = ions->hit_w; P.cell = ions->cell; P.flags = ions->flags; P.group = ions->group;
    P.n = ions->n;
    P.u_lo = e; P.u_hi = e + det->nu; P.w_lo = e + 2 * det->nu; P.w_hi = e + 2 * det->nu + det->nw;
    P.nu = det->nu; P.nw = det->nw; P.n_hist = n_hist;
    P.inv_pu = uniform_inv_pitch(det->u_lo, det->u_hi, det->nu);
    P.inv_pw = uniform_inv_pitch(det->w_lo, det->w_hi, det->nw);
    P.counts = counts; P.summary = summary;
    unsigned blocks = (unsigned)((ions->n + 255) / 256);
    if ((long long)n_hist * det->nw * det->nu <= HIST_SMEM_BINS) k_histogram<true><<<blocks, 256, 0, st>>>(P);
    else k_histogram<false><<<blocks, 256, 0, st>>>(P);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}

// ------------------------------------------------------------------------------------------
// Weighted counters: q = floor(w 2^32 + 1/2) per plane-crossing ion, 64-bit
// integer atomics, so the sums do not depend on the order of accumulation.
// Per-segment sums: block-private shared counters flushed once when the matrix fits (<= 4096 x 8 B), else one global
// atomic per ion (distinct addresses for the most part).  The four summary sums of a histogram, which every crossing ion
// of the grid used to add to the same three addresses, are reduced over the warp first when its ions belong to one
// histogram (the rule: groups are contiguous runs of ions), so a warp issues at most four atomics on them.
#define WHIST_SMEM_BINS 4096

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool SMEM>
__global__ void __launch_bounds__(256) k_histogram_weighted(const int32_t* __restrict__ cell, const double* __restrict__ weight,
                                                            const uint16_t* __restrict__ group, uint32_t n, int n_hist, int ncell,
                                                            unsigned long long* __restrict__ wcounts, unsigned long long* __restrict__ wsummary) {
    __shared__ unsigned long long sh[SMEM ? WHIST_SMEM_BINS : 1];
    const int nbins = n_hist * ncell;
    if (SMEM) {
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) sh[b] = 0ull;
        __syncthreads();
    }
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    int g = -1, c = TAIGA_CELL_MISS;
    unsigned long long q = 0ull;
    if (i < n) {
        const int gi = group ? (int)group[i] : 0;
        c = cell[i];
        if (gi < n_hist && c >= TAIGA_CELL_MISS) {
            g = gi;
            double wv = weight[i];
            if (!(wv >= 0.0)) wv = 0.0;                // negative / NaN weights count as 0
            if (wv > 1048576.0) wv = 1048576.0;        // keeps q < 2^52 (weights are <= 1 for this method)
            q = (unsigned long long)floor(fma(wv, 4294967296.0, 0.5));
        }
    }
    const bool crosser = g >= 0;
    if (crosser && c >= 0) {
        if (SMEM) atomicAdd(&sh[g * ncell + c], q);
        else atomicAdd(&wcounts[(size_t)g * ncell + c], q);
    }
    const unsigned long long q_in = (crosser && c >= 0) ? q : 0ull, q_out = (crosser && c < 0) ? q : 0ull;
    const unsigned long long q2 = crosser ? (__umul64hi(q, q) << 32 | (q * q) >> 32) : 0ull;
    const unsigned FULL = 0xffffffffu;
    const unsigned act = __ballot_sync(FULL, crosser);
    const int gmin = __reduce_min_sync(FULL, crosser ? g : 0x7fffffff), gmax = __reduce_max_sync(FULL, crosser ? g : -1);
    if (act && gmin == gmax) {                         // one histogram in this warp: reduce, then four atomics
        const unsigned long long s_in = warp_sum_u64(q_in), s_out = warp_sum_u64(q_out), s2 = warp_sum_u64(q2);
        if ((threadIdx.x & 31) == 0) {
            unsigned long long* ws = wsummary + (size_t)gmin * 4;
            if (s_in) atomicAdd(ws + 0, s_in);
            if (s_out) atomicAdd(ws + 1, s_out);
            if (s2) atomicAdd(ws + 2, s2);
            atomicAdd(ws + 3, (unsigned long long)__popc(act));
        }
    } else if (crosser) {                              // a warp across a group border, or interleaved groups
        unsigned long long* ws = wsummary + (size_t)g * 4;
        atomicAdd(ws + (c >= 0 ? 0 : 1), q);
        atomicAdd(ws + 2, q2);
        atomicAdd(ws + 3, 1ull);
    }
    if (SMEM) {
        __syncthreads();
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) {
            const unsigned long long v = sh[b];
            if (v) atomicAdd(&wcounts[b], v);
        }
    }
}

int tg_histogram_weighted(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                          unsigned long long* wcounts, unsigned long long* wsummary) {
    const uint32_t n = (uint32_t)ions->n;
    const int ncell = det->nu * det->nw;
    const double* wt = ions->weight ? ions->weight : ions->w0;
    if ((long long)n_hist * ncell <= WHIST_SMEM_BINS)
        k_histogram_weighted<true><<<(n + 255) / 256, 256, 0, ctx->stream>>>(ions->cell, wt, ions->group, n, n_hist, ncell, wcounts, wsummary);
    else
        k_histogram_weighted<false><<<(n + 255) / 256, 256, 0, ctx->stream>>>(ions->cell, wt, ions->group, n, n_hist, ncell, wcounts, wsummary);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}

// ------------------------------------------------------------------------------------------
// taiga_detector_histogram_static (include/taiga.h): k_histogram again, for callers that must not allocate.
//
// tg_histogram above keeps its device copy of the segment edges in ctx->edges (cudaMalloc on the first call and
// whenever a larger detector comes along) and stages the host arrays through ctx->stage (cudaMallocHost).  A caller
// that runs the binning inside a loop it has promised to keep free of allocations -- a between-shot evaluation that
// shares the GPU with other streams (cudaMalloc / cudaFree stall every stream of the device), or a process whose
// memory pool has already taken the device's memory, where a late cudaMalloc simply fails -- cannot use that.
// Here the edge copy lives in the fixed array below, part of the library image: every GPU that loads libtaiga.so
// holds these 32 KB until the process exits, whether or not this entry point is ever called.
#define TG_STATIC_EDGE_DOUBLES 4096                       // 2 (nu + nw) doubles: nu + nw <= TAIGA_STATIC_MAX_SEGMENTS = 2048
#define TG_STATIC_MAX_DEVICES 64
static __device__ __align__(256) double g_static_edges[TG_STATIC_EDGE_DOUBLES];
// Device address of g_static_edges per CUDA ordinal.  In host code `g_static_edges` is only a handle for the symbol
// API, not an address a kernel may be given; the address is asked for once per device, with that device current.
static double* g_static_edges_dev[TG_STATIC_MAX_DEVICES];

int tg_histogram_static(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                        unsigned long long* counts, unsigned long long* summary) {
    const size_t nu = (size_t)det->nu, nw = (size_t)det->nw, ne = 2 * (nu + nw);
    if (ne > TG_STATIC_EDGE_DOUBLES) {
        TG_SET_ERR(ctx, "histogram_static: nu + nw = %zu segments exceed the fixed edge table (TAIGA_STATIC_MAX_SEGMENTS = %d); "
                        "use taiga_detector_histogram, which allocates", nu + nw, TG_STATIC_EDGE_DOUBLES / 2);
        return TAIGA_E_ARG;
    }
    if (ctx->device < 0 || ctx->device >= TG_STATIC_MAX_DEVICES) {
        TG_SET_ERR(ctx, "histogram_static: device ordinal %d outside [0, %d)", ctx->device, TG_STATIC_MAX_DEVICES);
        return TAIGA_E_ARG;
    }
    double* e = g_static_edges_dev[ctx->device];
    if (!e) {          // first call on this device (the caller has made ctx->device current): resolve the symbol
        TG_CUDA(ctx, cudaGetSymbolAddress((void**)&e, g_static_edges));
        g_static_edges_dev[ctx->device] = e;           // every thread that gets here stores the same value
    }
    cudaStream_t st = ctx->stream;
    // Straight from the caller's arrays, in stream order behind earlier users of the table on this stream; the runtime
    // has read a pageable source by the time each call returns.  Every entry the kernel reads is rewritten here, so
    // nothing in the array has to start at zero and the previous call's contents do not matter.
    TG_CUDA(ctx, cudaMemcpyAsync(e, det->u_lo, nu * sizeof(double), cudaMemcpyHostToDevice, st));
    TG_CUDA(ctx, cudaMemcpyAsync(e + nu, det->u_hi, nu * sizeof(double), cudaMemcpyHostToDevice, st));
    TG_CUDA(ctx, cudaMemcpyAsync(e + 2 * nu, det->w_lo, nw * sizeof(double), cudaMemcpyHostToDevice, st));
    TG_CUDA(ctx, cudaMemcpyAsync(e + 2 * nu + nw, det->w_hi, nw * sizeof(double), cudaMemcpyHostToDevice, st));
    HistParams P;
    P.hit_u = ions->hit_u; P.hit_w = ions->hit_w; P.cell = ions->cell; P.flags = ions->flags; P.group = ions->group;
    P.n = ions->n;
    P.u_lo = e; P.u_hi = e + nu; P.w_lo = e + 2 * nu; P.w_hi = e + 2 * nu + nw;
    P.nu = det->nu; P.nw = det->nw; P.n_hist = n_hist;
    P.inv_pu = uniform_inv_pitch(det->u_lo, det->u_hi, det->nu);
    P.inv_pw = uniform_inv_pitch(det->w_lo, det->w_hi, det->nw);
    P.counts = counts; P.summary = summary;
    unsigned blocks = (unsigned)((ions->n + 255) / 256);
    if ((long long)n_hist * det->nw * det->nu <= HIST_SMEM_BINS) k_histogram<true><<<blocks, 256, 0, st>>>(P);
    else k_histogram<false><<<blocks, 256, 0, st>>>(P);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}
