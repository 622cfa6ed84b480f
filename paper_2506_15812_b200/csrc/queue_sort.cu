// Ordering of the ion queue for taiga_trace (a3): counting sort by birth cell.
#include "taiga_internal.h"

// ------------------------------------------------------------------------------------------
// Ordering of the ion queue: counting sort by birth cell (R-major, so that deep-born = long
// running ions are dequeued first and the ions sharing a warp fly through the same cells);
// time-sliced and (R,Z,phi) fields: key = (radial band, slice / toroidal sub-cell, R bin, Z bin).
// Output is written by ion index, so the order never shows in the results.
#define SORT_NBR 512
#define SORT_NBZ 256
#define SORT_BAND 64                   // fine R bins per radial band (8 bands)
#define SCAN_ITEMS 8
#define SCAN_TPB 1024

struct SortParams {
    const double *x, *y, *z, *t0;
    uint32_t n;
    double Rmin, Zmin, minwR, minwZ, s0, inv_ds;
    int n_major, nS, kind;
    unsigned long long* bbox;          // [4]: min a, max a, min b, max b (bit patterns of doubles >= 0)
};

__device__ __forceinline__ void sort_ab(const SortParams& S, uint32_t i, double& a, double& b) {
    double X = S.x[i], Y = S.y[i];
    a = fmax(sqrt(fma(X, X, Y * Y)) - S.Rmin, 0.0);
    b = fmax(S.z[i] - S.Zmin, 0.0);
    if (!(a < 1e30)) a = 0.0;          // NaN / inf guards
    if (!(b < 1e30)) b = 0.0;
}

__global__ void k_sort_bbox(SortParams S) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    double a = 0, b = 0;
    bool v = i < S.n;
    if (v) sort_ab(S, i, a, b);
    unsigned long long amin = v ? (unsigned long long)__double_as_longlong(a) : ~0ull, amax = v ? (unsigned long long)__double_as_longlong(a) : 0ull;
    unsigned long long bmin = v ? (unsigned long long)__double_as_longlong(b) : ~0ull, bmax = v ? (unsigned long long)__double_as_longlong(b) : 0ull;
    for (int o = 16; o > 0; o >>= 1) {
        amin = min(amin, __shfl_xor_sync(0xffffffffu, amin, o)); amax = max(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        bmin = min(bmin, __shfl_xor_sync(0xffffffffu, bmin, o)); bmax = max(bmax, __shfl_xor_sync(0xffffffffu, bmax, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&S.bbox[0], amin); atomicMax(&S.bbox[1], amax);
        atomicMin(&S.bbox[2], bmin); atomicMax(&S.bbox[3], bmax);
    }
}

__device__ __forceinline__ uint32_t sort_key(const SortParams& S, uint32_t i) {
    double a, b;
    sort_ab(S, i, a, b);
    double a0 = __longlong_as_double((long long)S.bbox[0]), a1 = __longlong_as_double((long long)S.bbox[1]);
    double b0 = __longlong_as_double((long long)S.bbox[2]), b1 = __longlong_as_double((long long)S.bbox[3]);
    double wR = fmax((a1 - a0) / SORT_NBR, S.minwR), wZ = fmax((b1 - b0) / SORT_NBZ, S.minwZ);
    int bR = min(max((int)((a - a0) / wR), 0), SORT_NBR - 1), bZ = min(max((int)((b - b0) / wZ), 0), SORT_NBZ - 1);
    int m = 0;
    if (S.n_major > 1 && S.kind == 1) {             // time slices: major key = slice of birth
        int k = min(max((int)floor((S.t0[i] - S.s0) * S.inv_ds), 0), S.nS - 1);
        m = (int)(((long long)k * S.n_major) / S.nS);
    } else if (S.n_major > 1) {                     // phi planes: major key = toroidal (sub-)cell of birth
        double xs = (atan2(S.y[i], S.x[i]) - S.s0) * S.inv_ds;
        xs -= (double)S.nS * floor(xs / (double)S.nS);
        m = min(max((int)(xs * (double)S.n_major / (double)S.nS), 0), S.n_major - 1);
    }
    // radial band (SORT_BAND fine bins) first, then the slice / toroidal sub-cell, then the fine bins: every slice's deep-born
    // (trapped, step-limit) ions are dequeued at the head of the queue instead of at the head of their slice's section,
    // where the late slices' tiles outlived the rest of the kernel by 14 % (BASELINE config 4, profiles/r2_experiments.md)
    const int band = bR / SORT_BAND, fine = bR % SORT_BAND;
    return (uint32_t)(((band * S.n_major + m) * SORT_BAND + fine) * SORT_NBZ + bZ);
}

__global__ void k_sort_count(SortParams S, uint32_t* bins) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < S.n) atomicAdd(&bins[sort_key(S, i)], 1u);
}

// exclusive scan of `bins` in blocks of SCAN_TPB*SCAN_ITEMS; block totals to sums[]
__global__ void __launch_bounds__(SCAN_TPB) k_scan_blocks(uint32_t* bins, uint32_t nb, uint32_t* sums) {
    __shared__ uint32_t wsum[32];
    uint32_t base = (blockIdx.x * SCAN_TPB + threadIdx.x) * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], tot = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < nb) ? bins[base + k] : 0u; tot += v[k]; }
    uint32_t inc = tot;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t u = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += u; }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = wsum[lane], si = s;
        for (int o = 1; o < 32; o <<= 1) { uint32_t u = __shfl_up_sync(0xffffffffu, si, o); if (lane >= o) si += u; }
        wsum[lane] = si - s;
        if (lane == 31 && sums) sums[blockIdx.x] = si;
    }
    __syncthreads();
    uint32_t run = wsum[w] + inc - tot;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < nb) bins[base + k] = run; run += v[k]; }
}

__global__ void k_sort_scatter(SortParams S, uint32_t* bins, const uint32_t* sums, uint32_t* order) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S.n) return;
    uint32_t key = sort_key(S, i);
    uint32_t pos = atomicAdd(&bins[key], 1u) + sums[key / (SCAN_TPB * SCAN_ITEMS)];
    order[pos] = i;
}

int tg_build_order(taiga_ctx* ctx, const taiga_ions* ions) {
    const FieldDev& f = ctx->field;
    uint32_t n = (uint32_t)ions->n;
    int n_major = (f.kind == 1 && ions->t0) ? (f.nS < 64 ? f.nS : 64) : (f.kind == 2 ? 64 : 1);
    uint32_t nb = (uint32_t)n_major * SORT_NBR * SORT_NBZ;
    uint32_t nblk = (nb + SCAN_TPB * SCAN_ITEMS - 1) / (SCAN_TPB * SCAN_ITEMS);   // <= 1024
    int rc = tg_reserve(ctx, &ctx->order, &ctx->cap_order, (size_t)n);
    if (rc) return rc;
    rc = tg_reserve(ctx, &ctx->bins, &ctx->cap_bins, (size_t)nb + 2 * SCAN_TPB * SCAN_ITEMS);
    if (rc) return rc;
    uint32_t* sums = ctx->bins + nb;                 // nblk entries (+ padding for the second scan)
    cudaStream_t st = ctx->stream;
    TG_CUDA(ctx, cudaMemsetAsync(ctx->bins, 0, ((size_t)nb + 2 * SCAN_TPB * SCAN_ITEMS) * sizeof(uint32_t), st));
    unsigned long long init[4] = {~0ull, 0ull, ~0ull, 0ull};
    TG_CUDA(ctx, cudaMemcpyAsync(ctx->counters + 8, init, sizeof(init), cudaMemcpyHostToDevice, st));
    SortParams S;
    S.x = ions->x; S.y = ions->y; S.z = ions->z; S.t0 = ions->t0; S.n = n;
    S.Rmin = f.Rmin; S.Zmin = f.Zmin;
    int sub = ctx->opt_sort_sub > 0 ? ctx->opt_sort_sub : 4;
    S.minwR = 1.0 / (f.inv_hR * sub); S.minwZ = 1.0 / (f.inv_hZ * sub);
    S.s0 = f.s0; S.inv_ds = f.inv_ds; S.n_major = n_major; S.nS = f.nS; S.kind = f.kind;
    S.bbox = ctx->counters + 8;
    unsigned gb = (n + 255) / 256;
    k_sort_bbox<<<gb, 256, 0, st>>>(S);
    k_sort_count<<<gb, 256, 0, st>>>(S, ctx->bins);
    k_scan_blocks<<<nblk, SCAN_TPB, 0, st>>>(ctx->bins, nb, sums);
    k_scan_blocks<<<1, SCAN_TPB, 0, st>>>(sums, nblk, nullptr);
    k_sort_scatter<<<gb, 256, 0, st>>>(S, ctx->bins, sums, ctx->order);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}

