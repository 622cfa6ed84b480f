// Roofline denominator: register-resident DFMA microkernel (MEASURED_PEAKS.json
// has no FP64 entry, so the FP64 issue rate is measured in the same run as the benchmark).
#include "taiga_internal.h"

// Four independent chains per thread, each with its own multiplicand register and one shared addend: measures
// 0.98-0.99 of 148 x 64 DFMA/clk at 8-32 warps per SM (profiles/r2a_microbench.md).  Two other forms fall short of the
// issue limit and are NOT the roofline: eight chains sharing both operands (the round-1 kernel: 0.91, register-bank
// conflicts on the shared pair) and chains with three distinct source registers (0.67: a DFMA reading three different
// 64-bit registers is limited by register-file bandwidth).
#define PEAK_CHAINS 4
#define PEAK_INNER 64

__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters, double a0, double b) {
    double v[PEAK_CHAINS], a[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) { v[c] = (double)(threadIdx.x + c) * 1e-3; a[c] = a0 + c * 1e-9; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < PEAK_INNER; ++k) {
#pragma unroll
            for (int c = 0; c < PEAK_CHAINS; ++c) v[c] = fma(v[c], a[c], b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) s += v[c];
    if (s == 123.456) out[0] = s;               // keeps the chains alive, never true in practice
}

int tg_fp64_peak(taiga_ctx* ctx, double ms, double* rate) {
    cudaStream_t st = ctx->stream;
    cudaEvent_t e0, e1;
    TG_CUDA(ctx, cudaEventCreate(&e0));
    TG_CUDA(ctx, cudaEventCreate(&e1));
    double* dummy = (double*)ctx->counters + 12;
    unsigned grid = (unsigned)ctx->sm_count * 4;      // 4 x 256 threads = 32 warps per SM
    int iters = 256;
    float t = 0.f;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, st);
        k_dfma_peak<<<grid, 256, 0, st>>>(dummy, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); TG_CUDA(ctx, e); }
        cudaEventElapsedTime(&t, e0, e1);
        double n = (double)grid * 256.0 * (double)iters * PEAK_INNER * PEAK_CHAINS;
        if (rep >= 2) { double r = n / (t * 1e-3); if (r > best) best = r; }
        if (rep == 1 && t > 0.f) { double scale = ms / t; iters = (int)(iters * scale) + 1; if (iters > (1 << 22)) iters = 1 << 22; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    TG_CUDA(ctx, cudaGetLastError());
    *rate = best;
    return TAIGA_OK;
}

// FP64 tensor pipe: DMMA.8x8x4 (256 FMA per warp instruction) issue rate, in FMA per second.  On B200 it equals the
// DFMA rate (the two share the FP64 datapath: k_mixed_peak below), but reads each operand
// register for 8 FMAs: the denominator of the warp-cooperative tracer (trace_mma.cu).
__global__ void __launch_bounds__(256) k_dmma_peak(double* out, int iters, double a0, double b0) {
    double c[4][2], a[4], b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { c[i][0] = (double)threadIdx.x; c[i][1] = (double)i; a[i] = a0 + i * 1e-9; b[i] = b0 + i * 1e-9; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k)
#pragma unroll
            for (int i = 0; i < 4; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a[i]), "d"(b[i]));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

int tg_dmma_peak(taiga_ctx* ctx, double ms, double* rate) {
    cudaStream_t st = ctx->stream;
    cudaEvent_t e0, e1;
    TG_CUDA(ctx, cudaEventCreate(&e0));
    TG_CUDA(ctx, cudaEventCreate(&e1));
    double* dummy = (double*)ctx->counters + 12;
    unsigned grid = (unsigned)ctx->sm_count * 2;      // 2 x 256 threads = 16 warps per SM
    int iters = 256;
    float t = 0.f;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, st);
        k_dmma_peak<<<grid, 256, 0, st>>>(dummy, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); TG_CUDA(ctx, e); }
        cudaEventElapsedTime(&t, e0, e1);
        double n = (double)grid * 256.0 * (double)iters * 16.0 * 4.0 * 8.0;     // 8 FMA per lane and DMMA
        if (rep >= 2) { double r = n / (t * 1e-3); if (r > best) best = r; }
        if (rep == 1 && t > 0.f) { double scale = ms / t; iters = (int)(iters * scale) + 1; if (iters > (1 << 22)) iters = 1 << 22; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    TG_CUDA(ctx, cudaGetLastError());
    *rate = best;
    return TAIGA_OK;
}

// DFMA and DMMA chains interleaved, one DMMA (8 FMA per lane) per 8 DFMA: if the two had datapaths of their own the sum
// would approach twice the DFMA rate.  Measured: it stays below the DFMA rate, so 148 x 64 FMA/clk is the one FP64 roofline
// of the SM whichever instruction carries the work (profiles/r2a_microbench.md).
__global__ void __launch_bounds__(256) k_mixed_peak(double* out, int iters, double a0, double b0) {
    double c[2][2], a[2], b[2], v[4], m[4];
#pragma unroll
    for (int i = 0; i < 2; ++i) { c[i][0] = (double)threadIdx.x; c[i][1] = (double)i; a[i] = a0 + i * 1e-9; b[i] = b0 + i * 1e-9; }
#pragma unroll
    for (int i = 0; i < 4; ++i) { v[i] = (double)(threadIdx.x + i) * 1e-3; m[i] = a0 + i * 1e-9; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a[i]), "d"(b[i]));
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int j = 0; j < 4; ++j) v[j] = fma(v[j], m[j], b0);
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 2; ++i) s += c[i][0] + c[i][1];
#pragma unroll
    for (int i = 0; i < 4; ++i) s += v[i];
    if (s == 123.456) out[0] = s;
}

int tg_mixed_peak(taiga_ctx* ctx, double ms, double* rate) {
    cudaStream_t st = ctx->stream;
    cudaEvent_t e0, e1;
    TG_CUDA(ctx, cudaEventCreate(&e0));
    TG_CUDA(ctx, cudaEventCreate(&e1));
    double* dummy = (double*)ctx->counters + 12;
    unsigned grid = (unsigned)ctx->sm_count * 2;      // 16 warps per SM
    int iters = 256;
    float t = 0.f;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, st);
        k_mixed_peak<<<grid, 256, 0, st>>>(dummy, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); TG_CUDA(ctx, e); }
        cudaEventElapsedTime(&t, e0, e1);
        double n = (double)grid * 256.0 * (double)iters * 16.0 * 2.0 * (8.0 + 8.0);     // per lane: 8 FMA per DMMA + 8 DFMA
        if (rep >= 2) { double r = n / (t * 1e-3); if (r > best) best = r; }
        if (rep == 1 && t > 0.f) { double scale = ms / t; iters = (int)(iters * scale) + 1; if (iters > (1 << 22)) iters = 1 << 22; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    TG_CUDA(ctx, cudaGetLastError());
    *rate = best;
    return TAIGA_OK;
}

// ------------------------------------------------------------------------------------------
// Roofline denominator of the uncached field gathers (kinds 1 and 2): bytes per second that L1-resident
// 256-bit loads deliver to the registers of a kernel shaped like k_trace's gather (8 warps per SM, every
// lane reading a whole 1536-B "cell" with 48 x LDG.E.256).  spread = number of distinct cells the lanes
// of a warp read (1: all lanes the same addresses ... 32: every lane its own cell).
__global__ void __launch_bounds__(128) k_l1_gather_peak(const double* __restrict__ tab, int ncell, int spread, int iters, double* out) {
    int lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    double acc = 0.0;
    for (int it = 0; it < iters; ++it) {
        int cell = (warp * 7 + it * 3 + (lane % spread)) % ncell;
        const double* c = tab + (size_t)cell * 192;
#pragma unroll
        for (int k = 0; k < 48; ++k) {
            double a, b, d, e;
            asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(d), "=d"(e) : "l"(c + 4 * k));
            acc += (a + b) + (d + e);              // three adds per 32 bytes: the loads, not the ALU, are the work
        }
    }
    if (acc == 123.456) out[0] = acc;
}

int tg_l1_gather_peak(taiga_ctx* ctx, double ms, int spread, double* bytes_per_s) {
    cudaStream_t st = ctx->stream;
    const int ncell = 32;                              // 48 KB: L1-resident
    double* tab = nullptr;
    TG_CUDA(ctx, cudaMalloc((void**)&tab, (size_t)ncell * 192 * sizeof(double)));
    cudaMemsetAsync(tab, 0, (size_t)ncell * 192 * sizeof(double), st);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double* dummy = (double*)ctx->counters + 12;
    unsigned grid = (unsigned)ctx->sm_count * 2;       // 2 x 128 threads = 8 warps per SM, as k_trace
    if (spread < 1) spread = 1;
    if (spread > 32) spread = 32;
    int iters = 64;
    float t = 0.f;
    double best = 0.0;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 6 && err == cudaSuccess; ++rep) {
        cudaEventRecord(e0, st);
        k_l1_gather_peak<<<grid, 128, 0, st>>>(tab, ncell, spread, iters, dummy);
        cudaEventRecord(e1, st);
        err = cudaEventSynchronize(e1);
        if (err != cudaSuccess) break;
        cudaEventElapsedTime(&t, e0, e1);
        double n = (double)grid * 128.0 * (double)iters * 1536.0;
        if (rep >= 2) { double r = n / (t * 1e-3); if (r > best) best = r; }
        if (rep == 1 && t > 0.f) { double scale = ms / t; iters = (int)(iters * scale) + 1; if (iters > (1 << 22)) iters = 1 << 22; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(tab);
    TG_CUDA(ctx, err);
    TG_CUDA(ctx, cudaGetLastError());
    *bytes_per_s = best;
    return TAIGA_OK;
}
