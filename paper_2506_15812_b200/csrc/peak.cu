// Roofline denominator: register-resident DFMA microkernel (MEASURED_PEAKS.json
// has no FP64 entry, so the FP64 issue rate is measured in the same run as the benchmark).
#include "taiga_internal.h"

#define PEAK_CHAINS 8
#define PEAK_INNER 64

__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters, double a, double b) {
    double v[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) v[c] = (double)(threadIdx.x + c) * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < PEAK_INNER; ++k) {
#pragma unroll
            for (int c = 0; c < PEAK_CHAINS; ++c) v[c] = fma(v[c], a, b);
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
