// Device-side evaluation of the field tables (all kinds, uncached path).
// B(R,Z) = sum_ab c_ab p^a w^b  (stored bicubic spline coefficients),
// kind 1: linear blend of two slices in t, kind 2: sum_c q^c (bicubic_c) periodic in phi.
#pragma once
#include "taiga_internal.h"

// 16 coefficients [a][b] at c (32-byte aligned: one 128-B line, four 256-bit loads): Horner in w
// inside, in p outside.
__device__ __forceinline__ void tg_ld4(const double* p, double& a, double& b, double& c, double& d) {
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ double tg_bicubic(const double* __restrict__ c, double p, double w) {
    double a0, a1, a2, a3, b0, b1, b2, b3, c0, c1, c2, c3, d0, d1, d2, d3;
    tg_ld4(c, a0, a1, a2, a3); tg_ld4(c + 4, b0, b1, b2, b3);
    tg_ld4(c + 8, c0, c1, c2, c3); tg_ld4(c + 12, d0, d1, d2, d3);
    double r0 = fma(fma(fma(a3, w, a2), w, a1), w, a0);
    double r1 = fma(fma(fma(b3, w, b2), w, b1), w, b0);
    double r2 = fma(fma(fma(c3, w, c2), w, c1), w, c0);
    double r3 = fma(fma(fma(d3, w, d2), w, d1), w, d0);
    return fma(fma(fma(r3, p, r2), p, r1), p, r0);
}

__device__ __forceinline__ int tg_clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// fp32 variant (BASELINE config 5 "fp64 and fp32 variants"): 16 fp32 coefficients, two 256-bit loads
__device__ __forceinline__ float tg_bicubic32(const float* __restrict__ c, float p, float w) {
    float4 a0 = __ldg(reinterpret_cast<const float4*>(c)), a1 = __ldg(reinterpret_cast<const float4*>(c + 4));
    float4 a2 = __ldg(reinterpret_cast<const float4*>(c + 8)), a3 = __ldg(reinterpret_cast<const float4*>(c + 12));
    float r0 = fmaf(fmaf(fmaf(a0.w, w, a0.z), w, a0.y), w, a0.x);
    float r1 = fmaf(fmaf(fmaf(a1.w, w, a1.z), w, a1.y), w, a1.x);
    float r2 = fmaf(fmaf(fmaf(a2.w, w, a2.z), w, a2.y), w, a2.x);
    float r3 = fmaf(fmaf(fmaf(a3.w, w, a3.z), w, a3.y), w, a3.x);
    return fmaf(fmaf(fmaf(r3, p, r2), p, r1), p, r0);
}

// cell index and in-cell coordinate along one axis; outside the grid the boundary cell
// extrapolates (reading A12).
__device__ __forceinline__ int tg_locate(double x, double inv_h, double off, int ncell, double& frac) {
    double pt = fma(x, inv_h, -off);
    int i = tg_clampi(__double2int_rd(pt), 0, ncell - 1);
    frac = pt - (double)i;
    return i;
}

// kind 2, fp32 variant: cell and in-cell coordinates located in fp64 (no cancellation), the 189 FMAs
// of the tricubic evaluation and the table in fp32.
__device__ __forceinline__ void tg_field_cyl32(const FieldDev& f, double R, double Z, double s,
                                               double& BR, double& BZ, double& Bp) {
    double p, w;
    int i = tg_locate(R, f.inv_hR, f.offR, f.cR, p);
    int j = tg_locate(Z, f.inv_hZ, f.offZ, f.cZ, w);
    double xs = (s - f.s0) * f.inv_ds;
    xs = xs - (double)f.nS * floor(xs / (double)f.nS);
    int k = tg_clampi(__double2int_rd(xs), 0, f.nS - 1);
    float pf = (float)p, wf = (float)w, qf = (float)(xs - (double)k);
    const float* c = f.table32 + (((size_t)k * f.cR + i) * f.cZ + j) * 192;
    float out[3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        const float* d = c + m * 64;
        float e0 = tg_bicubic32(d, pf, wf), e1 = tg_bicubic32(d + 16, pf, wf);
        float e2 = tg_bicubic32(d + 32, pf, wf), e3 = tg_bicubic32(d + 48, pf, wf);
        out[m] = fmaf(fmaf(fmaf(e3, qf, e2), qf, e1), qf, e0);
    }
    BR = (double)out[0]; BZ = (double)out[1]; Bp = (double)out[2];
}

// (B_R, B_Z, B_phi) at (R, Z, s); s = time (kind 1) or phi (kind 2).
__device__ __forceinline__ void tg_field_cyl(const FieldDev& f, double R, double Z, double s,
                                             double& BR, double& BZ, double& Bp) {
    double p, w;
    int i = tg_locate(R, f.inv_hR, f.offR, f.cR, p);
    int j = tg_locate(Z, f.inv_hZ, f.offZ, f.cZ, w);
    size_t cell = (size_t)i * f.cZ + j;
    if (f.kind == 0) {
        const double* c = f.table + cell * 48;
        BR = tg_bicubic(c, p, w); BZ = tg_bicubic(c + 16, p, w); Bp = tg_bicubic(c + 32, p, w);
    } else if (f.kind == 1) {
        double xs = (s - f.s0) * f.inv_ds;
        int k = tg_clampi(__double2int_rd(xs), 0, f.nS - 2);
        double tau = fmin(fmax(xs - (double)k, 0.0), 1.0);
        const double* c = f.table + (cell * f.nS + k) * 48;
        double a0 = tg_bicubic(c, p, w), a1 = tg_bicubic(c + 16, p, w), a2 = tg_bicubic(c + 32, p, w);
        double b0 = tg_bicubic(c + 48, p, w), b1 = tg_bicubic(c + 64, p, w), b2 = tg_bicubic(c + 80, p, w);
        BR = fma(tau, b0 - a0, a0); BZ = fma(tau, b1 - a1, a1); Bp = fma(tau, b2 - a2, a2);
    } else {
        double xs = (s - f.s0) * f.inv_ds;
        xs = xs - (double)f.nS * floor(xs / (double)f.nS);
        int k = tg_clampi(__double2int_rd(xs), 0, f.nS - 1);
        double q = xs - (double)k;
        const double* c = f.table + (((size_t)k * f.cR + i) * f.cZ + j) * 192;
        double out[3];
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            const double* d = c + m * 64;
            double e0 = tg_bicubic(d, p, w), e1 = tg_bicubic(d + 16, p, w);
            double e2 = tg_bicubic(d + 32, p, w), e3 = tg_bicubic(d + 48, p, w);
            out[m] = fma(fma(fma(e3, q, e2), q, e1), q, e0);
        }
        BR = out[0]; BZ = out[1]; Bp = out[2];
    }
}
