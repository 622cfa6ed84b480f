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

// cell index and in-cell coordinate along one axis; outside the grid the boundary cell
// extrapolates (reading A12).
__device__ __forceinline__ int tg_locate(double x, double inv_h, double off, int ncell, double& frac) {
    double pt = fma(x, inv_h, -off);
    int i = tg_clampi(__double2int_rd(pt), 0, ncell - 1);
    frac = pt - (double)i;
    return i;
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
