// Device-side evaluation of the field tables (all kinds, uncached path).
// B(R,Z) = sum_ab c_ab p^a w^b  (stored bicubic spline coefficients),
// kind 1: linear blend of two slices in t, kind 2: sum_c q^c (bicubic_c) periodic in phi.
#pragma once
#include "taiga_internal.h"

__device__ __forceinline__ double2 tg_ld2(const double* p) {
    return __ldg(reinterpret_cast<const double2*>(p));
}

// 16 coefficients [a][b] at c (16-byte aligned): Horner in w inside, in p outside.
__device__ __forceinline__ double tg_bicubic(const double* __restrict__ c, double p, double w) {
    double2 a0 = tg_ld2(c + 0), a1 = tg_ld2(c + 2), b0 = tg_ld2(c + 4), b1 = tg_ld2(c + 6);
    double2 c0 = tg_ld2(c + 8), c1 = tg_ld2(c + 10), d0 = tg_ld2(c + 12), d1 = tg_ld2(c + 14);
    double r0 = fma(fma(fma(a1.y, w, a1.x), w, a0.y), w, a0.x);
    double r1 = fma(fma(fma(b1.y, w, b1.x), w, b0.y), w, b0.x);
    double r2 = fma(fma(fma(c1.y, w, c1.x), w, c0.y), w, c0.x);
    double r3 = fma(fma(fma(d1.y, w, d1.x), w, d0.y), w, d0.x);
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
