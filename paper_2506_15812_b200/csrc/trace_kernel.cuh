// a3 + a4: Runge-Kutta-Nystrom integrator, termination and plane interpolation: the kernel template (one lane = one ion).
// Instantiated by trace.cu (production path, loss, Bezier) and trace_variants.cu (electric field, other solvers).
//
// PAPER.md Eq. 3 (L172) with E = 0; Eq. 5-6 (L218-235) under readings A1-A3:
//   k1 = a(r, v);  k2 = a(r + v dt/2 + k1 dt^2/8, v + k1 dt/2);
//   k3 = a(r + v dt/2 + K dt^2/8, v + k2 dt/2), K = k1 (classical) | k2 (printed Eq. 6);
//   k4 = a(r + v dt + k3 dt^2/2, v + k3 dt);
//   r' = r + v dt + (k1+k2+k3) dt^2/6;   v' = v + (k1+2k2+2k3+k4) dt/6.
// L326/L338: stop at the detector plane, linear interpolation from the previous step;
// L318: error value for trapped / unreachable ions.
//
// B200 design (not the paper's one-thread-per-ion launch):
//  * one persistent kernel, 8 warps per SM; each LANE owns one ion whose state lives in
//    registers; finished lanes are refilled from a global queue of ions ordered by birth cell
//    (deep-born = long-running ions first), so warps stay full through the long tail and the
//    ions sharing a warp sit in the same few field cells;
//  * the velocity is carried as u = (q/m) v, so a = u x B needs no scaling per evaluation;
//  * classical variant: k2 and k3 share their position, so B is evaluated 3x, not 4x, per step;
//  * kind 0 (static 2-D): the 48 coefficients of the lane's current cell are cached in
//    registers and re-read (12 x 256-bit loads, one 128-B line per component) only when the
//    lane leaves the cell (~0.35 times per step);
//  * 1/R by MUFU.RSQ64H seed + one cubic (Halley) step: 6 FP64 instructions instead of ~30.
#pragma once
#include "trace_common.cuh"

template <int KIND>
struct CellCache;                              // register cache of the current cell (kind 0)
template <>
struct CellCache<0> {
    double c[48];
    double oR, oZ;                             // offR + i, offZ + j of the cached cell
    int i, j;                                  // its indices
};
template <>
struct CellCache<1> {                          // slice k of the current cell (PRED 2: the slice difference is gathered per
    double c[48];                              // evaluation) or its blend H_k + tau D_k at time coordinate `tau` (PRED 3)
    double oR, oZ;
    int k, cell;                               // cached slice, linear cell index i * cZ + j
    double tau;
};
template <>
struct CellCache<2> {};

__device__ __forceinline__ double tg_horner16(const double* c, double p, double w) {
    double r0 = fma(fma(fma(c[3], w, c[2]), w, c[1]), w, c[0]);
    double r1 = fma(fma(fma(c[7], w, c[6]), w, c[5]), w, c[4]);
    double r2 = fma(fma(fma(c[11], w, c[10]), w, c[9]), w, c[8]);
    double r3 = fma(fma(fma(c[15], w, c[14]), w, c[13]), w, c[12]);
    return fma(fma(fma(r3, p, r2), p, r1), p, r0);
}

// Re-read the register cache for the cell that contains the global cell coordinates (pR, pZ)
// (clamped to the grid: outside it the boundary cell extrapolates, reading A12).
__device__ __forceinline__ void tg_refill(const TraceParams& P, CellCache<0>& cc, unsigned& reloads, double pR, double pZ) {
    int i = tg_clampi(__double2int_rd(pR), 0, P.f.cR - 1), j = tg_clampi(__double2int_rd(pZ), 0, P.f.cZ - 1);
    cc.oR = P.f.offR + (double)i; cc.oZ = P.f.offZ + (double)j; cc.i = i; cc.j = j;
    const double* src = P.f.table + ((size_t)i * P.f.cZ + j) * 48;      // 384-B aligned
#pragma unroll
    for (int k = 0; k < 12; ++k)       // 12 x LDG.E.256 (sm_100: 256-bit global loads)
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "+d"(cc.c[4 * k]), "+d"(cc.c[4 * k + 1]), "+d"(cc.c[4 * k + 2]), "+d"(cc.c[4 * k + 3])
                     : "l"(src + 4 * k));
    ++reloads;
}

// (B_R, B_Z, B_phi) at (X,Y,Z,t) given R = sqrt(X^2+Y^2); cached path also returns the in-cell
// coordinates (tR, tZ) relative to the cached cell.
// FIRST (stage 1 of a step, cached path): also reports whether (R,Z) lies outside the grid; a
// point inside the cached cell is inside the grid, so the four comparisons run only on a refill.
// 4 predicated 256-bit loads into 16 cached coefficients (rolling refill)
__device__ __forceinline__ void tg_ldpred16(const double* src, int need, double* c) {
#pragma unroll
    for (int k = 0; k < 4; ++k)
        asm volatile("{ .reg .pred p; setp.ne.s32 p, %5, 0; @p ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4]; }"
                     : "+d"(c[4 * k]), "+d"(c[4 * k + 1]), "+d"(c[4 * k + 2]), "+d"(c[4 * k + 3])
                     : "l"(src + 4 * k), "r"(need));
}

// kind 1: re-read slice k of the cell containing the global cell coordinates (pR, pZ)
__device__ __forceinline__ void tg_refill1(const TraceParams& P, CellCache<1>& cc, unsigned& reloads, double pR, double pZ, int k) {
    int i = tg_clampi(__double2int_rd(pR), 0, P.f.cR - 1), j = tg_clampi(__double2int_rd(pZ), 0, P.f.cZ - 1);
    cc.oR = P.f.offR + (double)i; cc.oZ = P.f.offZ + (double)j; cc.k = k; cc.cell = i * P.f.cZ + j;
    const double* src = P.f.table + ((size_t)cc.cell * P.f.nS + k) * 48;
#pragma unroll
    for (int q = 0; q < 12; ++q)
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "+d"(cc.c[4 * q]), "+d"(cc.c[4 * q + 1]), "+d"(cc.c[4 * q + 2]), "+d"(cc.c[4 * q + 3])
                     : "l"(src + 4 * q));
    ++reloads;
}

template <int KIND, bool CACHED, bool FIRST = false, bool ROLL = false>
__device__ __forceinline__ void tg_fieldCyl(const TraceParams& P, CellCache<KIND>& cc, unsigned& reloads, bool& outside,
                                            double X, double Y, double Z, double t, double R,
                                            double& BR, double& BZ, double& Bp, double& tR, double& tZ,
                                            double dR = 0.0, double dZ = 0.0) {
    if constexpr (KIND == 0 && CACHED && ROLL) {
        // Rolling predictive refill: the next stage's in-cell coordinates are predicted to ~1e-3
        // cell (tRp, tZp); if they leave the cached cell, each part of the cache is re-read for
        // the successor cell once this stage's Horner sums have consumed it, so the L2 round trip
        // overlaps the rest of the stage.  Every stage still verifies its true coordinates
        // against the cached cell first, so a wrong guess costs a second refill and nothing else.
        tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        if (!(tg_in01(tR) && tg_in01(tZ))) {
            if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
            tg_refill(P, cc, reloads, fma(R, P.f.inv_hR, -P.f.offR), fma(Z, P.f.inv_hZ, -P.f.offZ));
            tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        }
        double tRp = tR + dR, tZp = tZ + dZ;
        // Branch-free (30.6 against 31.5 ms with a divergent block, profiles/r2_experiments.md): the predicted point is at most
        // one cell away in each direction, so the successor's indices are the cached ones -1 / 0 / +1 from the sign and the
        // exponent of the predicted coordinates; a wrong guess is corrected by the next stage's verify.
        const unsigned hR = (unsigned)__double2hiint(tRp), hZ = (unsigned)__double2hiint(tZp);
        const int i2 = tg_clampi(cc.i + (int)(hR >= 0x3FF00000u) - 2 * (int)(hR >> 31), 0, P.f.cR - 1);
        const int j2 = tg_clampi(cc.j + (int)(hZ >= 0x3FF00000u) - 2 * (int)(hZ >> 31), 0, P.f.cZ - 1);
        const int need = (i2 != cc.i) | (j2 != cc.j);
        cc.i = i2; cc.j = j2;
        cc.oR = P.f.offR + (double)i2; cc.oZ = P.f.offZ + (double)j2;
        const double* src = P.f.table + ((size_t)i2 * P.f.cZ + j2) * 48;
        reloads += need;
        BR = tg_horner16(cc.c, tR, tZ);      tg_ldpred16(src, need, cc.c);
        BZ = tg_horner16(cc.c + 16, tR, tZ); tg_ldpred16(src + 16, need, cc.c + 16);
        Bp = tg_horner16(cc.c + 32, tR, tZ); tg_ldpred16(src + 32, need, cc.c + 32);
    } else if constexpr (KIND == 1 && CACHED) {
        // Time slices: B(t) = H(T_k) + tau H(T_k+1 - T_k).  Slice k of the current cell is cached in
        // registers with the same rolling predictive refill as kind 0; only the slice DIFFERENCE is
        // gathered (384 instead of 768 bytes per lane and evaluation).
        double xs = (t - P.f.s0) * P.f.inv_ds;
        int k = tg_clampi(__double2int_rd(xs), 0, P.f.nS - 2);
        double tau = fmin(fmax(xs - (double)k, 0.0), 1.0);
        tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        if (!(tg_in01(tR) && tg_in01(tZ)) || k != cc.k) {
            if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
            tg_refill1(P, cc, reloads, fma(R, P.f.inv_hR, -P.f.offR), fma(Z, P.f.inv_hZ, -P.f.offZ), k);
            tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        }
        const double* dsrc = P.f.dtable + ((size_t)cc.cell * (P.f.nS - 1) + k) * 48;   // of the CURRENT cell
        double tRp = tR + dR, tZp = tZ + dZ;
        int need = ROLL && !(tg_in01(tRp) && tg_in01(tZp));
        const double* src = P.f.table;
        if (need) {
            int i = tg_clampi(__double2int_rd(tRp + (cc.oR - P.f.offR)), 0, P.f.cR - 1);
            int j = tg_clampi(__double2int_rd(tZp + (cc.oZ - P.f.offZ)), 0, P.f.cZ - 1);
            cc.oR = P.f.offR + (double)i; cc.oZ = P.f.offZ + (double)j; cc.cell = i * P.f.cZ + j;
            src += ((size_t)cc.cell * P.f.nS + k) * 48;
            ++reloads;
        }
        double a0 = tg_horner16(cc.c, tR, tZ);      tg_ldpred16(src, need, cc.c);
        double a1 = tg_horner16(cc.c + 16, tR, tZ); tg_ldpred16(src + 16, need, cc.c + 16);
        double a2 = tg_horner16(cc.c + 32, tR, tZ); tg_ldpred16(src + 32, need, cc.c + 32);
        BR = fma(tau, tg_bicubic(dsrc, tR, tZ), a0);
        BZ = fma(tau, tg_bicubic(dsrc + 16, tR, tZ), a1);
        Bp = fma(tau, tg_bicubic(dsrc + 32, tR, tZ), a2);
    } else if constexpr (KIND == 0 && CACHED) {
        tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        if (!(tg_in01(tR) && tg_in01(tZ))) {
            if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
            tg_refill(P, cc, reloads, fma(R, P.f.inv_hR, -P.f.offR), fma(Z, P.f.inv_hZ, -P.f.offZ));
            tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        }
        BR = tg_horner16(cc.c, tR, tZ); BZ = tg_horner16(cc.c + 16, tR, tZ); Bp = tg_horner16(cc.c + 32, tR, tZ);
    } else {
        if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
        double s = t;
        if constexpr (KIND == 2) s = atan2(Y, X);
        if (KIND == 2 && P.f.table32) tg_field_cyl32(P.f, R, Z, s, BR, BZ, Bp);
        else tg_field_cyl(P.f, R, Z, s, BR, BZ, Bp);
    }
}

// Kind 1, blended cache (PRED 3).  B(t) = H_k + tau (H_k+1 - H_k) is linear in tau, so the lane keeps the BLENDED
// coefficients C = H_k + tau_c D_k of its cell in registers and moves them along in time instead of gathering D_k at
// every evaluation: stages 1 and 4 (tau = tau_c) are a Horner sum over registers; stage 2 (STREAM) streams D_k once,
// advances C to the time of the step end, tau_n, and evaluates B = H(C) + (tau - tau_n) H(D_k) at its own time.  One
// 384-B gather per ion-step instead of three, 231 instead of 279 FP64 instructions.  A new cell or slice re-blends
// from the two tables (768 B); rounding differs from H_k + tau D_k only by the few additions since the last re-blend.
template <bool FIRST, bool STREAM>
__device__ __forceinline__ void tg_field_blend(const TraceParams& P, CellCache<1>& cc, unsigned& reloads, bool& outside,
                                               double R, double Z, double t, double t_next, double& BR, double& BZ, double& Bp) {
    const double xs = (t - P.f.s0) * P.f.inv_ds;
    const int k = tg_clampi(__double2int_rd(xs), 0, P.f.nS - 2);
    const double tau = fmin(fmax(xs - (double)k, 0.0), 1.0);
    double tR = fma(R, P.f.inv_hR, -cc.oR), tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
    const bool hit = tg_in01(tR) && tg_in01(tZ) && k == cc.k;
    double out[3];
    if (!hit) {                                // another cell or slice: locate it (clamped: the boundary cell extrapolates)
        if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
        int i = tg_clampi(__double2int_rd(fma(R, P.f.inv_hR, -P.f.offR)), 0, P.f.cR - 1);
        int j = tg_clampi(__double2int_rd(fma(Z, P.f.inv_hZ, -P.f.offZ)), 0, P.f.cZ - 1);
        cc.oR = P.f.offR + (double)i; cc.oZ = P.f.offZ + (double)j; cc.k = k; cc.cell = i * P.f.cZ + j;
        tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        ++reloads;
    }
    const double* hsrc = P.f.table + ((size_t)cc.cell * P.f.nS + cc.k) * 48;
    const double* dsrc = P.f.dtable + ((size_t)cc.cell * (P.f.nS - 1) + cc.k) * 48;
    if constexpr (!STREAM) {
        if (!hit || tau != cc.tau) {           // re-blend at this evaluation's time
#pragma unroll
            for (int m = 0; m < 3; ++m) {
                double d[16];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    tg_ld4(hsrc + m * 16 + 4 * q, cc.c[m * 16 + 4 * q], cc.c[m * 16 + 4 * q + 1], cc.c[m * 16 + 4 * q + 2], cc.c[m * 16 + 4 * q + 3]);
                    tg_ld4(dsrc + m * 16 + 4 * q, d[4 * q], d[4 * q + 1], d[4 * q + 2], d[4 * q + 3]);
                }
#pragma unroll
                for (int q = 0; q < 16; ++q) cc.c[m * 16 + q] = fma(tau, d[q], cc.c[m * 16 + q]);
            }
            cc.tau = tau;
        }
#pragma unroll
        for (int m = 0; m < 3; ++m) out[m] = tg_horner16(cc.c + m * 16, tR, tZ);
    } else {
        const double tau_n = fmin(fmax((t_next - P.f.s0) * P.f.inv_ds - (double)cc.k, 0.0), 1.0);
        if (!hit) {                            // C = H_k, to be advanced from tau_c = 0
#pragma unroll
            for (int q = 0; q < 12; ++q)
                tg_ld4(hsrc + 4 * q, cc.c[4 * q], cc.c[4 * q + 1], cc.c[4 * q + 2], cc.c[4 * q + 3]);
            cc.tau = 0.0;
        }
        const double adv = tau_n - cc.tau, back = tau - tau_n;
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            double d[16];
#pragma unroll
            for (int q = 0; q < 4; ++q) tg_ld4(dsrc + m * 16 + 4 * q, d[4 * q], d[4 * q + 1], d[4 * q + 2], d[4 * q + 3]);
            const double hD = tg_horner16(d, tR, tZ);
#pragma unroll
            for (int q = 0; q < 16; ++q) cc.c[m * 16 + q] = fma(adv, d[q], cc.c[m * 16 + q]);
            out[m] = fma(back, hD, tg_horner16(cc.c + m * 16, tR, tZ));
        }
        cc.tau = tau_n;
    }
    BR = out[0]; BZ = out[1]; Bp = out[2];
}

// Kind 1, blended cache with the slice difference in shared memory (PRED 4).  As tg_field_blend, but D_k of the lane's
// cell lives in the lane's own 384-B shared-memory slot (stride TG_SLOT = 400 B: the 16-B chunks of eight consecutive
// lanes cover all 32 banks, so a warp-wide LDS.128 is 4 wavefronts whatever cells the lanes sit in).  The slot is
// filled by cp.async when the lane enters a cell (no register staging, no write-back port), so the once-per-step stream
// of D_k no longer goes through divergent 256-bit L1 gathers: those cost 8 / 16 / 32 wavefronts per load with 1 / 2 /
// >= 4 cells per warp (taiga_measure_l1_gather_peak) and kept the L1 data pipe 71 % busy (profiles/r2_trace_ncu.md).
#define TG_SLOT 400
__device__ __forceinline__ void tg_lds2(unsigned a, double& x, double& y) {
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(x), "=d"(y) : "r"(a) : "memory");
}
template <bool FIRST, bool STREAM>
__device__ __forceinline__ void tg_field_blend_sm(const TraceParams& P, CellCache<1>& cc, unsigned& reloads, bool& outside, unsigned sd,
                                                  double R, double Z, double t, double t_next, double& BR, double& BZ, double& Bp) {
    const double xs = (t - P.f.s0) * P.f.inv_ds;
    const int k = tg_clampi(__double2int_rd(xs), 0, P.f.nS - 2);
    const double tau = fmin(fmax(xs - (double)k, 0.0), 1.0);
    double tR = fma(R, P.f.inv_hR, -cc.oR), tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
    const bool hit = tg_in01(tR) && tg_in01(tZ) && k == cc.k;
    double out[3];
    if (!hit) {                                // another cell or slice: D_k -> my slot (asynchronous), H_k -> C
        if constexpr (FIRST) outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
        int i = tg_clampi(__double2int_rd(fma(R, P.f.inv_hR, -P.f.offR)), 0, P.f.cR - 1);
        int j = tg_clampi(__double2int_rd(fma(Z, P.f.inv_hZ, -P.f.offZ)), 0, P.f.cZ - 1);
        cc.oR = P.f.offR + (double)i; cc.oZ = P.f.offZ + (double)j; cc.k = k; cc.cell = i * P.f.cZ + j;
        tR = fma(R, P.f.inv_hR, -cc.oR); tZ = fma(Z, P.f.inv_hZ, -cc.oZ);
        const double* hsrc = P.f.table + ((size_t)cc.cell * P.f.nS + cc.k) * 48;
        const double* dsrc = P.f.dtable + ((size_t)cc.cell * (P.f.nS - 1) + cc.k) * 48;
        // a copy of an earlier refill may still be in flight (a new ion starts at tau = 0 exactly and blends nothing, so its
        // first evaluation does not wait): two copies into one slot complete in any order, the older must have landed first
        asm volatile("cp.async.wait_all;" ::: "memory");
#pragma unroll
        for (int q = 0; q < 24; ++q)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sd + 16 * q), "l"(dsrc + 2 * q) : "memory");
#pragma unroll
        for (int q = 0; q < 12; ++q)
            tg_ld4(hsrc + 4 * q, cc.c[4 * q], cc.c[4 * q + 1], cc.c[4 * q + 2], cc.c[4 * q + 3]);
        cc.tau = 0.0;
        ++reloads;
    }
    if constexpr (!STREAM) {
        if (tau != cc.tau) {                   // bring C to this evaluation's time (after a refill: from H_k)
            asm volatile("cp.async.wait_all;" ::: "memory");
            const double adv = tau - cc.tau;
#pragma unroll
            for (int q = 0; q < 24; ++q) {
                double d0, d1;
                tg_lds2(sd + 16 * q, d0, d1);
                cc.c[2 * q] = fma(adv, d0, cc.c[2 * q]); cc.c[2 * q + 1] = fma(adv, d1, cc.c[2 * q + 1]);
            }
            cc.tau = tau;
        }
#pragma unroll
        for (int m = 0; m < 3; ++m) out[m] = tg_horner16(cc.c + m * 16, tR, tZ);
    } else {
        const double tau_n = fmin(fmax((t_next - P.f.s0) * P.f.inv_ds - (double)cc.k, 0.0), 1.0);
        asm volatile("cp.async.wait_all;" ::: "memory");
        const double adv = tau_n - cc.tau, back = tau - tau_n;
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            double d[16];
#pragma unroll
            for (int q = 0; q < 8; ++q) tg_lds2(sd + 128 * m + 16 * q, d[2 * q], d[2 * q + 1]);
            const double hD = tg_horner16(d, tR, tZ);
#pragma unroll
            for (int q = 0; q < 16; ++q) cc.c[m * 16 + q] = fma(adv, d[q], cc.c[m * 16 + q]);
            out[m] = fma(back, hD, tg_horner16(cc.c + m * 16, tR, tZ));
        }
        cc.tau = tau_n;
    }
    BR = out[0]; BZ = out[1]; Bp = out[2];
}

// Predictive refill (kind 0, cached): right after the Horner evaluation of one stage has read the
// cached coefficients for the last time, the in-cell coordinates of the NEXT stage are predicted
// to ~1e-3 cell (tRp, tZp); if they fall outside the cached cell its successor is loaded now, so
// that the L2 round trip overlaps the rotation, cross product and 1/R chain in between.  The next
// stage still tests its true coordinates against the cached cell, so a wrong guess costs a second
// refill and nothing else.
__device__ __forceinline__ void tg_predict(const TraceParams& P, CellCache<0>& cc, unsigned& reloads, double tRp, double tZp,
                                           double BR, double BZ, double Bp) {
    asm volatile("" ::"d"(BR), "d"(BZ), "d"(Bp));      // the stage's Horner sums are complete: the old coefficients are dead
    if (!(tg_in01(tRp) && tg_in01(tZp)))
        tg_refill(P, cc, reloads, tRp + (cc.oR - P.f.offR), tZp + (cc.oZ - P.f.offZ));
}

// Cartesian B at a stage point (on-demand cache refill / uncached gather); solvers other than RKN
template <int KIND, bool CACHED>
__device__ __forceinline__ void tg_fieldXYZ(const TraceParams& P, CellCache<KIND>& cc, unsigned& reloads,
                                            double Xs, double Ys, double Zs, double ts, double& bx, double& by, double& bz) {
    double r2 = fma(Xs, Xs, Ys * Ys), ri = tg_rsqrt(r2), Rs = r2 * ri, br, bp, tR, tZ;
    bool dummy = false;
    tg_fieldCyl<KIND, CACHED>(P, cc, reloads, dummy, Xs, Ys, Zs, ts, Rs, br, bz, bp, tR, tZ);
    tg_rotate(Xs, Ys, ri, br, bp, bx, by);
}

// SOLVER: 0 Runge-Kutta-Nystrom (Eq. 5-6), 2 linearised RK4 (Eq. 4), 3 Boris (Eq. 7-8; P.variant 3 =
// Verlet form with leap-frog start, 4 = Eq. 8 as printed).  HAS_E: uniform E of Eq. 3 added to every k.
// LOSS: integrate Eq. 2 along the trajectory (trapezoid over step end points) and write exp(-integral).
// BEZ: quadratic Bezier instead of linear interpolation to the plane (reading Z1).
// REGROUP (uncached kinds): the CTA draws tiles of THREADS ions and, every P.regroup_every steps, re-sorts
// its ions over the lanes by field cell through shared memory, so that the lanes of a warp gather from as
// few distinct cells as possible: L1 delivers 128 B/clk/SM when a warp reads one cell, 64 with two, 32 with
// four or more (taiga_measure_l1_gather_peak).
template <int KIND, bool CACHED, int THREADS, int MAXREG, int PRED = 0, int SOLVER = 0, bool HAS_E = false, bool LOSS = false,
          bool BEZ = false, bool REGROUP = false>
__global__ void __launch_bounds__(THREADS) __maxnreg__(MAXREG) k_trace(const TraceParams P) {
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    CellCache<KIND> cc;
    if constexpr (KIND == 1 && CACHED) { cc.k = -1; cc.cell = 0; cc.tau = -1.0; }
    if constexpr (KIND == 0 && CACHED) { cc.i = 0; cc.j = 0; }
    if constexpr (KIND <= 1 && CACHED) { cc.oR = 1e300; cc.oZ = 1e300;
#pragma unroll
        for (int k = 0; k < 48; ++k) cc.c[k] = 0.0; }
    double X = 0, Y = 0, Z = 0, Ux = 0, Uy = 0, Uz = 0, t = 0, s0 = -1.0;
    double Lam = 0.0, nu0 = 0.0;               // LOSS: integral of nu dt, nu at the last step end point
    uint32_t idx = 0, nst = 0;
    bool alive = false, exhausted = false;
    unsigned reloads = 0, ion_steps = 0;       // per lane; < 2^32 for any run the queue allows
    unsigned long long warp_steps = 0;

    [[maybe_unused]] unsigned sd = 0;          // PRED 4: shared address of this lane's slice-difference slot
    if constexpr (KIND == 1 && PRED == 4) {
        extern __shared__ __align__(16) unsigned char tg_dyn_smem[];
        sd = (unsigned)__cvta_generic_to_shared(tg_dyn_smem) + threadIdx.x * TG_SLOT;
    }
    [[maybe_unused]] int since = 0;            // REGROUP: iterations since the last CTA sync point
    while (true) {
      unsigned am;
      if constexpr (REGROUP) {
        __shared__ double sh_d[8][THREADS];
        __shared__ uint32_t sh_u[2][THREADS];
        __shared__ int sh_key[2][THREADS];
        __shared__ unsigned long long s_base;
        const int tid = threadIdx.x;
        if (since == 0) {                      // every warp of the CTA arrives here at the same iteration count
            int nalive = __syncthreads_count(alive);
            if (nalive == 0) {                 // CTA-wide tile of THREADS consecutive queue entries
                if (exhausted) break;
                if (tid == 0) s_base = atomicAdd(&P.counters[0], (unsigned long long)THREADS);
                __syncthreads();
                unsigned long long q = s_base + tid;
                if (s_base + THREADS >= P.n) exhausted = true;
                if (q < P.n) {
                    idx = P.order ? P.order[q] : (uint32_t)q;
                    X = P.x[idx]; Y = P.y[idx]; Z = P.z[idx];
                    Ux = P.qm * P.vx[idx]; Uy = P.qm * P.vy[idx]; Uz = P.qm * P.vz[idx];
                    t = P.t0 ? P.t0[idx] : 0.0;
                    nst = 0;
                    s0 = fma(P.det.normal[0], X, fma(P.det.normal[1], Y, fma(P.det.normal[2], Z, -P.nrD)));
                    alive = true;
                    if (!(s0 < 0.0)) {
                        P.hit_u[idx] = 0.0; P.hit_w[idx] = 0.0; P.cell[idx] = TAIGA_CELL_BADSTART; P.steps[idx] = 0;
                        P.flags[idx] = (fabs(s0) < TG_GRAZE) ? TAIGA_FLAG_PLANE : 0;
                        alive = false;
                    }
                }
            } else {                           // re-sort the CTA's ions over its lanes by field cell
                int key = 0x7fffffff;
                if (alive) {
                    double p_, w_;
                    int i = tg_locate(sqrt(fma(X, X, Y * Y)), P.f.inv_hR, P.f.offR, P.f.cR, p_);
                    int j = tg_locate(Z, P.f.inv_hZ, P.f.offZ, P.f.cZ, w_);
                    int k = 0;
                    if constexpr (KIND == 2) {
                        double xs = (atan2(Y, X) - P.f.s0) * P.f.inv_ds;
                        xs -= (double)P.f.nS * floor(xs / (double)P.f.nS);
                        k = tg_clampi(__double2int_rd(xs), 0, P.f.nS - 1);
                    }
                    key = (k * P.f.cR + i) * P.f.cZ + j;
                }
                sh_key[0][tid] = key;
                __syncthreads();
                int rank = 0;
#pragma unroll 8
                for (int o = 0; o < THREADS; ++o) { int ko = sh_key[0][o]; rank += (ko < key) | ((ko == key) & (o < tid)); }
                sh_d[0][rank] = X; sh_d[1][rank] = Y; sh_d[2][rank] = Z; sh_d[3][rank] = Ux; sh_d[4][rank] = Uy; sh_d[5][rank] = Uz;
                sh_d[6][rank] = t; sh_d[7][rank] = s0; sh_u[0][rank] = idx; sh_u[1][rank] = nst; sh_key[1][rank] = key;
                __syncthreads();
                X = sh_d[0][tid]; Y = sh_d[1][tid]; Z = sh_d[2][tid]; Ux = sh_d[3][tid]; Uy = sh_d[4][tid]; Uz = sh_d[5][tid];
                t = sh_d[6][tid]; s0 = sh_d[7][tid]; idx = sh_u[0][tid]; nst = sh_u[1][tid]; alive = sh_key[1][tid] != 0x7fffffff;
            }
        }
        since = (since + 1 >= P.regroup_every) ? 0 : since + 1;
        am = __ballot_sync(FULL, alive);
        if (am == 0) continue;                 // this warp idles until the next sync point
      } else {
        am = __ballot_sync(FULL, alive);
        unsigned freem = ~am;
        int nfree = __popc(freem);
        if (nfree >= P.refill_min && !exhausted) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(&P.counters[0], (unsigned long long)nfree);
            base = __shfl_sync(FULL, base, 0);
            if (base + nfree >= P.n) exhausted = true;
            unsigned long long q = base + __popc(freem & ((1u << lane) - 1u));
            if (!alive && q < P.n) {
                idx = P.order ? P.order[q] : (uint32_t)q;
                X = P.x[idx]; Y = P.y[idx]; Z = P.z[idx];
                Ux = P.qm * P.vx[idx]; Uy = P.qm * P.vy[idx]; Uz = P.qm * P.vz[idx];
                t = P.t0 ? P.t0[idx] : 0.0;
                nst = 0;
                if constexpr (LOSS) Lam = 0.0;
                s0 = fma(P.det.normal[0], X, fma(P.det.normal[1], Y, fma(P.det.normal[2], Z, -P.nrD)));
                alive = true;
                if (!(s0 < 0.0)) {             // O4: must start in front of the plane
                    P.hit_u[idx] = 0.0; P.hit_w[idx] = 0.0; P.cell[idx] = TAIGA_CELL_BADSTART; P.steps[idx] = 0;
                    P.flags[idx] = (fabs(s0) < TG_GRAZE) ? TAIGA_FLAG_PLANE : 0;
                    if constexpr (LOSS) P.weight[idx] = P.w0 ? P.w0[idx] : 1.0;
                    alive = false;
                }
            }
            am = __ballot_sync(FULL, alive);
        }
        if (am == 0) { if (exhausted) break; else continue; }
      }
      // Steps repeat here until a lane of the warp finishes: the loop head above (vote, queue refill, exit test) has nothing
      // to decide before that and costs 13 control instructions per step (profiles/r2_experiments.md)
      bool again;
      do {
        const bool was_alive = alive;
        ++warp_steps;
        if (alive) {
            // ---- stage 1 at (r, u); its grid test is the out-of-grid test of the previous step (O4)
            double R2 = fma(X, X, Y * Y), R, rinv = tg_rsq<KIND == 0>(R2, R);
            double Bx, By, Bz, BR, Bp, tR, tZ;
            bool outside = false, dummy = false;
            double dR = 0.0, dZ = 0.0;         // predicted half-step displacement in cells
            if constexpr (PRED == 1 || PRED == 2) { dR = (fma(X, Ux, Y * Uy) * rinv) * P.pa1R; dZ = Uz * P.pa1Z; }
            if constexpr (KIND == 1 && PRED == 3) tg_field_blend<true, false>(P, cc, reloads, outside, R, Z, t, 0.0, BR, Bz, Bp);
            else if constexpr (KIND == 1 && PRED == 4) tg_field_blend_sm<true, false>(P, cc, reloads, outside, sd, R, Z, t, 0.0, BR, Bz, Bp);
            else tg_fieldCyl<KIND, CACHED, true, PRED == 2>(P, cc, reloads, outside, X, Y, Z, t, R, BR, Bz, Bp, tR, tZ, dR, dZ);
            double nu1 = 0.0;
            if constexpr (LOSS) {                  // trapezoid of the step that ended at this point (not of a step that left the grid)
                nu1 = tg_loss_rate(P, R, Z);
                if (nst > 0 && !outside) Lam = fma(P.hdt, nu0 + nu1, Lam);
            }
            if (outside || nst == P.max_steps) {
                uint8_t fl = 0;
                if constexpr (LOSS) P.weight[idx] = (P.w0 ? P.w0[idx] : 1.0) * ((outside && nst == 0) ? 1.0 : exp(-Lam));
                if (outside && (fabs(R - P.f.Rmin) < TG_GRAZE || fabs(R - P.f.Rmax) < TG_GRAZE ||
                                fabs(Z - P.f.Zmin) < TG_GRAZE || fabs(Z - P.f.Zmax) < TG_GRAZE)) fl = TAIGA_FLAG_GRID;
                P.hit_u[idx] = 0.0; P.hit_w[idx] = 0.0;
                P.cell[idx] = outside ? (nst == 0 ? TAIGA_CELL_BADSTART : TAIGA_CELL_OUT) : TAIGA_CELL_MAXSTEPS;
                P.steps[idx] = nst; P.flags[idx] = fl;
                alive = false;
            } else {
                double Xn, Yn, Zn;
                double c1x = 0.0, c1y = 0.0, c1z = 0.0;      // BEZ: r_n + v_n dt/2
                if constexpr (BEZ) { c1x = fma(Ux, P.a1, X); c1y = fma(Uy, P.a1, Y); c1z = fma(Uz, P.a1, Z); }
                if constexpr (SOLVER == 0) {
                if constexpr (PRED == 1) tg_predict(P, cc, reloads, tR + dR, tZ + dZ, BR, Bz, Bp);
                tg_rotate(X, Y, rinv, BR, Bp, Bx, By);
                double k1x = fma(Uy, Bz, -(Uz * By)), k1y = fma(Uz, Bx, -(Ux * Bz)), k1z = fma(Ux, By, -(Uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, X, Y, Z, k1x, k1y, k1z);
                // ---- stage 2 (and 3, classical: same position)
                double Xm = fma(k1x, P.a2, fma(Ux, P.a1, X)), Ym = fma(k1y, P.a2, fma(Uy, P.a1, Y)), Zm = fma(k1z, P.a2, fma(Uz, P.a1, Z));
                double ux = fma(k1x, P.b1, Ux), uy = fma(k1y, P.b1, Uy), uz = fma(k1z, P.b1, Uz);
                double tm = t + 0.5 * P.dt;
                R2 = fma(Xm, Xm, Ym * Ym); rinv = tg_rsq<KIND == 0>(R2, R);
                if constexpr (KIND == 1 && PRED == 3) tg_field_blend<false, true>(P, cc, reloads, dummy, R, Zm, tm, t + P.dt, BR, Bz, Bp);
                else if constexpr (KIND == 1 && PRED == 4) tg_field_blend_sm<false, true>(P, cc, reloads, dummy, sd, R, Zm, tm, t + P.dt, BR, Bz, Bp);
                else tg_fieldCyl<KIND, CACHED, false, PRED == 2>(P, cc, reloads, dummy, Xm, Ym, Zm, tm, R, BR, Bz, Bp, tR, tZ, dR, dZ);
                if constexpr (PRED == 1) tg_predict(P, cc, reloads, tR + dR, tZ + dZ, BR, Bz, Bp);
                tg_rotate(Xm, Ym, rinv, BR, Bp, Bx, By);
                double k2x = fma(uy, Bz, -(uz * By)), k2y = fma(uz, Bx, -(ux * Bz)), k2z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xm, Ym, Zm, k2x, k2y, k2z);
                ux = fma(k2x, P.b1, Ux); uy = fma(k2y, P.b1, Uy); uz = fma(k2z, P.b1, Uz);
                if (P.variant) {               // printed Eq. 6: k3 position increment from k2
                    Xm = fma(k2x, P.a2, fma(Ux, P.a1, X)); Ym = fma(k2y, P.a2, fma(Uy, P.a1, Y)); Zm = fma(k2z, P.a2, fma(Uz, P.a1, Z));
                    R2 = fma(Xm, Xm, Ym * Ym); rinv = tg_rsq<KIND == 0>(R2, R);
                    if constexpr (KIND == 1 && PRED == 3) tg_field_blend<false, false>(P, cc, reloads, dummy, R, Zm, tm, 0.0, BR, Bz, Bp);
                    else if constexpr (KIND == 1 && PRED == 4) tg_field_blend_sm<false, false>(P, cc, reloads, dummy, sd, R, Zm, tm, 0.0, BR, Bz, Bp);
                    else tg_fieldCyl<KIND, CACHED>(P, cc, reloads, dummy, Xm, Ym, Zm, tm, R, BR, Bz, Bp, tR, tZ);   // on-demand verify / refill
                    tg_rotate(Xm, Ym, rinv, BR, Bp, Bx, By);
                }
                double k3x = fma(uy, Bz, -(uz * By)), k3y = fma(uz, Bx, -(ux * Bz)), k3z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xm, Ym, Zm, k3x, k3y, k3z);
                // ---- stage 4
                double Xe = fma(k3x, 4.0 * P.a2, fma(Ux, 2.0 * P.a1, X)), Ye = fma(k3y, 4.0 * P.a2, fma(Uy, 2.0 * P.a1, Y)),
                       Ze = fma(k3z, 4.0 * P.a2, fma(Uz, 2.0 * P.a1, Z));
                ux = fma(k3x, 2.0 * P.b1, Ux); uy = fma(k3y, 2.0 * P.b1, Uy); uz = fma(k3z, 2.0 * P.b1, Uz);
                R2 = fma(Xe, Xe, Ye * Ye); rinv = tg_rsq<KIND == 0>(R2, R);
                if constexpr (KIND == 1 && PRED == 3) tg_field_blend<false, false>(P, cc, reloads, dummy, R, Ze, t + P.dt, 0.0, BR, Bz, Bp);
                else if constexpr (KIND == 1 && PRED == 4) tg_field_blend_sm<false, false>(P, cc, reloads, dummy, sd, R, Ze, t + P.dt, 0.0, BR, Bz, Bp);
                else tg_fieldCyl<KIND, CACHED>(P, cc, reloads, dummy, Xe, Ye, Ze, t + P.dt, R, BR, Bz, Bp, tR, tZ);
                tg_rotate(Xe, Ye, rinv, BR, Bp, Bx, By);
                double k4x = fma(uy, Bz, -(uz * By)), k4y = fma(uz, Bx, -(ux * Bz)), k4z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xe, Ye, Ze, k4x, k4y, k4z);
                // ---- Eq. 5
                double Tx = k2x + k3x, Ty = k2y + k3y, Tz = k2z + k3z;
                Xn = fma(k1x + Tx, P.c6, fma(Ux, P.dtq, X)); Yn = fma(k1y + Ty, P.c6, fma(Uy, P.dtq, Y));
                Zn = fma(k1z + Tz, P.c6, fma(Uz, P.dtq, Z));
                Ux = fma(fma(2.0, Tx, k1x + k4x), P.d6, Ux);
                Uy = fma(fma(2.0, Ty, k1y + k4y), P.d6, Uy);
                Uz = fma(fma(2.0, Tz, k1z + k4z), P.d6, Uz);
                } else {
                tg_rotate(X, Y, rinv, BR, Bp, Bx, By);
                if constexpr (SOLVER == 2) {
                    // ---- Eq. 4: classical RK4 on y = (r, v); with u = (q/m) v and k = dv/dt:
                    //  r2 = r + v dt/2;            r3 = r + v dt/2 + k1 dt^2/4;   r4 = r + v dt + k2 dt^2/2
                    //  r' = r + v dt + (k1+k2+k3) dt^2/6;   v' = v + (k1+2k2+2k3+k4) dt/6
                    double k1x = fma(Uy, Bz, -(Uz * By)), k1y = fma(Uz, Bx, -(Ux * Bz)), k1z = fma(Ux, By, -(Uy * Bx));
                    tg_add_qE(P, X, Y, Z, k1x, k1y, k1z);
                    double ux = fma(k1x, P.b1, Ux), uy = fma(k1y, P.b1, Uy), uz = fma(k1z, P.b1, Uz);
                    double Xs = fma(Ux, P.a1, X), Ys = fma(Uy, P.a1, Y), Zs = fma(Uz, P.a1, Z);
                    tg_fieldXYZ<KIND, CACHED>(P, cc, reloads, Xs, Ys, Zs, t + 0.5 * P.dt, Bx, By, Bz);
                    double k2x = fma(uy, Bz, -(uz * By)), k2y = fma(uz, Bx, -(ux * Bz)), k2z = fma(ux, By, -(uy * Bx));
                    tg_add_qE(P, Xs, Ys, Zs, k2x, k2y, k2z);
                    ux = fma(k2x, P.b1, Ux); uy = fma(k2y, P.b1, Uy); uz = fma(k2z, P.b1, Uz);
                    Xs = fma(k1x, 2.0 * P.a2, fma(Ux, P.a1, X)); Ys = fma(k1y, 2.0 * P.a2, fma(Uy, P.a1, Y)); Zs = fma(k1z, 2.0 * P.a2, fma(Uz, P.a1, Z));
                    tg_fieldXYZ<KIND, CACHED>(P, cc, reloads, Xs, Ys, Zs, t + 0.5 * P.dt, Bx, By, Bz);
                    double k3x = fma(uy, Bz, -(uz * By)), k3y = fma(uz, Bx, -(ux * Bz)), k3z = fma(ux, By, -(uy * Bx));
                    tg_add_qE(P, Xs, Ys, Zs, k3x, k3y, k3z);
                    ux = fma(k3x, 2.0 * P.b1, Ux); uy = fma(k3y, 2.0 * P.b1, Uy); uz = fma(k3z, 2.0 * P.b1, Uz);
                    Xs = fma(k2x, 4.0 * P.a2, fma(Ux, 2.0 * P.a1, X)); Ys = fma(k2y, 4.0 * P.a2, fma(Uy, 2.0 * P.a1, Y)); Zs = fma(k2z, 4.0 * P.a2, fma(Uz, 2.0 * P.a1, Z));
                    tg_fieldXYZ<KIND, CACHED>(P, cc, reloads, Xs, Ys, Zs, t + P.dt, Bx, By, Bz);
                    double k4x = fma(uy, Bz, -(uz * By)), k4y = fma(uz, Bx, -(ux * Bz)), k4z = fma(ux, By, -(uy * Bx));
                    tg_add_qE(P, Xs, Ys, Zs, k4x, k4y, k4z);
                    double Tx = k2x + k3x, Ty = k2y + k3y, Tz = k2z + k3z;
                    Xn = fma(k1x + Tx, P.c6, fma(Ux, P.dtq, X)); Yn = fma(k1y + Ty, P.c6, fma(Uy, P.dtq, Y));
                    Zn = fma(k1z + Tz, P.c6, fma(Uz, P.dtq, Z));
                    Ux = fma(fma(2.0, Tx, k1x + k4x), P.d6, Ux);
                    Uy = fma(fma(2.0, Ty, k1y + k4y), P.d6, Uy);
                    Uz = fma(fma(2.0, Tz, k1z + k4z), P.d6, Uz);
                } else {
                    // ---- Eq. 7-8: Boris push with B, E at r(t0).  In u = (q/m) v units:
                    //  u- = u + eh;  t = B (q/m) h/2;  s = 2t/(1+t.t);  u* = u- + u- x t;  u+ = u- + u* x s;  u' = u+ + eh
                    double eh0 = P.eh[0], eh1 = P.eh[1], eh2 = P.eh[2];      // half kick (q/m)^2 E dt/2 with E at r(t0)
                    if (P.f.etable) {
                        double gx = 0.0, gy = 0.0, gz = 0.0;
                        tg_add_qE(P, X, Y, Z, gx, gy, gz);
                        eh0 = gx * P.b1; eh1 = gy * P.b1; eh2 = gz * P.b1;
                    }
                    auto push = [&](double hb, double he) {      // hb = (q/m) h/2, he = h/dt
                        double ax = fma(he, eh0, Ux), ay = fma(he, eh1, Uy), az = fma(he, eh2, Uz);
                        double tx = Bx * hb, ty = By * hb, tz = Bz * hb;
                        double sc = 2.0 / (1.0 + fma(tx, tx, fma(ty, ty, tz * tz)));
                        double bx = ax + fma(ay, tz, -(az * ty)), by = ay + fma(az, tx, -(ax * tz)), bz = az + fma(ax, ty, -(ay * tx));
                        double sx = tx * sc, sy = ty * sc, sz = tz * sc;
                        Ux = fma(he, eh0, ax + fma(by, sz, -(bz * sy)));
                        Uy = fma(he, eh1, ay + fma(bz, sx, -(bx * sz)));
                        Uz = fma(he, eh2, az + fma(bx, sy, -(by * sx)));
                    };
                    if (nst == 0 && P.variant == 3) push(-0.5 * P.b1, -0.5);   // leap-frog start: v(t0) -> v(t0 - dt/2)
                    double ox = Ux, oy = Uy, oz = Uz;
                    push(P.b1, 1.0);
                    if (P.variant == 4) { Xn = fma(ox, P.dtq, X); Yn = fma(oy, P.dtq, Y); Zn = fma(oz, P.dtq, Z); }   // Eq. 8 as printed
                    else { Xn = fma(Ux, P.dtq, X); Yn = fma(Uy, P.dtq, Y); Zn = fma(Uz, P.dtq, Z); }
                }
                }
                ++nst; ++ion_steps;
                double s1 = fma(P.det.normal[0], Xn, fma(P.det.normal[1], Yn, fma(P.det.normal[2], Zn, -P.nrD)));
                if (s1 >= 0.0) {               // O4: s0 < 0 <= s1 -> interpolate to the plane (L326, L338)
                    double lam = s0 / (s0 - s1);
                    [[maybe_unused]] double frac = lam;          // frac: fraction of the crossing step up to the plane (Bezier: its tau)
                    double px = fma(lam, Xn - X, X) - P.det.origin[0], py = fma(lam, Yn - Y, Y) - P.det.origin[1],
                           pz = fma(lam, Zn - Z, Z) - P.det.origin[2];
                    if constexpr (BEZ) {
                        // control point = mean of r_n + v_n dt/2 and r_n+1 - v_n+1 dt/2; root of the plane distance
                        // (1-tau)^2 s0 + 2 (1-tau) tau sc + tau^2 s1 in [0,1], cancellation-free form
                        double qx = 0.5 * (c1x + fma(-Ux, P.a1, Xn)), qy = 0.5 * (c1y + fma(-Uy, P.a1, Yn)), qz = 0.5 * (c1z + fma(-Uz, P.a1, Zn));
                        double sc = fma(P.det.normal[0], qx, fma(P.det.normal[1], qy, fma(P.det.normal[2], qz, -P.nrD)));
                        double qa = s0 - 2.0 * sc + s1, qb = 2.0 * (sc - s0), disc = fma(qb, qb, -4.0 * qa * s0), tau = lam;
                        if (disc >= 0.0) {
                            double sq = sqrt(disc);
                            tau = (qb >= 0.0) ? (-2.0 * s0) / (qb + sq) : (sq - qb) / (2.0 * qa);
                        }
                        tau = fmin(fmax(tau, 0.0), 1.0);
                        frac = tau;
                        double w0 = (1.0 - tau) * (1.0 - tau), w1 = 2.0 * (1.0 - tau) * tau, w2 = tau * tau;
                        px = fma(w0, X, fma(w1, qx, w2 * Xn)) - P.det.origin[0];
                        py = fma(w0, Y, fma(w1, qy, w2 * Yn)) - P.det.origin[1];
                        pz = fma(w0, Z, fma(w1, qz, w2 * Zn)) - P.det.origin[2];
                    }
                    P.hit_u[idx] = fma(px, P.det.eu[0], fma(py, P.det.eu[1], pz * P.det.eu[2]));
                    P.hit_w[idx] = fma(px, P.det.ew[0], fma(py, P.det.ew[1], pz * P.det.ew[2]));
                    P.cell[idx] = TAIGA_CELL_MISS;      // segment assigned by the histogram kernel (a5)
                    if constexpr (LOSS) {               // crossing step: up to the plane, nu interpolated linearly (reading L2)
                        double nun = tg_loss_rate(P, sqrt(fma(Xn, Xn, Yn * Yn)), Zn);
                        double nuh = fma(frac, nun - nu1, nu1);
                        P.weight[idx] = (P.w0 ? P.w0[idx] : 1.0) * exp(-fma(frac * P.hdt, nu1 + nuh, Lam));
                    }
                    P.steps[idx] = nst;
                    P.flags[idx] = (fabs(s0) < TG_GRAZE || fabs(s1) < TG_GRAZE) ? TAIGA_FLAG_PLANE : 0;
                    alive = false;
                }
                X = Xn; Y = Yn; Z = Zn; t += P.dt; s0 = s1;
                if constexpr (LOSS) nu0 = nu1;
            }
        }
        again = !REGROUP && __all_sync(FULL, was_alive == alive);
      } while (again);
    }
    // per-warp statistics
    unsigned long long rl = reloads, is = ion_steps;
    for (int o = 16; o > 0; o >>= 1) {
        rl += __shfl_down_sync(FULL, rl, o);
        is += __shfl_down_sync(FULL, is, o);
    }
    if (lane == 0) {
        atomicAdd(&P.counters[1], warp_steps);
        atomicAdd(&P.counters[2], rl);
        atomicAdd(&P.counters[3], is);
    }
}

// Every instantiation of k_trace, one line each: {kind, cached, registers, PRED, SOLVER, HAS_E, LOSS, BEZ, REGROUP}.
//   kind 0, RKN: register cell cache with rolling predictive refill (PRED 2; 8 x 32 threads/SM, 210 registers),
//   predictive refill after each Horner (1), refill on demand (0; the 4-evaluation solvers), 168 registers, no cache;
//   kind 1: time-blended cell cache in registers, slice difference in per-lane shared-memory slots (PRED 4, default) or
//   gathered through L1 (3), slice cache with rolling refill (2), no cache (0);
//   kind 2 with option mma = 0 or precision = 32: per-lane gathers (REGROUP: CTA re-sort by cell); the default for kind 2
//   is the warp-cooperative kernel of trace_mma.cu.
struct TgVariant { int kind, cached, regs, pred, solver, hasE, loss, bez, regroup; void (*fn)(const TraceParams); int threads; };
#define TG_V(K, C, R, P, S, E, L, B, G) {K, C, R, P, S, E, L, B, G, k_trace<K, (C) != 0, 128, R, P, S, (E) != 0, (L) != 0, (B) != 0, (G) != 0>, 128}
#define TG_VT(K, C, R, P, T) {K, C, R, P, 0, 0, 0, 0, 0, k_trace<K, (C) != 0, T, R, P, 0, false, false, false, false>, T}
