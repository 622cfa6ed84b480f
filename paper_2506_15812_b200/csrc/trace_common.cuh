// Shared by the tracer kernels (trace.cu: one lane evaluates its own cell; trace_mma.cu: the warp evaluates
// cooperatively on the FP64 tensor pipe): launch parameters and the small per-lane device helpers.
#pragma once
#include "field_device.cuh"

struct TraceParams {
    FieldDev f;
    DetDev det;
    LossDev loss;                     // secondary-ionisation loss model (LOSS kernels)
    double hdt;                       // dt/2
    double* weight;
    const double* w0;                 // initial statistical weight (null = 1)
    double nrD;                       // normal . origin
    double a1, a2, b1;                // dt/(2 qm), dt^2/8, qm dt/2   (stage 2/3)
    double c6, d6, dtq;               // dt^2/6, qm dt/6, dt/qm
    double qm, dt;
    double qE[3], eh[3];              // (q/m) E [m/s^2];  (q/m)^2 E dt/2 (Boris half kick in u units)
    double pa1R, pa1Z;                // a1/hR, a1/hZ: half-step displacement in cells per unit u (predictive refill)
    uint32_t max_steps, n;
    int variant, refill_min;
    int regroup_every;
    const double *x, *y, *z, *vx, *vy, *vz, *t0;
    const uint32_t* order;
    double *hit_u, *hit_w;
    int32_t* cell;
    uint32_t* steps;
    uint8_t* flags;
    unsigned long long* counters;     // [0] queue head, [1] warp-steps, [2] reloads / DMMA sets, [3] ion-steps
    const double* frag;               // kinds 1, 2: the table in DMMA B-fragment order (trace_mma.cu)
    int key_shift;                    // regroup sort key = cell >> key_shift (< 2^23)
    int refill_cta;                   // trace_mma: refill the CTA's free lanes once this many are free
    const double2* phi_tab;           // kind 2, trace_mma: (cos, sin) of the lower plane of each of the phi_n toroidal cells
    int phi_n;
};

#define TG_GRAZE 1e-9

__device__ __forceinline__ double tg_rsqrt(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-(a * y), y, 1.0);          // 1 - a y^2, |e| <~ 2^-22
    double q = fma(0.375, e, 0.5);
    return fma(y * e, q, y);                   // y (1 + e/2 + 3 e^2/8): cubic convergence
}

// 1/sqrt(a) and sqrt(a) together; the square root comes off the same correction one dependent operation earlier
// (sqrt(a) = t (1 + e q) with t = a y), which is what the cell coordinate of the next Horner sum waits for
__device__ __forceinline__ double tg_rsqrt_sqrt(double a, double& root) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double t = a * y;
    double e = fma(-t, y, 1.0);
    double q = fma(0.375, e, 0.5);
    root = fma(t * e, q, t);
    return fma(y * e, q, y);
}

// EARLY: the form above (kind 0: 31.62 -> 31.53 ms on BASELINE config 2); otherwise sqrt(a) = a / sqrt(a) after the correction,
// one instruction fewer (the kind-1 kernel sits at the register limit and is 7 % slower with the early form)
template <bool EARLY>
__device__ __forceinline__ double tg_rsq(double a, double& root) {
    if constexpr (EARLY) return tg_rsqrt_sqrt(a, root);
    else { const double y = tg_rsqrt(a); root = a * y; return y; }
}

// t in [0,1)  <=>  sign 0 and exponent < 1023  <=>  (unsigned) hi word < 0x3FF00000
__device__ __forceinline__ bool tg_in01(double t) { return (unsigned)__double2hiint(t) < 0x3FF00000u; }

// O0: B_X = B_R c - B_phi s, B_Y = B_R s + B_phi c
__device__ __forceinline__ void tg_rotate(double X, double Y, double rinv, double BR, double Bp, double& Bx, double& By) {
    double c = X * rinv, s_ = Y * rinv;
    Bx = fma(BR, c, -(Bp * s_));
    By = fma(BR, s_, Bp * c);
}

// Acceleration (q/m) E(r) of Eq. 3 added to (ax, ay, az): the uniform field (P.qE) plus, when loaded, the gridded
// E_R, E_Z, E_phi of taiga_load_efield: located and gathered per evaluation (boundary cell extrapolates), rotated to
// Cartesian components like B (O0).  PAPER.md L172-177, reading E1.
__device__ __forceinline__ void tg_add_qE(const TraceParams& P, double Xs, double Ys, double Zs, double& ax, double& ay, double& az) {
    double ex = P.qE[0], ey = P.qE[1], ez = P.qE[2];
    if (P.f.etable) {
        const double R2 = fma(Xs, Xs, Ys * Ys), ri = tg_rsqrt(R2), Rs = R2 * ri;
        double p, w;
        const int i = tg_locate(Rs, P.f.inv_hR, P.f.offR, P.f.cR, p);
        const int j = tg_locate(Zs, P.f.inv_hZ, P.f.offZ, P.f.cZ, w);
        const double* c = P.f.etable + ((size_t)i * P.f.cZ + j) * 48;
        const double eR = tg_bicubic(c, p, w), eZ = tg_bicubic(c + 16, p, w), eP = tg_bicubic(c + 32, p, w);
        double gx, gy;
        tg_rotate(Xs, Ys, ri, eR, eP, gx, gy);
        ex = fma(P.qm, gx, ex); ey = fma(P.qm, gy, ey); ez = fma(P.qm, eZ, ez);
    }
    ax += ex; ay += ey; az += ez;
}

// nu(psi(R,Z)): psi from its bicubic table (boundary cell extrapolates), the rate
// profile linear in psi between its points, held constant outside.
__device__ __forceinline__ double tg_loss_rate(const TraceParams& P, double R, double Z) {
    double p, w;
    int i = tg_locate(R, P.f.inv_hR, P.f.offR, P.f.cR, p);
    int j = tg_locate(Z, P.f.inv_hZ, P.f.offZ, P.f.cZ, w);
    double psi = tg_bicubic(P.loss.psi + ((size_t)i * P.f.cZ + j) * 48, p, w);
    double x = (psi - P.loss.psi0) * P.loss.inv_dpsi;
    if (!(x > 0.0)) return __ldg(P.loss.rate);
    if (x >= (double)(P.loss.n - 1)) return __ldg(P.loss.rate + P.loss.n - 1);
    int k = __double2int_rd(x);
    double r0 = __ldg(P.loss.rate + k), r1 = __ldg(P.loss.rate + k + 1);
    return fma(x - (double)k, r1 - r0, r0);
}

