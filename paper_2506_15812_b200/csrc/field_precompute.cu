// a1: field-coefficient precompute.  Interpolating tensor-product cubic
// spline, not-a-knot in R and Z, periodic in phi (kind 2).
//
// not-a-knot on a unit-spaced line, unknowns M_i = S''(x_i):
//   M_{i-1} + 4 M_i + M_{i+1} = 6 (y_{i-1} - 2 y_i + y_{i+1}),   i = 1..n-2
//   M_0 - 2 M_1 + M_2 = 0   =>  substituting into row 1:  M_1 = y_0 - 2 y_1 + y_2
//   (same at the far end), so the system is tridiagonal in M_2..M_{n-3} with known ends.
// The map y -> M is linear, M = H y, and because the (1,4,1) system is diagonally dominant the
// entries of H decay like (2-sqrt 3)^|i-j| = 0.268^|i-j|: beyond |i-j| = 36 they are below
// 3e-21 of the diagonal.  So instead of one serial Thomas solve per grid line (a few hundred
// threads, latency bound) the band of H is built once per line length on the device (k_spline_band:
// one thread per column runs the reduction above on a unit vector) and every node is then an independent 73-point
// stencil: one thread per node, coalesced, exact to rounding.  One thread per (cell, component)
// finally assembles the 16 power-basis coefficients from {y, y_zz, y_rr, y_rrzz} at 4 corners.
#include "field_device.cuh"

#define TG_BAND_W 36

// M[t] = sum_q H[i][q] y[q] along one grid direction.  band[(q-i+W)*n + i] = H[i][q].
// `stride`: distance between consecutive nodes of a line; i = (t / stride) % n.
__global__ void k_second_deriv(const double* __restrict__ y, double* __restrict__ M, const double* __restrict__ band,
                               int n, long long stride, long long total) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= total) return;
    int i = (int)((t / stride) % n);
    int lo = max(0, i - TG_BAND_W), hi = min(n - 1, i + TG_BAND_W);
    double acc = 0.0;
    for (int q = lo; q <= hi; ++q)
        acc = fma(band[(size_t)(q - i + TG_BAND_W) * n + i], y[t + (long long)(q - i) * stride], acc);
    M[t] = acc;
}

// Band of H for line length n, built on the device: thread q solves the system for y = e_q.  The response decays like
// 0.268^|i-q|, so the tridiagonal solve runs on the window |i - q| <= W + TG_BAND_MARGIN only (M = 0 beyond it: an error
// below 0.268^(W + margin) ~ 1e-35 of the diagonal on the rows that are kept); windows that reach a grid end use the
// exact not-a-knot rows  M_1 = d2(1), M_0 = 2 M_1 - M_2  (and their mirror images).
#define TG_BAND_MARGIN 24
#define TG_BAND_WIN (2 * (TG_BAND_W + TG_BAND_MARGIN) + 8)
__global__ void k_spline_band(double* __restrict__ band, int n) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int lo = max(0, q - TG_BAND_W - TG_BAND_MARGIN), hi = min(n - 1, q + TG_BAND_W + TG_BAND_MARGIN);
    double M[TG_BAND_WIN], cp[TG_BAND_WIN];
    auto Y = [&](int i) { return i == q ? 1.0 : 0.0; };
    auto d2 = [&](int i) { return (Y(i - 1) - 2.0 * Y(i)) + Y(i + 1); };
    for (int i = lo; i <= hi; ++i) M[i - lo] = 0.0;
    const double M1 = d2(1), Mn2 = d2(n - 2);                       // exact end rows (zero unless q is within 2 of that end)
    const int a = max(lo, 2), b = min(hi, n - 3);                   // unknowns of the (1,4,1) rows
    double dprev = 0.0, cprev = 0.0;
    for (int i = a; i <= b; ++i) {                                  // Thomas, forward
        double rhs = 6.0 * d2(i);
        if (i == 2) rhs -= M1;
        if (i == n - 3) rhs -= Mn2;
        const double c = (i == a) ? 0.25 : 1.0 / (4.0 - cprev);
        const double dp = (i == a) ? rhs * c : (rhs - dprev) * c;
        cp[i - lo] = c; M[i - lo] = dp; dprev = dp; cprev = c;
    }
    for (int i = b - 1; i >= a; --i) M[i - lo] = M[i - lo] - cp[i - lo] * M[i + 1 - lo];
    if (lo <= 1 && 1 <= hi) M[1 - lo] = M1;
    if (lo <= n - 2 && n - 2 <= hi) M[n - 2 - lo] = Mn2;
    if (lo == 0) M[0] = 2.0 * M[1 - lo] - M[2 - lo];
    if (hi == n - 1) M[n - 1 - lo] = 2.0 * M[n - 2 - lo] - M[n - 3 - lo];
    for (int i = max(0, q - TG_BAND_W); i <= min(n - 1, q + TG_BAND_W); ++i)
        band[(size_t)(q - i + TG_BAND_W) * n + i] = M[i - lo];
}

// band operator of one grid direction (ax 0: Z, 1: R), cached per line length; no host work, no synchronisation
static int tg_ensure_band(taiga_ctx* ctx, int ax, int n) {
    if (ctx->band_n[ax] == n) return TAIGA_OK;
    size_t cap = ctx->band_cap[ax], need = (size_t)(2 * TG_BAND_W + 1) * n;
    int rc = tg_reserve(ctx, &ctx->band[ax], &cap, need);
    ctx->band_cap[ax] = cap;
    if (rc) return rc;
    TG_CUDA(ctx, cudaMemsetAsync(ctx->band[ax], 0, need * sizeof(double), ctx->stream));
    k_spline_band<<<(n + 63) / 64, 64, 0, ctx->stream>>>(ctx->band[ax], n);
    TG_CUDA(ctx, cudaGetLastError());
    ctx->band_n[ax] = n;
    return TAIGA_OK;
}

// kind 2: first column G of the inverse of the circulant (1,4,1) matrix of the periodic spline, closed form: with
// r = sqrt(3) - 2 (root of r^2 + 4 r + 1) the infinite chain has g_k = r^|k| / (2 sqrt 3); summing the periodic images
// gives G_k = (r^k + r^(n-k)) / ((1 - r^n) 2 sqrt 3) = G_(n-k).  Both powers come from the same forward products r^k, which
// fade to zero far from the diagonal (the right value to rounding) instead of being divided back up from r^n (which
// loses digits as n grows and underflows at n ~ 540; taiga_load_field takes n <= TG_MAX_PLANES = 128 anyway).
__global__ void k_circulant_inverse_col(double* __restrict__ G, int n) {
    if (blockIdx.x || threadIdx.x) return;
    const double s3 = sqrt(3.0), r = s3 - 2.0;
    double up = 1.0;
    for (int k = 0; k < n; ++k) { G[k] = up; up *= r; }             // r^k; up ends as r^n
    const double norm = 1.0 / ((1.0 - up) * 2.0 * s3);
    G[0] = (1.0 + up) * norm;
    for (int k = 1; 2 * k <= n; ++k) { const double v = (G[k] + G[n - k]) * norm; G[k] = v; G[n - k] = v; }
}

// power-basis coefficients of one interval from end values g0,g1 and end second derivatives G0,G1
__device__ __forceinline__ void seg_coef(double g0, double g1, double G0, double G1, double c[4]) {
    c[0] = g0;
    c[1] = (g1 - g0) - (2.0 * G0 + G1) / 6.0;
    c[2] = G0 / 2.0;
    c[3] = (G1 - G0) / 6.0;
}

// thread per (slice, cell, comp).  nodal arrays of one component: 4 planes of [nS][nR][nZ].
// out index by `mode`: 0 -> kind-0/1 internal layout, 1 -> temp layout [k][cell][comp][16] for kind 2
__global__ void k_assemble(const double* __restrict__ y, const double* __restrict__ Mz, const double* __restrict__ Myr,
                           const double* __restrict__ Mzr, double* __restrict__ out, int nS, int nR, int nZ,
                           int comp, int mode) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int cR = nR - 1, cZ = nZ - 1;
    long long ncell = (long long)cR * cZ;
    if (t >= ncell * nS) return;
    int k = (int)(t / ncell);
    long long cell = t % ncell;
    int i = (int)(cell / cZ), j = (int)(cell % cZ);
    long long n00 = ((long long)k * nR + i) * nZ + j, n10 = n00 + nZ;
    double cz[2][4], Dz[2][4];                 // w-coefficients of y and of y_rr at R-nodes i, i+1
    seg_coef(y[n00], y[n00 + 1], Mz[n00], Mz[n00 + 1], cz[0]);
    seg_coef(y[n10], y[n10 + 1], Mz[n10], Mz[n10 + 1], cz[1]);
    seg_coef(Myr[n00], Myr[n00 + 1], Mzr[n00], Mzr[n00 + 1], Dz[0]);
    seg_coef(Myr[n10], Myr[n10 + 1], Mzr[n10], Mzr[n10 + 1], Dz[1]);
    double* o = (mode == 0) ? out + ((cell * nS + k) * 3 + comp) * 16
                            : out + (((long long)k * ncell + cell) * 3 + comp) * 16;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        double ca[4];
        seg_coef(cz[0][b], cz[1][b], Dz[0][b], Dz[1][b], ca);
#pragma unroll
        for (int a = 0; a < 4; ++a) o[a * 4 + b] = ca[a];
    }
}

// kind 2: periodic spline in phi of every bicubic coefficient.  G = first column of the inverse
// of the circulant (1,4,1) matrix.  thread per (cell, comp, ab).
#define TG_MAX_PLANES 128
__global__ void k_phi_spline(const double* __restrict__ bic, const double* __restrict__ G, double* __restrict__ out,
                             int nS, long long ncell) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncell * 48) return;
    long long cell = t / 48;
    int comp = (int)((t % 48) / 16), ab = (int)(t % 16);
    double c[TG_MAX_PLANES], rhs[TG_MAX_PLANES];
    for (int k = 0; k < nS; ++k) c[k] = bic[(((long long)k * ncell + cell) * 3 + comp) * 16 + ab];
    for (int k = 0; k < nS; ++k) rhs[k] = 6.0 * ((c[(k + nS - 1) % nS] - 2.0 * c[k]) + c[(k + 1) % nS]);
    double Mprev = 0.0, M0 = 0.0;
    for (int kk = 0; kk <= nS; ++kk) {          // M_k for k = 0..nS (M_nS = M_0), emit interval k-1
        int k = kk % nS;
        double M = 0.0;
        for (int m = 0; m < nS; ++m) M = fma(G[(k - m + nS) % nS], rhs[m], M);
        if (kk == 0) M0 = M;
        if (kk == nS) M = M0;
        if (kk > 0) {
            double d[4];
            seg_coef(c[kk - 1], c[k], Mprev, M, d);
            double* o = out + (((long long)(kk - 1) * ncell + cell) * 3 + comp) * 64;
#pragma unroll
            for (int e = 0; e < 4; ++e) o[e * 16 + ab] = d[e];
        }
        Mprev = M;
    }
}

// form-1 input (per-cell coefficients [nS][cell][per]) <-> internal layout
__global__ void k_relayout(const double* __restrict__ src, double* __restrict__ dst, int kind, int nS, long long ncell,
                           int comp, int to_internal) {
    int per = (kind == 2) ? 64 : 16;
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncell * nS * per) return;
    int e = (int)(t % per);
    long long cell = (t / per) % ncell;
    int k = (int)(t / per / ncell);
    long long in = (kind == 2) ? (((long long)k * ncell + cell) * 3 + comp) * 64 + e
                               : ((cell * nS + k) * 3 + comp) * 16 + e;
    if (to_internal) dst[in] = src[t]; else dst[t] = src[in];
}

__global__ void k_field_eval(FieldDev f, unsigned long long n, const double* R, const double* Z, const double* s,
                             double* BR, double* BZ, double* Bp) {
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double a, b, c;
    tg_field_cyl(f, R[i], Z[i], s ? s[i] : 0.0, a, b, c);
    BR[i] = a; BZ[i] = b; Bp[i] = c;
}

// kind 1: D[cell][k] = T[cell][k+1] - T[cell][k], so that B(t) = H(T_k) + tau H(D_k) and the tracer can keep
// T_k in registers and gather only D_k (half the bytes of gathering both slices)
__global__ void k_slice_diff(const double* __restrict__ T, double* __restrict__ D, long long ncell, int nS) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long tot = ncell * (nS - 1) * 48;
    if (t >= tot) return;
    int e = (int)(t % 48);
    long long ck = t / 48, cell = ck / (nS - 1);
    int k = (int)(ck % (nS - 1));
    const double* a = T + ((cell * nS + k) * 48 + e);
    D[t] = a[48] - a[0];
}

// kind 1, register-cached kernel only (trace.cu): the slice differences, built on first use
int tg_build_dtable(taiga_ctx* ctx) {
    FieldDev& f = ctx->field;
    if (ctx->dtable_valid) { f.dtable = ctx->dtable; return TAIGA_OK; }
    const long long ncell = (long long)f.cR * f.cZ;
    size_t nd = (size_t)ncell * (f.nS - 1) * 48;
    int rc = tg_reserve(ctx, &ctx->dtable, &ctx->cap_dtable, nd);
    if (rc) return rc;
    k_slice_diff<<<(unsigned)((nd + 255) / 256), 256, 0, ctx->stream>>>(ctx->table, ctx->dtable, ncell, f.nS);
    TG_CUDA(ctx, cudaGetLastError());
    f.dtable = ctx->dtable; ctx->dtable_valid = true;
    return TAIGA_OK;
}

int tg_precompute(taiga_ctx* ctx, const taiga_grid* g, const taiga_coeffs* c) {
    const int nR = g->nR, nZ = g->nZ, nS = g->nS, cR = nR - 1, cZ = nZ - 1;
    const long long ncell = (long long)cR * cZ, nnode = (long long)nS * nR * nZ;
    const int per = (g->kind == 2) ? 64 : 16;
    if (g->kind == 2 && nS > TG_MAX_PLANES) { TG_SET_ERR(ctx, "kind 2: nS <= %d", TG_MAX_PLANES); return TAIGA_E_ARG; }
    size_t table_n = (size_t)ncell * nS * 3 * per;
    size_t tcap = ctx->table_bytes / sizeof(double);
    int rc = tg_reserve(ctx, &ctx->table, &tcap, table_n);
    ctx->table_bytes = tcap * sizeof(double);
    if (rc) return rc;
    cudaStream_t st = ctx->stream;
    const double* src[3] = {c->BR, c->BZ, c->Bphi};
    const int TPB = 128;

    if (c->form == 1) {
        size_t need = (size_t)ncell * nS * per, scap = ctx->scratch_bytes / sizeof(double);
        if (!c->on_device) { rc = tg_reserve(ctx, &ctx->scratch, &scap, need); ctx->scratch_bytes = scap * sizeof(double); if (rc) return rc; }
        for (int m = 0; m < 3; ++m) {
            const double* s = src[m];
            if (!c->on_device) { TG_CUDA(ctx, cudaMemcpyAsync(ctx->scratch, src[m], need * sizeof(double), cudaMemcpyHostToDevice, st)); s = ctx->scratch; }
            k_relayout<<<(unsigned)((need + TPB - 1) / TPB), TPB, 0, st>>>(s, ctx->table, g->kind, nS, ncell, m, 1);
        }
        if (!c->on_device) TG_CUDA(ctx, cudaStreamSynchronize(st));      // host arrays: read during the call only
    } else {
        // scratch: y[3] | Mz[3] | Myr[3] | Mzr[3] (3 components) | temp bicubic (kind 2) | G
        size_t n_tmp = (g->kind == 2) ? (size_t)ncell * nS * 48 : 0;
        size_t need = 12 * (size_t)nnode + n_tmp + TG_MAX_PLANES, scap = ctx->scratch_bytes / sizeof(double);
        rc = tg_reserve(ctx, &ctx->scratch, &scap, need);
        ctx->scratch_bytes = scap * sizeof(double);
        if (rc) return rc;
        double *y = ctx->scratch, *Mz = y + 3 * nnode, *Myr = Mz + 3 * nnode, *Mzr = Myr + 3 * nnode;
        double *tmp = Mzr + 3 * nnode, *G = tmp + n_tmp;
        // band operators, cached per line length (device-built)
        for (int ax = 0; ax < 2; ++ax) { rc = tg_ensure_band(ctx, ax, ax ? nR : nZ); if (rc) return rc; }
        if (g->kind == 2) { k_circulant_inverse_col<<<1, 32, 0, st>>>(G, nS); TG_CUDA(ctx, cudaGetLastError()); }
        for (int m = 0; m < 3; ++m)
            TG_CUDA(ctx, cudaMemcpyAsync(y + (size_t)m * nnode, src[m], nnode * sizeof(double),
                                         c->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
        // host arrays are "read during the call only" (taiga.h): a copy from pinned or registered host memory is truly
        // asynchronous, so wait for it here; device inputs (the timed paths) are not synchronised
        if (!c->on_device) TG_CUDA(ctx, cudaStreamSynchronize(st));
        long long tot = 3 * nnode;
        unsigned gb = (unsigned)((tot + TPB - 1) / TPB);
        k_second_deriv<<<gb, TPB, 0, st>>>(y, Mz, ctx->band[0], nZ, 1, tot);          // y_zz
        k_second_deriv<<<gb, TPB, 0, st>>>(y, Myr, ctx->band[1], nR, nZ, tot);        // y_rr
        k_second_deriv<<<gb, TPB, 0, st>>>(Mz, Mzr, ctx->band[1], nR, nZ, tot);       // y_rrzz
        for (int m = 0; m < 3; ++m) {
            long long nt = ncell * nS;
            size_t o = (size_t)m * nnode;
            k_assemble<<<(unsigned)((nt + TPB - 1) / TPB), TPB, 0, st>>>(y + o, Mz + o, Myr + o, Mzr + o,
                                                                      g->kind == 2 ? tmp : ctx->table, nS, nR, nZ, m,
                                                                      g->kind == 2 ? 1 : 0);
        }
        if (g->kind == 2) {
            long long nt = ncell * 48;
            k_phi_spline<<<(unsigned)((nt + TPB - 1) / TPB), TPB, 0, st>>>(tmp, G, ctx->table, nS, ncell);
        }
    }
    TG_CUDA(ctx, cudaGetLastError());
    FieldDev& f = ctx->field;
    f.kind = g->kind; f.nR = nR; f.nZ = nZ; f.nS = nS; f.cR = cR; f.cZ = cZ;
    f.Rmin = g->Rmin; f.Rmax = g->Rmax; f.Zmin = g->Zmin; f.Zmax = g->Zmax;
    double hR = (g->Rmax - g->Rmin) / cR, hZ = (g->Zmax - g->Zmin) / cZ;
    f.inv_hR = 1.0 / hR; f.inv_hZ = 1.0 / hZ;
    f.offR = g->Rmin / hR; f.offZ = g->Zmin / hZ;
    f.s0 = g->s0; f.inv_ds = (g->kind == 0) ? 0.0 : 1.0 / g->ds;
    f.table = ctx->table; f.table32 = nullptr; f.dtable = nullptr; f.etable = nullptr;
    return TAIGA_OK;
}

// Eq. 2: nu = n_e sqrt(t) exp(-1/t) / (E12^1.5 (6 + t)) 1e-11 m^3/s, t = T_e / E12
__global__ void k_mcwhirter(const double* __restrict__ ne, const double* __restrict__ Te, double E12, int n, double* __restrict__ rate) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double T = Te[k], r = 0.0;
    if (T > 0.0) {
        double t = T / E12;
        r = ne[k] * (sqrt(t) * exp(-1.0 / t) / (E12 * sqrt(E12) * (6.0 + t))) * 1e-11;
    }
    rate[k] = r;
}

// psi(R,Z): the a1 spline machinery on one more scalar (same band operators, kind-0 cell layout).
int tg_load_loss(taiga_ctx* ctx, const double* psi_nodal, int on_device, const taiga_loss_profile* prof) {
    const FieldDev& f = ctx->field;
    const int nR = f.nR, nZ = f.nZ;
    const long long nnode = (long long)nR * nZ, ncell = (long long)f.cR * f.cZ;
    cudaStream_t st = ctx->stream;
    const int TPB = 128;
    int rc = tg_reserve(ctx, &ctx->psi_table, &ctx->cap_psi, (size_t)ncell * 48);
    if (rc) return rc;
    rc = tg_reserve(ctx, &ctx->loss_rate, &ctx->cap_rate, (size_t)prof->n);
    if (rc) return rc;
    size_t need = 4 * (size_t)nnode + 2 * (size_t)prof->n, scap = ctx->scratch_bytes / sizeof(double);
    rc = tg_reserve(ctx, &ctx->scratch, &scap, need);
    ctx->scratch_bytes = scap * sizeof(double);
    if (rc) return rc;
    double *y = ctx->scratch, *Mz = y + nnode, *Myr = Mz + nnode, *Mzr = Myr + nnode, *pne = Mzr + nnode, *pte = pne + prof->n;
    for (int ax = 0; ax < 2; ++ax) { rc = tg_ensure_band(ctx, ax, ax ? nR : nZ); if (rc) return rc; }   // normally cached by load_field
    TG_CUDA(ctx, cudaMemcpyAsync(y, psi_nodal, nnode * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    TG_CUDA(ctx, cudaMemcpyAsync(pne, prof->ne_m3, prof->n * sizeof(double), cudaMemcpyHostToDevice, st));
    TG_CUDA(ctx, cudaMemcpyAsync(pte, prof->Te_eV, prof->n * sizeof(double), cudaMemcpyHostToDevice, st));
    unsigned gb = (unsigned)((nnode + TPB - 1) / TPB);
    k_second_deriv<<<gb, TPB, 0, st>>>(y, Mz, ctx->band[0], nZ, 1, nnode);
    k_second_deriv<<<gb, TPB, 0, st>>>(y, Myr, ctx->band[1], nR, nZ, nnode);
    k_second_deriv<<<gb, TPB, 0, st>>>(Mz, Mzr, ctx->band[1], nR, nZ, nnode);
    k_assemble<<<(unsigned)((ncell + TPB - 1) / TPB), TPB, 0, st>>>(y, Mz, Myr, Mzr, ctx->psi_table, 1, nR, nZ, 0, 0);
    k_mcwhirter<<<(prof->n + TPB - 1) / TPB, TPB, 0, st>>>(pne, pte, prof->E12_eV, prof->n, ctx->loss_rate);
    TG_CUDA(ctx, cudaGetLastError());
    TG_CUDA(ctx, cudaStreamSynchronize(st));          // host profile arrays may be freed by the caller
    ctx->loss.psi = ctx->psi_table; ctx->loss.rate = ctx->loss_rate; ctx->loss.n = prof->n;
    ctx->loss.psi0 = prof->psi0; ctx->loss.inv_dpsi = 1.0 / prof->dpsi;
    return TAIGA_OK;
}

// Gridded electric field (taiga_load_efield): three static 2-D components on the loaded grid, the kind-0 table layout,
// built by the same stencil and assembly kernels as B.
int tg_load_efield(taiga_ctx* ctx, const taiga_coeffs* c) {
    FieldDev& f = ctx->field;
    if (!c) { f.etable = nullptr; return TAIGA_OK; }
    const int nR = f.nR, nZ = f.nZ;
    const long long nnode = (long long)nR * nZ, ncell = (long long)f.cR * f.cZ;
    cudaStream_t st = ctx->stream;
    const int TPB = 128;
    int rc = tg_reserve(ctx, &ctx->etable, &ctx->cap_etable, (size_t)ncell * 48);
    if (rc) return rc;
    size_t need = 12 * (size_t)nnode, scap = ctx->scratch_bytes / sizeof(double);
    rc = tg_reserve(ctx, &ctx->scratch, &scap, need);
    ctx->scratch_bytes = scap * sizeof(double);
    if (rc) return rc;
    double *y = ctx->scratch, *Mz = y + 3 * nnode, *Myr = Mz + 3 * nnode, *Mzr = Myr + 3 * nnode;
    for (int ax = 0; ax < 2; ++ax) { rc = tg_ensure_band(ctx, ax, ax ? nR : nZ); if (rc) return rc; }
    const double* src[3] = {c->BR, c->BZ, c->Bphi};
    for (int m = 0; m < 3; ++m)
        TG_CUDA(ctx, cudaMemcpyAsync(y + (size_t)m * nnode, src[m], nnode * sizeof(double),
                                     c->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    long long tot = 3 * nnode;
    unsigned gb = (unsigned)((tot + TPB - 1) / TPB);
    k_second_deriv<<<gb, TPB, 0, st>>>(y, Mz, ctx->band[0], nZ, 1, tot);
    k_second_deriv<<<gb, TPB, 0, st>>>(y, Myr, ctx->band[1], nR, nZ, tot);
    k_second_deriv<<<gb, TPB, 0, st>>>(Mz, Mzr, ctx->band[1], nR, nZ, tot);
    for (int m = 0; m < 3; ++m) {
        size_t o = (size_t)m * nnode;
        k_assemble<<<(unsigned)((ncell + TPB - 1) / TPB), TPB, 0, st>>>(y + o, Mz + o, Myr + o, Mzr + o, ctx->etable, 1, nR, nZ, m, 0);
    }
    TG_CUDA(ctx, cudaGetLastError());
    if (!c->on_device) TG_CUDA(ctx, cudaStreamSynchronize(st));      // pageable or pinned host arrays may be reused by the caller
    f.etable = ctx->etable;
    return TAIGA_OK;
}

int tg_field_eval(taiga_ctx* ctx, uint64_t n, const double* R, const double* Z, const double* s, double* BR, double* BZ, double* Bp) {
    k_field_eval<<<(unsigned)((n + 127) / 128), 128, 0, ctx->stream>>>(ctx->field, n, R, Z, s, BR, BZ, Bp);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}

int tg_field_table(taiga_ctx* ctx, int comp, double* host) {
    const FieldDev& f = ctx->field;
    int per = (f.kind == 2) ? 64 : 16;
    long long ncell = (long long)f.cR * f.cZ;
    size_t need = (size_t)ncell * f.nS * per;
    double* tmp = nullptr;
    TG_CUDA(ctx, cudaMalloc((void**)&tmp, need * sizeof(double)));
    k_relayout<<<(unsigned)((need + 127) / 128), 128, 0, ctx->stream>>>(ctx->table, tmp, f.kind, f.nS, ncell, comp, 0);
    cudaError_t e = cudaMemcpyAsync(host, tmp, need * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(tmp);
    TG_CUDA(ctx, e);
    return TAIGA_OK;
}
