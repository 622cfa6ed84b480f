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
// threads, latency bound) the band of H is built once per line length on the host (O(n^2), by
// running the reduction above on unit vectors) and every node is then an independent 73-point
// stencil: one thread per node, coalesced, exact to rounding.  One thread per (cell, component)
// finally assembles the 16 power-basis coefficients from {y, y_zz, y_rr, y_rrzz} at 4 corners.
#include <vector>

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

// host: band of H for line length n (Thomas reduction applied to unit vectors)
static std::vector<double> spline_band(int n) {
    std::vector<double> band((size_t)(2 * TG_BAND_W + 1) * n, 0.0), cp(n, 0.0), M(n), y(n);
    for (int i = 2; i <= n - 3; ++i) cp[i] = (i == 2) ? 0.25 : 1.0 / (4.0 - cp[i - 1]);
    for (int q = 0; q < n; ++q) {
        // response to y = e_q is non-negligible only for |i-q| <= W (+2 for the end rows); solve on a window
        int lo = q - TG_BAND_W - 3, hi = q + TG_BAND_W + 3;
        if (lo < 0) lo = 0;
        if (hi > n - 1) hi = n - 1;
        auto Y = [&](int i) { return i == q ? 1.0 : 0.0; };
        auto d2 = [&](int i) { return (Y(i - 1) - 2.0 * Y(i)) + Y(i + 1); };
        // full-length solve restricted to rows where the right-hand side can be non-zero is not
        // possible for a tridiagonal system, so solve the whole line (O(n) per column, O(n^2) total)
        double M1 = d2(1), Mn2 = d2(n - 2), dprev = 0.0;
        std::fill(M.begin(), M.end(), 0.0);
        M[1] = M1; M[n - 2] = Mn2;
        for (int i = 2; i <= n - 3; ++i) {
            double rhs = 6.0 * d2(i);
            if (i == 2) rhs -= M1;
            if (i == n - 3) rhs -= Mn2;
            double dp = (i == 2) ? rhs * cp[i] : (rhs - dprev) * cp[i];
            M[i] = dp; dprev = dp;
        }
        for (int i = n - 4; i >= 2; --i) M[i] = M[i] - cp[i] * M[i + 1];
        M[0] = 2.0 * M[1] - M[2];
        M[n - 1] = 2.0 * M[n - 2] - M[n - 3];
        for (int i = lo; i <= hi; ++i) {
            int d = q - i + TG_BAND_W;
            if (d >= 0 && d <= 2 * TG_BAND_W) band[(size_t)d * n + i] = M[i];
        }
    }
    return band;
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

// first column of inverse of circulant(4,1,0,...,0,1), by Gaussian elimination (n <= 128)
static std::vector<double> circulant_inverse_col(int n) {
    std::vector<double> A((size_t)n * n, 0.0), x(n, 0.0);
    for (int i = 0; i < n; ++i) { A[(size_t)i * n + i] += 4.0; A[(size_t)i * n + (i + 1) % n] += 1.0; A[(size_t)i * n + (i + n - 1) % n] += 1.0; }
    x[0] = 1.0;
    for (int c = 0; c < n; ++c)                   // diagonally dominant: no pivoting needed
        for (int r = c + 1; r < n; ++r) {
            double f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
            if (f == 0.0) continue;
            for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= f * A[(size_t)c * n + k];
            x[r] -= f * x[c];
        }
    for (int r = n - 1; r >= 0; --r) {
        double s = x[r];
        for (int k = r + 1; k < n; ++k) s -= A[(size_t)r * n + k] * x[k];
        x[r] = s / A[(size_t)r * n + r];
    }
    return x;
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
    } else {
        // scratch: y[3] | Mz[3] | Myr[3] | Mzr[3] (3 components) | temp bicubic (kind 2) | G
        size_t n_tmp = (g->kind == 2) ? (size_t)ncell * nS * 48 : 0;
        size_t need = 12 * (size_t)nnode + n_tmp + TG_MAX_PLANES, scap = ctx->scratch_bytes / sizeof(double);
        rc = tg_reserve(ctx, &ctx->scratch, &scap, need);
        ctx->scratch_bytes = scap * sizeof(double);
        if (rc) return rc;
        double *y = ctx->scratch, *Mz = y + 3 * nnode, *Myr = Mz + 3 * nnode, *Mzr = Myr + 3 * nnode;
        double *tmp = Mzr + 3 * nnode, *G = tmp + n_tmp;
        // band operators, cached per line length
        for (int ax = 0; ax < 2; ++ax) {
            int n = ax ? nR : nZ;
            if (ctx->band_n[ax] != n) {
                std::vector<double> b = spline_band(n);
                size_t cap = ctx->band_cap[ax];
                rc = tg_reserve(ctx, &ctx->band[ax], &cap, b.size());
                ctx->band_cap[ax] = cap;
                if (rc) return rc;
                TG_CUDA(ctx, cudaMemcpyAsync(ctx->band[ax], b.data(), b.size() * sizeof(double), cudaMemcpyHostToDevice, st));
                TG_CUDA(ctx, cudaStreamSynchronize(st));
                ctx->band_n[ax] = n;
            }
        }
        if (g->kind == 2) {
            std::vector<double> Gh = circulant_inverse_col(nS);
            TG_CUDA(ctx, cudaMemcpyAsync(G, Gh.data(), nS * sizeof(double), cudaMemcpyHostToDevice, st));
            TG_CUDA(ctx, cudaStreamSynchronize(st));
        }
        for (int m = 0; m < 3; ++m)
            TG_CUDA(ctx, cudaMemcpyAsync(y + (size_t)m * nnode, src[m], nnode * sizeof(double),
                                         c->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
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
    f.table = ctx->table; f.table32 = nullptr; f.dtable = nullptr;
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
    for (int ax = 0; ax < 2; ++ax) {                 // band operators (normally cached by load_field)
        int n = ax ? nR : nZ;
        if (ctx->band_n[ax] != n) {
            std::vector<double> b = spline_band(n);
            size_t cap = ctx->band_cap[ax];
            rc = tg_reserve(ctx, &ctx->band[ax], &cap, b.size());
            ctx->band_cap[ax] = cap;
            if (rc) return rc;
            TG_CUDA(ctx, cudaMemcpyAsync(ctx->band[ax], b.data(), b.size() * sizeof(double), cudaMemcpyHostToDevice, st));
            TG_CUDA(ctx, cudaStreamSynchronize(st));
            ctx->band_n[ax] = n;
        }
    }
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
