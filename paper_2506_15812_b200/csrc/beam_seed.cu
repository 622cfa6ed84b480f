// a2: beam seeding (PAPER.md L314 stochastic initialisation on the GPU; L128-134 linear beam
// model).  One thread per ion; counter-based Philox4x32-10 keyed by (seed, global ion index) so
// the result is independent of launch geometry and sharding; every draw is a tabulated-CDF
// inversion using only +,-,*,/,fma,sqrt (IEEE, explicitly rounded intrinsics so that nvcc
// never contracts them): bit-identical on any IEEE-754 machine.
#include "taiga_internal.h"

struct SeedParams {
    double v0, origin[3], axis[3], eT[3], eZ[3];
    const double* cdf_depth;  int n_depth;  double depth_max;
    const double* cdf_normal; int n_normal; double z_max;
    double sigma_pos, sigma_ang;
    unsigned long long first_index, seed, n;
    unsigned short group; double t0;
    int profile; double radius;
};

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 52-bit uniform in (0,1): ((w0>>6)*2^26 + (w1>>6) + 0.5) * 2^-52, exact in fp64
__device__ __forceinline__ double u52(uint32_t w0, uint32_t w1) {
    unsigned long long n = ((unsigned long long)(w0 >> 6) << 26) + (unsigned long long)(w1 >> 6);
    return __dmul_rn(__dadd_rn((double)n, 0.5), 0x1p-52);
}

// find j with F_j <= U < F_{j+1}; x = fma(t, dx, j*dx), t = (U-F_j)/(F_{j+1}-F_j), dx = x_max/K
__device__ __forceinline__ double cdf_invert(const double* __restrict__ F, int K, double x_max, double U) {
    int lo = 0, hi = K;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(F + mid) <= U) lo = mid; else hi = mid;
    }
    double dx = __ddiv_rn(x_max, (double)K);
    double Fl = __ldg(F + lo), Fh = __ldg(F + lo + 1);
    double t = __ddiv_rn(__dsub_rn(U, Fl), __dsub_rn(Fh, Fl));
    return __fma_rn(t, dx, __dmul_rn((double)lo, dx));
}

__global__ void __launch_bounds__(256) k_beam_seed(SeedParams P, double* __restrict__ x, double* __restrict__ y,
                                                   double* __restrict__ z, double* __restrict__ vx,
                                                   double* __restrict__ vy, double* __restrict__ vz,
                                                   unsigned short* __restrict__ group, double* __restrict__ t0) {
    unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= P.n) return;
    unsigned long long idx = P.first_index + j;
    uint32_t w[12];
#pragma unroll
    for (uint32_t b = 0; b < 3; ++b)
        philox4x32_10((uint32_t)idx, (uint32_t)(idx >> 32), b, 0u, (uint32_t)P.seed, (uint32_t)(P.seed >> 32), w + 4 * b);
    double U[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) U[k] = u52(w[2 * k], w[2 * k + 1]);
    double zw = __dmul_rn(2.0, P.z_max);
    double d = cdf_invert(P.cdf_depth, P.n_depth, P.depth_max, U[0]);
    double z1 = __dsub_rn(cdf_invert(P.cdf_normal, P.n_normal, zw, U[1]), P.z_max);
    double z2 = __dsub_rn(cdf_invert(P.cdf_normal, P.n_normal, zw, U[2]), P.z_max);
    double r[3], v[3], scale = P.sigma_pos;
    if (P.profile == TAIGA_PROFILE_DISC) {
        // uniform over the disc ("5 mm diameter"): rejection from the square; retry k reads
        // counter (i lo, i hi, 2 + k, 0); +, -, * only, explicitly rounded
        double a = __dsub_rn(__dmul_rn(2.0, U[1]), 1.0), c2 = __dsub_rn(__dmul_rn(2.0, U[2]), 1.0);
        for (uint32_t k = 1; __dadd_rn(__dmul_rn(a, a), __dmul_rn(c2, c2)) > 1.0; ++k) {
            if (k > 64) { a = 0.0; c2 = 0.0; break; }
            uint32_t q[4];
            philox4x32_10((uint32_t)idx, (uint32_t)(idx >> 32), 2u + k, 0u, (uint32_t)P.seed, (uint32_t)(P.seed >> 32), q);
            a = __dsub_rn(__dmul_rn(2.0, u52(q[0], q[1])), 1.0);
            c2 = __dsub_rn(__dmul_rn(2.0, u52(q[2], q[3])), 1.0);
        }
        z1 = a; z2 = c2; scale = P.radius;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)   // r = (origin + d axis) + scale (z1 eT + z2 eZ)
        r[c] = __dadd_rn(__dadd_rn(P.origin[c], __dmul_rn(d, P.axis[c])),
                         __dmul_rn(scale, __dadd_rn(__dmul_rn(z1, P.eT[c]), __dmul_rn(z2, P.eZ[c]))));
    if (P.sigma_ang == 0.0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = __dmul_rn(P.v0, P.axis[c]);
    } else {
        double z3 = __dsub_rn(cdf_invert(P.cdf_normal, P.n_normal, zw, U[3]), P.z_max);
        double z4 = __dsub_rn(cdf_invert(P.cdf_normal, P.n_normal, zw, U[4]), P.z_max);
        double thT = __dmul_rn(P.sigma_ang, z3), thZ = __dmul_rn(P.sigma_ang, z4);
        double nrm = __dsqrt_rn(__dadd_rn(__dadd_rn(1.0, __dmul_rn(thT, thT)), __dmul_rn(thZ, thZ)));
#pragma unroll
        for (int c = 0; c < 3; ++c)   // v = v0 ((axis + thT eT) + thZ eZ) / nrm
            v[c] = __ddiv_rn(__dmul_rn(P.v0, __dadd_rn(__dadd_rn(P.axis[c], __dmul_rn(thT, P.eT[c])), __dmul_rn(thZ, P.eZ[c]))), nrm);
    }
    x[j] = r[0]; y[j] = r[1]; z[j] = r[2];
    vx[j] = v[0]; vy[j] = v[1]; vz[j] = v[2];
    if (group) group[j] = P.group;
    if (t0) t0[j] = P.t0;
}

// Deterministic initialisation (a grid of representative ions along the beam, each
// weighted by the ionisation density).  Reading D1: nd x nT x nZ cells, ion at the cell centre,
// weight = product of the tabulated-CDF increments over the cell (CDFs linear between points).
// Explicitly rounded intrinsics in a fixed operation order: bit-identical on any IEEE-754 machine.
__device__ __forceinline__ double cdf_value(const double* __restrict__ F, int K, double x_max, double x) {
    double t = __ddiv_rn(x, __ddiv_rn(x_max, (double)K));
    if (!(t > 0.0)) return __ldg(F);
    if (t >= (double)K) return __ldg(F + K);
    int j = __double2int_rd(t);
    double Fl = __ldg(F + j), Fh = __ldg(F + j + 1);
    return __fma_rn(__dsub_rn(t, (double)j), __dsub_rn(Fh, Fl), Fl);
}

__global__ void __launch_bounds__(256) k_beam_seed_grid(SeedParams P, int nd, int nT, int nZ, double z_lim,
                                                        double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                                                        double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                                                        double* __restrict__ w0, unsigned short* __restrict__ group,
                                                        double* __restrict__ t0) {
    unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= P.n) return;
    unsigned long long i = P.first_index + j;
    unsigned long long ib = i % (unsigned long long)nZ, ia = (i / (unsigned long long)nZ) % (unsigned long long)nT,
                       k = i / ((unsigned long long)nZ * (unsigned long long)nT);
    double dd = __ddiv_rn(P.depth_max, (double)nd), zl2 = __dmul_rn(2.0, z_lim), zw = __dmul_rn(2.0, P.z_max);
    double dT = __ddiv_rn(zl2, (double)nT), dZ = __ddiv_rn(zl2, (double)nZ);
    double d_lo = __dmul_rn((double)k, dd), d_hi = __dmul_rn((double)(k + 1), dd), d = __dmul_rn(__dadd_rn((double)k, 0.5), dd);
    double a_lo = __dsub_rn(__dmul_rn((double)ia, dT), z_lim), a_hi = __dsub_rn(__dmul_rn((double)(ia + 1), dT), z_lim),
           za = __dsub_rn(__dmul_rn(__dadd_rn((double)ia, 0.5), dT), z_lim);
    double b_lo = __dsub_rn(__dmul_rn((double)ib, dZ), z_lim), b_hi = __dsub_rn(__dmul_rn((double)(ib + 1), dZ), z_lim),
           zb = __dsub_rn(__dmul_rn(__dadd_rn((double)ib, 0.5), dZ), z_lim);
    double wd = __dsub_rn(cdf_value(P.cdf_depth, P.n_depth, P.depth_max, d_hi), cdf_value(P.cdf_depth, P.n_depth, P.depth_max, d_lo));
    double wT = __dsub_rn(cdf_value(P.cdf_normal, P.n_normal, zw, __dadd_rn(a_hi, P.z_max)),
                          cdf_value(P.cdf_normal, P.n_normal, zw, __dadd_rn(a_lo, P.z_max)));
    double wZ = __dsub_rn(cdf_value(P.cdf_normal, P.n_normal, zw, __dadd_rn(b_hi, P.z_max)),
                          cdf_value(P.cdf_normal, P.n_normal, zw, __dadd_rn(b_lo, P.z_max)));
    double r[3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
        r[c] = __dadd_rn(__dadd_rn(P.origin[c], __dmul_rn(d, P.axis[c])),
                         __dmul_rn(P.sigma_pos, __dadd_rn(__dmul_rn(za, P.eT[c]), __dmul_rn(zb, P.eZ[c]))));
    x[j] = r[0]; y[j] = r[1]; z[j] = r[2];
    vx[j] = __dmul_rn(P.v0, P.axis[0]); vy[j] = __dmul_rn(P.v0, P.axis[1]); vz[j] = __dmul_rn(P.v0, P.axis[2]);
    w0[j] = __dmul_rn(__dmul_rn(wd, wT), wZ);
    if (group) group[j] = P.group;
    if (t0) t0[j] = P.t0;
}

int tg_seed(taiga_ctx* ctx, const taiga_beam_params* p, uint64_t seed, taiga_ions* ions, double v0,
            const taiga_seed_grid* g) {
    size_t cd = ctx->cap_depth, cn = ctx->cap_normal;
    int rc = tg_reserve(ctx, &ctx->cdf_depth, &cd, (size_t)p->n_depth + 1);
    ctx->cap_depth = (int)cd;
    if (rc) return rc;
    rc = tg_reserve(ctx, &ctx->cdf_normal, &cn, (size_t)p->n_normal + 1);
    ctx->cap_normal = (int)cn;
    if (rc) return rc;
    // the tables are staged through a context-owned pinned buffer: the caller's arrays are read during the call only,
    // whatever kind of host memory they live in (a copy from pinned or registered memory is truly asynchronous)
    {
        const size_t nd = (size_t)p->n_depth + 1, nn = (size_t)p->n_normal + 1;
        int rs = tg_stage(ctx, (nd + nn) * sizeof(double));
        if (rs) return rs;
        double* h = (double*)ctx->stage;
        memcpy(h, p->cdf_depth, nd * sizeof(double));
        memcpy(h + nd, p->cdf_normal, nn * sizeof(double));
        TG_CUDA(ctx, cudaMemcpyAsync(ctx->cdf_depth, h, nd * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        TG_CUDA(ctx, cudaMemcpyAsync(ctx->cdf_normal, h + nd, nn * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        TG_CUDA(ctx, cudaEventRecord(ctx->stage_done, ctx->stream));
    }
    SeedParams P;
    P.v0 = v0;
    for (int c = 0; c < 3; ++c) { P.origin[c] = p->origin[c]; P.axis[c] = p->axis[c]; P.eT[c] = p->eT[c]; P.eZ[c] = p->eZ[c]; }
    P.cdf_depth = ctx->cdf_depth; P.n_depth = p->n_depth; P.depth_max = p->depth_max;
    P.cdf_normal = ctx->cdf_normal; P.n_normal = p->n_normal; P.z_max = p->z_max;
    P.sigma_pos = p->sigma_pos_m; P.sigma_ang = p->sigma_ang_rad;
    P.first_index = p->first_index; P.seed = seed; P.n = ions->n;
    P.group = p->group; P.t0 = p->t0;
    P.profile = p->profile; P.radius = p->radius_m;
    unsigned blocks = (unsigned)((ions->n + 255) / 256);
    if (g) k_beam_seed_grid<<<blocks, 256, 0, ctx->stream>>>(P, g->nd, g->nT, g->nZ, g->z_lim, ions->x, ions->y, ions->z, ions->vx,
                                                             ions->vy, ions->vz, ions->w0, ions->group, ions->t0);
    else k_beam_seed<<<blocks, 256, 0, ctx->stream>>>(P, ions->x, ions->y, ions->z, ions->vx, ions->vy, ions->vz, ions->group, ions->t0);
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}
