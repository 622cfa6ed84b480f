/* TEST INFRASTRUCTURE -- NOT PRODUCT CODE.  See taiga_oracle.h for scope, pins and build.
 *
 * Every function follows the passage it cites, step by step, in the paper's order and
 * notation; no blocking, fusion or reordering.  Scalar fp64, compiled with
 * -ffp-contract=off so that fma appears only where std::fma is written (O2.2).
 */
#include "taiga_oracle.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------ */
/* O2.1  Philox4x32-10 (Salmon et al. 2011), the counter-based generator SURVEY.md 8(c)
 * O2 fixes for the paper's "stochastic initialisation".                 */
extern "C" void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* O2.1  counter=(i_lo,i_hi,j,0), j=0,1,2 -> 12 words; U_k=((w_2k>>6)*2^26+(w_2k+1>>6)+0.5)*2^-52 */
extern "C" void orc_uniforms(uint64_t seed, uint64_t index, double U[5]) {
    uint32_t w[12];
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (uint32_t j = 0; j < 3; ++j) {
        uint32_t ctr[4] = {(uint32_t)index, (uint32_t)(index >> 32), j, 0u};
        orc_philox4x32_10(ctr, key, w + 4 * j);
    }
    for (int k = 0; k < 5; ++k) {
        uint64_t n = ((uint64_t)(w[2 * k] >> 6) << 26) + (uint64_t)(w[2 * k + 1] >> 6);
        U[k] = ((double)n + 0.5) * 0x1p-52;            /* n+0.5 needs 53 bits: exact */
    }
}

/* O2.2  find j with F_j <= U < F_{j+1} (upper-bound binary search), linear interpolation. */
extern "C" double orc_cdf_invert(const double* F, int K, double x_max, double U) {
    int lo = 0, hi = K;                       /* invariant: F[lo] <= U < F[hi] (F_0=0,F_K=1) */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (F[mid] <= U) lo = mid; else hi = mid;
    }
    double dx = x_max / (double)K;
    double t = (U - F[lo]) / (F[lo + 1] - F[lo]);
    return std::fma(t, dx, (double)lo * dx);
}

/* O2.3-4  PAPER.md L314 (profile used as CDF, random sampling), L128-134 (linear beam). */
extern "C" void orc_seed(const orc_beam* b, uint64_t seed, uint64_t first_index, uint64_t n,
                         double* x, double* y, double* z, double* vx, double* vy, double* vz) {
    for (uint64_t j = 0; j < n; ++j) {
        double U[5];
        orc_uniforms(seed, first_index + j, U);
        double d  = orc_cdf_invert(b->cdf_depth, b->n_depth, b->depth_max, U[0]);
        double z1 = orc_cdf_invert(b->cdf_normal, b->n_normal, 2.0 * b->z_max, U[1]) - b->z_max;
        double z2 = orc_cdf_invert(b->cdf_normal, b->n_normal, 2.0 * b->z_max, U[2]) - b->z_max;
        double z3 = orc_cdf_invert(b->cdf_normal, b->n_normal, 2.0 * b->z_max, U[3]) - b->z_max;
        double z4 = orc_cdf_invert(b->cdf_normal, b->n_normal, 2.0 * b->z_max, U[4]) - b->z_max;
        double r[3], v[3];
        double scale = b->sigma_pos;
        if (b->profile == 1) {
            /* Uniform disc of radius `radius` ("a 60 keV lithium atomic beam with a 5 mm
             * diameter"; reading A7' in DESIGN.md): rejection from the enclosing square, which is exactly
             * uniform on the disc and needs +,-,* only.  Try 0 takes (a, c) = (2 U_1 - 1, 2 U_2 - 1) from the
             * ion's standard uniforms; try k >= 1 takes two fresh uniforms from Philox counter
             * (i_lo, i_hi, 2 + k, 0), words (0,1) and (2,3); accepted when a^2 + c^2 <= 1.  After 64 rejected
             * tries (probability (1 - pi/4)^64 = 1e-43) the ion sits on the axis.                      */
            double a = 2.0 * U[1] - 1.0, c2 = 2.0 * U[2] - 1.0;
            uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
            uint64_t index = first_index + j;
            for (uint32_t k = 1; a * a + c2 * c2 > 1.0; ++k) {
                if (k > 64) { a = 0.0; c2 = 0.0; break; }
                uint32_t ctr[4] = {(uint32_t)index, (uint32_t)(index >> 32), 2u + k, 0u}, w[4];
                orc_philox4x32_10(ctr, key, w);
                uint64_t n0 = ((uint64_t)(w[0] >> 6) << 26) + (uint64_t)(w[1] >> 6);
                uint64_t n1 = ((uint64_t)(w[2] >> 6) << 26) + (uint64_t)(w[3] >> 6);
                a = 2.0 * (((double)n0 + 0.5) * 0x1p-52) - 1.0;
                c2 = 2.0 * (((double)n1 + 0.5) * 0x1p-52) - 1.0;
            }
            z1 = a; z2 = c2; scale = b->radius;
        }
        for (int c = 0; c < 3; ++c)
            r[c] = (b->origin[c] + d * b->axis[c]) + scale * (z1 * b->eT[c] + z2 * b->eZ[c]);
        if (b->sigma_ang == 0.0) {
            for (int c = 0; c < 3; ++c) v[c] = b->v0 * b->axis[c];
        } else {
            double thT = b->sigma_ang * z3, thZ = b->sigma_ang * z4;
            double nrm = std::sqrt((1.0 + thT * thT) + thZ * thZ);
            for (int c = 0; c < 3; ++c)
                v[c] = (b->v0 * ((b->axis[c] + thT * b->eT[c]) + thZ * b->eZ[c])) / nrm;
        }
        x[j] = r[0]; y[j] = r[1]; z[j] = r[2];
        vx[j] = v[0]; vy[j] = v[1]; vz[j] = v[2];
    }
}

/* Deterministic initialisation ("we define a grid with representative ions along
 * the beam, and each virtual ion gets a weight according to the ionization density function").
 * Reading D1: nd x nT x nZ cells; depth cell k = depth_max [k, k+1]/nd, cross-section
 * cells a, b = -z_lim + 2 z_lim [a, a+1]/nT (in units of sigma_pos) and likewise for nZ; the
 * representative ion sits at the cell centre, flies along the beam axis, and carries the weight
 * w0 = (F_d(hi) - F_d(lo)) (Phi(hi_T) - Phi(lo_T)) (Phi(hi_Z) - Phi(lo_Z)), the tabulated CDFs taken
 * linear between their points (the same tables the stochastic mode inverts).  Ion index
 * i = (k nT + a) nZ + b.                                                                      */
static inline double cdf_value(const double* F, int K, double x_max, double x) {
    double t = x / (x_max / (double)K);
    if (!(t > 0.0)) return F[0];
    if (t >= (double)K) return F[K];
    int j = (int)std::floor(t);
    return std::fma(t - (double)j, F[j + 1] - F[j], F[j]);
}
extern "C" void orc_seed_grid(const orc_beam* b, int nd, int nT, int nZ, double z_lim, uint64_t first_index, uint64_t n,
                              double* x, double* y, double* z, double* vx, double* vy, double* vz, double* w0) {
    for (uint64_t j = 0; j < n; ++j) {
        uint64_t i = first_index + j;
        uint64_t ib = i % (uint64_t)nZ, ia = (i / (uint64_t)nZ) % (uint64_t)nT, k = i / ((uint64_t)nZ * (uint64_t)nT);
        double dd = b->depth_max / (double)nd, dT = 2.0 * z_lim / (double)nT, dZ = 2.0 * z_lim / (double)nZ;
        double d_lo = (double)k * dd, d_hi = (double)(k + 1) * dd, d = ((double)k + 0.5) * dd;
        double a_lo = (double)ia * dT - z_lim, a_hi = (double)(ia + 1) * dT - z_lim, za = ((double)ia + 0.5) * dT - z_lim;
        double b_lo = (double)ib * dZ - z_lim, b_hi = (double)(ib + 1) * dZ - z_lim, zb = ((double)ib + 0.5) * dZ - z_lim;
        double wd = cdf_value(b->cdf_depth, b->n_depth, b->depth_max, d_hi) - cdf_value(b->cdf_depth, b->n_depth, b->depth_max, d_lo);
        double wT = cdf_value(b->cdf_normal, b->n_normal, 2.0 * b->z_max, a_hi + b->z_max) -
                    cdf_value(b->cdf_normal, b->n_normal, 2.0 * b->z_max, a_lo + b->z_max);
        double wZ = cdf_value(b->cdf_normal, b->n_normal, 2.0 * b->z_max, b_hi + b->z_max) -
                    cdf_value(b->cdf_normal, b->n_normal, 2.0 * b->z_max, b_lo + b->z_max);
        double r[3];
        for (int c = 0; c < 3; ++c)
            r[c] = (b->origin[c] + d * b->axis[c]) + b->sigma_pos * (za * b->eT[c] + zb * b->eZ[c]);
        x[j] = r[0]; y[j] = r[1]; z[j] = r[2];
        vx[j] = b->v0 * b->axis[0]; vy[j] = b->v0 * b->axis[1]; vz[j] = b->v0 * b->axis[2];
        w0[j] = (wd * wT) * wZ;
    }
}

/* ------------------------------------------------------------------------------------ */
/* O1  dense Gaussian elimination with partial pivoting, m right-hand sides (columns of B) */
static int solve_dense(int n, std::vector<double>& A, int m, double* B /*[n][m]*/) {
    for (int col = 0; col < n; ++col) {
        int piv = col;
        for (int r = col + 1; r < n; ++r)
            if (std::fabs(A[(size_t)r * n + col]) > std::fabs(A[(size_t)piv * n + col])) piv = r;
        if (A[(size_t)piv * n + col] == 0.0) return -1;
        if (piv != col) {
            for (int c = 0; c < n; ++c) std::swap(A[(size_t)piv * n + c], A[(size_t)col * n + c]);
            for (int c = 0; c < m; ++c) std::swap(B[(size_t)piv * m + c], B[(size_t)col * m + c]);
        }
        for (int r = col + 1; r < n; ++r) {
            double f = A[(size_t)r * n + col] / A[(size_t)col * n + col];
            if (f == 0.0) continue;
            for (int c = col; c < n; ++c) A[(size_t)r * n + c] -= f * A[(size_t)col * n + c];
            for (int c = 0; c < m; ++c) B[(size_t)r * m + c] -= f * B[(size_t)col * m + c];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        for (int c = 0; c < m; ++c) {
            double s = B[(size_t)r * m + c];
            for (int k = r + 1; k < n; ++k) s -= A[(size_t)r * n + k] * B[(size_t)k * m + c];
            B[(size_t)r * m + c] = s / A[(size_t)r * n + r];
        }
    }
    return 0;
}

/* O1  family of m 1-D interpolating cubic splines through Y[node][col] on a unit grid.
 * Unknowns: second derivatives M_i.  C2 continuity: M_{i-1}+4M_i+M_{i+1}=6(y_{i-1}-2y_i+y_{i+1}).
 * not-a-knot (A4): third derivative continuous at nodes 1 and n-2:
 *     M_0-2M_1+M_2=0,  M_{n-3}-2M_{n-2}+M_{n-1}=0.
 * periodic (kind 2, phi): indices cyclic, n unknowns, n intervals.
 * Output C[interval][col][0..3]: S = c0 + c1 p + c2 p^2 + c3 p^3 on the interval.        */
static int spline_family(bool periodic, int n, int m, const double* Y, double* C) {
    if ((!periodic && n < 4) || (periodic && n < 3)) return -1;
    std::vector<double> A((size_t)n * n, 0.0), M((size_t)n * m, 0.0);
    auto y = [&](int i, int c) { return Y[(size_t)(((i % n) + n) % n) * m + c]; };
    for (int i = 0; i < n; ++i) {
        bool interior = periodic || (i > 0 && i < n - 1);
        if (interior) {
            int im = periodic ? (i + n - 1) % n : i - 1, ip = periodic ? (i + 1) % n : i + 1;
            A[(size_t)i * n + im] += 1.0; A[(size_t)i * n + i] += 4.0; A[(size_t)i * n + ip] += 1.0;
            for (int c = 0; c < m; ++c)
                M[(size_t)i * m + c] = 6.0 * ((y(i - 1, c) - 2.0 * y(i, c)) + y(i + 1, c));
        } else if (i == 0) {
            A[0] = 1.0; A[1] = -2.0; A[2] = 1.0;
        } else {
            A[(size_t)i * n + n - 3] = 1.0; A[(size_t)i * n + n - 2] = -2.0; A[(size_t)i * n + n - 1] = 1.0;
        }
    }
    if (solve_dense(n, A, m, M.data()) != 0) return -2;
    int nint = periodic ? n : n - 1;
    for (int i = 0; i < nint; ++i) {
        int ip = periodic ? (i + 1) % n : i + 1;
        for (int c = 0; c < m; ++c) {
            double y0 = Y[(size_t)i * m + c], y1 = Y[(size_t)ip * m + c];
            double M0 = M[(size_t)i * m + c], M1 = M[(size_t)ip * m + c];
            double* o = C + ((size_t)i * m + c) * 4;
            o[0] = y0;
            o[1] = (y1 - y0) - (2.0 * M0 + M1) / 6.0;
            o[2] = M0 / 2.0;
            o[3] = (M1 - M0) / 6.0;
        }
    }
    return 0;
}

extern "C" int orc_spline_notaknot(int n, const double* y, double* c) { return spline_family(false, n, 1, y, c); }
extern "C" int orc_spline_periodic(int n, const double* y, double* c) { return spline_family(true, n, 1, y, c); }

/* O1  tensor product (bicubic spline fitted to the grid points, coefficients
 * extracted and stored): spline along Z for every R-node, then spline each of the four
 * w-coefficients along R; kind 2: then a periodic spline along phi of each of the 16.     */
extern "C" int orc_build_tables(int kind, int nR, int nZ, int nS, const double* nodal, double* coef) {
    const int cR = nR - 1, cZ = nZ - 1;
    std::vector<double> bic((size_t)nS * cR * cZ * 16);
    std::vector<double> yz((size_t)nZ * nR), cz((size_t)cZ * nR * 4);
    std::vector<double> yr((size_t)nR * cZ * 4), cr((size_t)cR * cZ * 4 * 4);
    for (int k = 0; k < nS; ++k) {
        const double* g = nodal + (size_t)k * nR * nZ;
        /* along Z: nodes j, columns i */
        for (int j = 0; j < nZ; ++j) for (int i = 0; i < nR; ++i) yz[(size_t)j * nR + i] = g[(size_t)i * nZ + j];
        if (spline_family(false, nZ, nR, yz.data(), cz.data())) return -1;   /* cz[j][i][b] */
        /* along R: nodes i, columns (j,b) */
        for (int i = 0; i < nR; ++i) for (int j = 0; j < cZ; ++j) for (int b = 0; b < 4; ++b)
            yr[((size_t)i * cZ + j) * 4 + b] = cz[((size_t)j * nR + i) * 4 + b];
        if (spline_family(false, nR, cZ * 4, yr.data(), cr.data())) return -1; /* cr[i][j][b][a] */
        for (int i = 0; i < cR; ++i) for (int j = 0; j < cZ; ++j) for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b)
            bic[((((size_t)k * cR + i) * cZ + j) * 4 + a) * 4 + b] = cr[((((size_t)i * cZ + j) * 4 + b) * 4) + a];
    }
    if (kind != ORC_F_RZPHI) { std::memcpy(coef, bic.data(), bic.size() * sizeof(double)); return 0; }
    /* along phi, periodic: nodes k, columns (i,j,a,b) */
    const size_t m = (size_t)cR * cZ * 16;
    std::vector<double> cp((size_t)nS * m * 4);
    if (spline_family(true, nS, (int)m, bic.data(), cp.data())) return -1;   /* cp[k][col][c] */
    for (int k = 0; k < nS; ++k) for (size_t cell = 0; cell < (size_t)cR * cZ; ++cell)
        for (int c = 0; c < 4; ++c) for (int ab = 0; ab < 16; ++ab)
            coef[(((size_t)k * cR * cZ + cell) * 4 + c) * 16 + ab] = cp[(((size_t)k * m) + cell * 16 + ab) * 4 + c];
    return 0;
}

/* O1  evaluation: B(R,Z)=sum_ab c_ab p^a w^b, p=(R-R_i)/h_R, w=(Z-Z_j)/h_Z,
 * i=clamp(floor((R-R_min)/h_R),0,nR-2) (outside the grid the boundary cell extrapolates). */
static inline int cell_index(double x, double xmin, double h, int n, double* frac) {
    int i = (int)std::floor((x - xmin) / h);
    if (i < 0) i = 0;
    if (i > n - 2) i = n - 2;
    *frac = (x - (xmin + (double)i * h)) / h;
    return i;
}
static inline double bicubic(const double* c, double p, double w) {
    double s = 0.0;
    for (int a = 3; a >= 0; --a) {
        double row = ((c[a * 4 + 3] * w + c[a * 4 + 2]) * w + c[a * 4 + 1]) * w + c[a * 4 + 0];
        s = s * p + row;
    }
    return s;
}

extern "C" void orc_field_cyl(const orc_field* f, double R, double Z, double s, double Bc[3]) {
    const int cR = f->nR - 1, cZ = f->nZ - 1;
    double hR = (f->Rmax - f->Rmin) / (double)cR, hZ = (f->Zmax - f->Zmin) / (double)cZ;
    double p, w;
    int i = cell_index(R, f->Rmin, hR, f->nR, &p);
    int j = cell_index(Z, f->Zmin, hZ, f->nZ, &w);
    size_t cell = (size_t)i * cZ + j;
    if (f->kind == ORC_F_RZ) {
        for (int c = 0; c < 3; ++c) Bc[c] = bicubic(f->coef[c] + cell * 16, p, w);
    } else if (f->kind == ORC_F_RZT) {
        /* B(t)=(1-tau)B_k+tau B_{k+1}, k=clamp(floor((t-s0)/ds),0,nS-2), tau=clamp(.,0,1): held
         * outside the slice range (A16).                                                  */
        double xs = (s - f->s0) / f->ds;
        int k = (int)std::floor(xs);
        if (k < 0) k = 0;
        if (k > f->nS - 2) k = f->nS - 2;
        double tau = xs - (double)k;
        if (tau < 0.0) tau = 0.0;
        if (tau > 1.0) tau = 1.0;
        size_t stride = (size_t)cR * cZ * 16;
        for (int c = 0; c < 3; ++c) {
            double b0 = bicubic(f->coef[c] + k * stride + cell * 16, p, w);
            double b1 = bicubic(f->coef[c] + (k + 1) * stride + cell * 16, p, w);
            Bc[c] = (1.0 - tau) * b0 + tau * b1;
        }
    } else { /* ORC_F_RZPHI: periodic tricubic, 64 coefficients per cell; s = phi (A17) */
        double xs = (s - f->s0) / f->ds;
        xs = xs - (double)f->nS * std::floor(xs / (double)f->nS);      /* into [0,nS) */
        int k = (int)std::floor(xs);
        if (k < 0) k = 0;
        if (k > f->nS - 1) k = f->nS - 1;
        double q = xs - (double)k;
        size_t base = ((size_t)k * cR * cZ + cell) * 64;
        for (int c = 0; c < 3; ++c) {
            const double* d = f->coef[c] + base;
            double acc = 0.0;
            for (int e = 3; e >= 0; --e) acc = acc * q + bicubic(d + e * 16, p, w);
            Bc[c] = acc;
        }
    }
}

/* O0  Cartesian <-> poloidal plane: R=sqrt(X^2+Y^2), c=X/R, s=Y/R,
 * B_X=B_R c-B_phi s, B_Y=B_R s+B_phi c.                                                   */
extern "C" void orc_field_B(const orc_field* f, const double r[3], double t, double B[3]) {
    switch (f->kind) {
    case ORC_F_UNIFORM: B[0] = f->par[0]; B[1] = f->par[1]; B[2] = f->par[2]; return;
    case ORC_F_GRADB:   B[0] = 0.0; B[1] = 0.0; B[2] = f->par[0] * (1.0 + f->par[1] * r[0]); return;
    case ORC_F_INVR:    B[0] = 0.0; B[1] = 0.0; B[2] = f->par[0] / std::sqrt(r[0] * r[0] + r[1] * r[1]); return;
    default: break;
    }
    double R = std::sqrt(r[0] * r[0] + r[1] * r[1]);
    double c = r[0] / R, s = r[1] / R;
    double Bc[3];
    if (f->kind == ORC_F_SOLOVEV) {
        double psa = f->par[0], R0 = f->par[1], a = f->par[2], kap = f->par[3], BT = f->par[4];
        double Z = r[2];
        Bc[0] = -2.0 * psa * R * Z / ((R0 * kap * a) * (R0 * kap * a));
        Bc[1] = psa * ((R * R - R0 * R0) / ((R0 * a) * (R0 * a)) + 2.0 * Z * Z / ((R0 * kap * a) * (R0 * kap * a)));
        Bc[2] = -BT * R0 / R;
    } else {
        double sarg = (f->kind == ORC_F_RZPHI) ? std::atan2(r[1], r[0]) : t;
        orc_field_cyl(f, R, r[2], sarg, Bc);
    }
    B[0] = Bc[0] * c - Bc[2] * s;
    B[1] = Bc[0] * s + Bc[2] * c;
    B[2] = Bc[1];
}

/* E(r) of Eq. 3 (L177: "mapped to a poloidal cross-section plane ... That is how the local magnetic
 * and electric field is given"): the uniform vector plus, when given, a static field tabulated like B -- E_R, E_Z, E_phi
 * on the (R, Z) grid, the same bicubic spline, the boundary cell extrapolating outside the grid (A12), rotated to
 * Cartesian components like B (O0).  Reading E1 in DESIGN.md.                                                       */
extern "C" void orc_field_E(const orc_field* f, const double r[3], double E[3]) {
    E[0] = f->E[0]; E[1] = f->E[1]; E[2] = f->E[2];
    if (!f->ecoef[0]) return;
    const int cR = f->nR - 1, cZ = f->nZ - 1;
    double hR = (f->Rmax - f->Rmin) / (double)cR, hZ = (f->Zmax - f->Zmin) / (double)cZ;
    double R = std::sqrt(r[0] * r[0] + r[1] * r[1]);
    double c = r[0] / R, s = r[1] / R;
    double p, w, Ec[3];
    int i = cell_index(R, f->Rmin, hR, f->nR, &p);
    int j = cell_index(r[2], f->Zmin, hZ, f->nZ, &w);
    size_t cell = (size_t)i * cZ + j;
    for (int m = 0; m < 3; ++m) Ec[m] = bicubic(f->ecoef[m] + cell * 16, p, w);
    E[0] = E[0] + (Ec[0] * c - Ec[2] * s);
    E[1] = E[1] + (Ec[0] * s + Ec[2] * c);
    E[2] = E[2] + Ec[1];
}

/* Eq. 3: a = (q/m)(E + v x B) */
static inline void accel(const orc_field* f, double qm, const double r[3], const double v[3], double t, double a[3]) {
    double B[3], E[3];
    orc_field_B(f, r, t, B);
    orc_field_E(f, r, E);
    a[0] = qm * (E[0] + (v[1] * B[2] - v[2] * B[1]));
    a[1] = qm * (E[1] + (v[2] * B[0] - v[0] * B[2]));
    a[2] = qm * (E[2] + (v[0] * B[1] - v[1] * B[0]));
}

/* O3  one Runge-Kutta-Nystrom step, Eq. 5-6 under readings A1-A3:
 *  k1=a(r,v,t); k2=a(r+v dt/2+k1 dt^2/8, v+k1 dt/2, t+dt/2);
 *  k3=a(r+v dt/2+K dt^2/8, v+k2 dt/2, t+dt/2), K=k1 (classical, variant 0) or k2 (printed, 1);
 *  k4=a(r+v dt+k3 dt^2/2, v+k3 dt, t+dt);
 *  r'=r+v dt+(k1+k2+k3) dt^2/6;  v'=v+(k1+2k2+2k3+k4) dt/6.                               */
static inline void rkn_step(const orc_field* f, double qm, int variant, const double r[3], const double v[3],
                            double t, double dt, double rn[3], double vn[3]) {
    double k1[3], k2[3], k3[3], k4[3], rs[3], vs[3];
    accel(f, qm, r, v, t, k1);
    for (int c = 0; c < 3; ++c) { rs[c] = r[c] + v[c] * (dt / 2.0) + k1[c] * (dt * dt / 8.0); vs[c] = v[c] + k1[c] * (dt / 2.0); }
    accel(f, qm, rs, vs, t + dt / 2.0, k2);
    const double* K = variant ? k2 : k1;
    for (int c = 0; c < 3; ++c) { rs[c] = r[c] + v[c] * (dt / 2.0) + K[c] * (dt * dt / 8.0); vs[c] = v[c] + k2[c] * (dt / 2.0); }
    accel(f, qm, rs, vs, t + dt / 2.0, k3);
    for (int c = 0; c < 3; ++c) { rs[c] = r[c] + v[c] * dt + k3[c] * (dt * dt / 2.0); vs[c] = v[c] + k3[c] * dt; }
    accel(f, qm, rs, vs, t + dt, k4);
    for (int c = 0; c < 3; ++c) {
        rn[c] = r[c] + v[c] * dt + (k1[c] + k2[c] + k3[c]) * (dt * dt / 6.0);
        vn[c] = v[c] + (k1[c] + 2.0 * k2[c] + 2.0 * k3[c] + k4[c]) * (dt / 6.0);
    }
}

/* Eq. 4: the equation of motion as a first-order system in the generalised
 * coordinate y = (r1,r2,r3,v1,v2,v3), dy/dt = f(y,t) with f_{1..3} = y_{4..6} and f_{4..6} =
 * (q/m)(E + v x B); "solved by a fourth-order Runge-Kutta method" (L210): the classical RK4
 *  K1=f(y,t); K2=f(y+K1 dt/2,t+dt/2); K3=f(y+K2 dt/2,t+dt/2); K4=f(y+K3 dt,t+dt);
 *  y'=y+(K1+2K2+2K3+K4) dt/6.   (Reading R1 in DESIGN.md: L191 calls the solver "quadratic";
 *  L210 and ref. [29] fix the fourth-order scheme.)                                          */
static inline void rk4_f(const orc_field* f, double qm, const double y[6], double t, double dy[6]) {
    dy[0] = y[3]; dy[1] = y[4]; dy[2] = y[5];
    accel(f, qm, y, y + 3, t, dy + 3);
}
static inline void rk4_step(const orc_field* f, double qm, const double r[3], const double v[3],
                            double t, double dt, double rn[3], double vn[3]) {
    double y[6] = {r[0], r[1], r[2], v[0], v[1], v[2]}, ys[6], K1[6], K2[6], K3[6], K4[6];
    rk4_f(f, qm, y, t, K1);
    for (int c = 0; c < 6; ++c) ys[c] = y[c] + K1[c] * (dt / 2.0);
    rk4_f(f, qm, ys, t + dt / 2.0, K2);
    for (int c = 0; c < 6; ++c) ys[c] = y[c] + K2[c] * (dt / 2.0);
    rk4_f(f, qm, ys, t + dt / 2.0, K3);
    for (int c = 0; c < 6; ++c) ys[c] = y[c] + K3[c] * dt;
    rk4_f(f, qm, ys, t + dt, K4);
    for (int c = 0; c < 3; ++c) {
        rn[c] = y[c] + (K1[c] + 2.0 * K2[c] + 2.0 * K3[c] + K4[c]) * (dt / 6.0);
        vn[c] = y[c + 3] + (K1[c + 3] + 2.0 * K2[c + 3] + 2.0 * K3[c + 3] + K4[c + 3]) * (dt / 6.0);
    }
}

static inline void cross3(const double a[3], const double b[3], double c[3]) {
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}

/* Eq. 7: Boris push of the velocity over a step h, B and E taken at r, t:
 *  v- = v + (q/m) E h/2;  t = (q/m) B h/2;  s = 2t/(1+t.t);  v* = v- + v- x t;
 *  v+ = v- + v* x s;  v' = v+ + (q/m) E h/2   (first line of Eq. 8).                         */
static inline void boris_velocity(const orc_field* f, double qm, const double r[3], const double v[3],
                                  double t, double h, double vn[3]) {
    double B[3], E[3], vm[3], tv[3], sv[3], vs[3], vp[3], c1[3], c2[3];
    orc_field_B(f, r, t, B);
    orc_field_E(f, r, E);
    double tt = 0.0;
    for (int c = 0; c < 3; ++c) { vm[c] = v[c] + qm * E[c] * (h / 2.0); tv[c] = qm * B[c] * (h / 2.0); tt += tv[c] * tv[c]; }
    for (int c = 0; c < 3; ++c) sv[c] = 2.0 * tv[c] / (1.0 + tt);
    cross3(vm, tv, c1);
    for (int c = 0; c < 3; ++c) vs[c] = vm[c] + c1[c];
    cross3(vs, sv, c2);
    for (int c = 0; c < 3; ++c) { vp[c] = vm[c] + c2[c]; vn[c] = vp[c] + qm * E[c] * (h / 2.0); }
}
/* Eq. 8, second line (L266): position.  As printed, r(t0+dt) = r(t0) + v(t0) dt uses the OLD
 * velocity: explicit Euler in r, first order, while the text calls the solver "a second-order
 * Verlet solver with a Boris push" (L249).  Reading R2: solver 3 is the Verlet /
 * leap-frog form of refs [32,33], r(t0+dt) = r(t0) + v' dt with the velocity living at half
 * steps (boris_start below); solver 4 is Eq. 8 exactly as printed, no start correction.      */
static inline void boris_step(const orc_field* f, double qm, bool printed, const double r[3], const double v[3],
                              double t, double dt, double rn[3], double vn[3]) {
    boris_velocity(f, qm, r, v, t, dt, vn);
    for (int c = 0; c < 3; ++c) rn[c] = r[c] + (printed ? v[c] : vn[c]) * dt;
}
/* leap-frog start of solver 3: v(t0) -> v(t0 - dt/2) by a Boris push over -dt/2 at (r0, t0) */
static inline void boris_start(const orc_field* f, double qm, const double r[3], double v[3], double t, double dt) {
    double vb[3];
    boris_velocity(f, qm, r, v, t, -dt / 2.0, vb);
    for (int c = 0; c < 3; ++c) v[c] = vb[c];
}

/* solver codes: 0 RKN classical (A1), 1 RKN with the printed k3, 2 linearised RK4 (Eq. 4),
 * 3 Boris-Verlet (Eq. 7-8, reading R2), 4 Boris with Eq. 8 as printed */
static inline void solver_step(const orc_field* f, double qm, int solver, const double r[3], const double v[3],
                               double t, double dt, double rn[3], double vn[3]) {
    if (solver == 2) rk4_step(f, qm, r, v, t, dt, rn, vn);
    else if (solver == 3 || solver == 4) boris_step(f, qm, solver == 4, r, v, t, dt, rn, vn);
    else rkn_step(f, qm, solver, r, v, t, dt, rn, vn);
}

extern "C" void orc_rkn_advance(const orc_field* f, double qm, int variant, double r[3], double v[3],
                                double* t, double dt, uint64_t nsteps) {
    if (variant == 3) boris_start(f, qm, r, v, *t, dt);     /* every call is a fresh start */
    for (uint64_t s = 0; s < nsteps; ++s) {
        double rn[3], vn[3];
        solver_step(f, qm, variant, r, v, *t, dt, rn, vn);
        for (int c = 0; c < 3; ++c) { r[c] = rn[c]; v[c] = vn[c]; }
        *t = *t + dt;
    }
}

static const double GRAZE = 1e-9;   /* grazing thresholds, fp64 */

static inline bool in_grid(const orc_field* f, const double r[3], bool* graze) {
    if (f->kind >= 10) return true;                       /* analytic test fields: no grid */
    double R = std::sqrt(r[0] * r[0] + r[1] * r[1]), Z = r[2];
    if (std::fabs(R - f->Rmin) < GRAZE || std::fabs(R - f->Rmax) < GRAZE ||
        std::fabs(Z - f->Zmin) < GRAZE || std::fabs(Z - f->Zmax) < GRAZE) *graze = true;
    return !(R < f->Rmin || R > f->Rmax || Z < f->Zmin || Z > f->Zmax);
}

/* O4  PAPER.md L326 ("stops when a particle passes through the detector plane or reaches the
 * maximum number of iterations ... an interpolation is applied to the detector plane using
 * coordinates from the previous iteration step"), L318 (error value), L338 (two-state
 * storage, linear interpolation), L330 (coordinate transformation to the plane).          */
/* L338: "We can use linear interpolation or quadratic Bezier interpolation to get the impact
 * coordinates", from "the position and velocity coordinates of the current and previous iteration
 * steps".  interp = 0: linear (O4 above).  interp = 1 (reading Z1 in DESIGN.md): the quadratic
 * Bezier curve B(tau) = (1-tau)^2 P0 + 2 (1-tau) tau P1 + tau^2 P2 with P0 = r_n, P2 = r_{n+1}
 * and the control point at the mean of the two tangent estimates,
 * P1 = [(r_n + v_n dt/2) + (r_{n+1} - v_{n+1} dt/2)] / 2; the hit is B(tau*) where the signed
 * plane distance s(tau) = (1-tau)^2 s0 + 2 (1-tau) tau sc + tau^2 s1 vanishes in [0,1]
 * (sc = n.(P1 - r_D)); tau* = 2 s0 / (2 s0 - 2 sc - sqrt(4 sc^2 - 4 s0 s1))... written below in
 * the cancellation-free form.  Exact for uniformly accelerated motion.                       */
static inline double bezier_hit(const double r[3], const double v[3], const double rn[3], const double vn[3],
                                double dt, double s0, double s1, const orc_detector* det, double p[3]) {
    double P1[3], sc = 0.0;
    for (int c = 0; c < 3; ++c) {
        P1[c] = 0.5 * ((r[c] + v[c] * (dt / 2.0)) + (rn[c] - vn[c] * (dt / 2.0)));
        sc += det->normal[c] * (P1[c] - det->origin[c]);
    }
    /* a tau^2 + b tau + c = 0, a = s0 - 2 sc + s1, b = 2 (sc - s0), c = s0 < 0 <= s1 */
    double a = s0 - 2.0 * sc + s1, b = 2.0 * (sc - s0), c = s0;
    double disc = b * b - 4.0 * a * c;
    double tau;
    if (!(disc >= 0.0)) tau = s0 / (s0 - s1);               /* no real root (cannot happen with s0<0<=s1): linear */
    else {
        double sq = std::sqrt(disc);
        tau = (b >= 0.0) ? (-2.0 * c) / (b + sq) : (-b + sq) / (2.0 * a);
    }
    if (!(tau >= 0.0)) tau = 0.0;
    if (tau > 1.0) tau = 1.0;
    double w0 = (1.0 - tau) * (1.0 - tau), w1 = 2.0 * (1.0 - tau) * tau, w2 = tau * tau;
    for (int k = 0; k < 3; ++k) p[k] = w0 * r[k] + w1 * P1[k] + w2 * rn[k];
    return tau;                                             /* the curve parameter of the hit (reading L2': loss integral) */
}

extern "C" void orc_trace(const orc_field* f, double qm, int variant, uint64_t n,
                          const double* x, const double* y, const double* z,
                          const double* vx, const double* vy, const double* vz, const double* t0,
                          double dt, uint32_t max_steps, const orc_detector* det,
                          int32_t* status, double* hit_u, double* hit_w, double* hit_xyz,
                          uint32_t* steps, uint8_t* flags, int nthreads) {
    orc_trace_interp(f, qm, variant, 0, n, x, y, z, vx, vy, vz, t0, dt, max_steps, det, status, hit_u, hit_w, hit_xyz,
                     steps, flags, nthreads);
}

extern "C" void orc_trace_interp(const orc_field* f, double qm, int variant, int interp, uint64_t n,
                          const double* x, const double* y, const double* z,
                          const double* vx, const double* vy, const double* vz, const double* t0,
                          double dt, uint32_t max_steps, const orc_detector* det,
                          int32_t* status, double* hit_u, double* hit_w, double* hit_xyz,
                          uint32_t* steps, uint8_t* flags, int nthreads) {
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (int64_t ii = 0; ii < (int64_t)n; ++ii) {
        uint64_t i = (uint64_t)ii;
        double r[3] = {x[i], y[i], z[i]}, v[3] = {vx[i], vy[i], vz[i]};
        double t = t0 ? t0[i] : 0.0;
        uint8_t fl = 0;
        bool gz = false;
        double s0 = det->normal[0] * (r[0] - det->origin[0]) + det->normal[1] * (r[1] - det->origin[1]) +
                    det->normal[2] * (r[2] - det->origin[2]);
        hit_u[i] = 0.0; hit_w[i] = 0.0;
        if (hit_xyz) hit_xyz[3 * i] = hit_xyz[3 * i + 1] = hit_xyz[3 * i + 2] = 0.0;
        if (std::fabs(s0) < GRAZE) fl |= 2;
        bool inside = in_grid(f, r, &gz);
        if (gz) fl |= 4;
        if (!(s0 < 0.0) || !inside) { status[i] = -4; steps[i] = 0; flags[i] = fl; continue; }
        if (variant == 3) boris_start(f, qm, r, v, t, dt);
        int32_t st = -2;
        uint32_t nst = max_steps;
        for (uint32_t step = 1; step <= max_steps; ++step) {
            double rn[3], vn[3];
            solver_step(f, qm, variant, r, v, t, dt, rn, vn);
            double s1 = det->normal[0] * (rn[0] - det->origin[0]) + det->normal[1] * (rn[1] - det->origin[1]) +
                        det->normal[2] * (rn[2] - det->origin[2]);
            if (std::fabs(s1) < GRAZE) fl |= 2;
            if (s0 < 0.0 && s1 >= 0.0) {
                double lam = s0 / (s0 - s1);
                double p[3];
                for (int c = 0; c < 3; ++c) p[c] = r[c] + lam * (rn[c] - r[c]);
                if (interp == 1) bezier_hit(r, v, rn, vn, dt, s0, s1, det, p);
                hit_u[i] = (p[0] - det->origin[0]) * det->eu[0] + (p[1] - det->origin[1]) * det->eu[1] + (p[2] - det->origin[2]) * det->eu[2];
                hit_w[i] = (p[0] - det->origin[0]) * det->ew[0] + (p[1] - det->origin[1]) * det->ew[1] + (p[2] - det->origin[2]) * det->ew[2];
                if (hit_xyz) { hit_xyz[3 * i] = p[0]; hit_xyz[3 * i + 1] = p[1]; hit_xyz[3 * i + 2] = p[2]; }
                st = 0; nst = step;
                break;
            }
            gz = false;
            inside = in_grid(f, rn, &gz);
            if (gz) fl |= 4;
            if (!inside) { st = -3; nst = step; break; }
            for (int c = 0; c < 3; ++c) { r[c] = rn[c]; v[c] = vn[c]; }
            t = t + dt;
            s0 = s1;
        }
        status[i] = st; steps[i] = nst; flags[i] = fl;
    }
}

/* ---- secondary-ionisation loss ------------------------------------- */

/* Eq. 2: McWhirter's rate of Li+ -> Li2+ (Na+ -> Na2+) per ion,
 *   nu = n_e * sqrt(t_e) exp(-1/t_e) / ((E12/1 eV)^{3/2} (6 + t_e)) * 1e-11 m^3/s,  t_e = T_e/E12,
 * n_e in m^-3, T_e and E12 in eV; result in 1/s.  T_e <= 0 gives 0 (the limit).               */
extern "C" double orc_mcwhirter_rate(double ne, double Te, double E12) {
    if (!(Te > 0.0)) return 0.0;
    double te = Te / E12;
    return ne * (std::sqrt(te) * std::exp(-1.0 / te) / (std::pow(E12, 1.5) * (6.0 + te))) * 1e-11;
}

/* L177: "These coordinates are mapped to a poloidal cross-section plane in each iteration step.
 * That is how ... the poloidal flux coordinate is determined.  The loss due to the secondary
 * ionization that is described by Equation 2 is numerically integrated with every step using the
 * one-dimensional secondary ionization profile."
 * psi(R,Z): bicubic spline table on the field's (R,Z) grid (same cell rule, boundary cell
 * extrapolates); nu(psi): table of n entries at psi0 + k dpsi, linear in between, held constant
 * outside (reading L1 in DESIGN.md).                                                          */
static inline double loss_rate(const orc_field* f, const orc_loss* L, const double r[3]) {
    const int cZ = f->nZ - 1;
    double hR = (f->Rmax - f->Rmin) / (double)(f->nR - 1), hZ = (f->Zmax - f->Zmin) / (double)cZ;
    double R = std::sqrt(r[0] * r[0] + r[1] * r[1]), p, w;
    int i = cell_index(R, f->Rmin, hR, f->nR, &p);
    int j = cell_index(r[2], f->Zmin, hZ, f->nZ, &w);
    double psi = bicubic(L->psi_coef + ((size_t)i * cZ + j) * 16, p, w);
    double x = (psi - L->psi0) / L->dpsi;
    if (!(x > 0.0)) return L->rate[0];
    if (x >= (double)(L->n - 1)) return L->rate[L->n - 1];
    int k = (int)std::floor(x);
    double fr = x - (double)k;
    return L->rate[k] + fr * (L->rate[k + 1] - L->rate[k]);
}

/* O4 with the loss integral.  "integrated with every step" (L177) is read as the trapezoidal rule
 * over the step end points (reading L2): Lam += dt (nu(r_n) + nu(r_{n+1}))/2; on the crossing step
 * only the fraction lam up to the plane counts, with nu interpolated linearly to the hit point:
 * Lam += lam dt (nu_n + nu_hit)/2, nu_hit = nu_n + lam (nu_{n+1} - nu_n).  weight = exp(-Lam): the
 * surviving fraction of singly ionised ions (dn1/dt = -nu n1).  Ions that do not cross get the
 * weight accumulated up to their last step.  Everything else is orc_trace, unchanged.         */
extern "C" void orc_trace_loss(const orc_field* f, const orc_loss* L, double qm, int variant, uint64_t n,
                               const double* x, const double* y, const double* z,
                               const double* vx, const double* vy, const double* vz, const double* t0,
                               double dt, uint32_t max_steps, const orc_detector* det,
                               int32_t* status, double* hit_u, double* hit_w,
                               uint32_t* steps, uint8_t* flags, const double* w0, double* weight, int nthreads) {
    orc_trace_loss_interp(f, L, qm, variant, 0, n, x, y, z, vx, vy, vz, t0, dt, max_steps, det, status, hit_u, hit_w, steps,
                          flags, w0, weight, nthreads);
}

/* The same with the plane interpolation of orc_trace_interp.  interp = 1 (Bezier, reading Z1): the fraction of the crossing
 * step that counts is the curve parameter tau of the hit instead of lam, nu interpolated linearly in tau (reading L2'). */
extern "C" void orc_trace_loss_interp(const orc_field* f, const orc_loss* L, double qm, int variant, int interp, uint64_t n,
                                      const double* x, const double* y, const double* z,
                                      const double* vx, const double* vy, const double* vz, const double* t0,
                                      double dt, uint32_t max_steps, const orc_detector* det,
                                      int32_t* status, double* hit_u, double* hit_w,
                                      uint32_t* steps, uint8_t* flags, const double* w0, double* weight, int nthreads) {
    orc_trace_interp(f, qm, variant, interp, n, x, y, z, vx, vy, vz, t0, dt, max_steps, det, status, hit_u, hit_w, nullptr,
                     steps, flags, nthreads);
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (int64_t ii = 0; ii < (int64_t)n; ++ii) {
        uint64_t i = (uint64_t)ii;
        double r[3] = {x[i], y[i], z[i]}, v[3] = {vx[i], vy[i], vz[i]};
        double t = t0 ? t0[i] : 0.0, Lam = 0.0;
        const double wi = w0 ? w0[i] : 1.0;                       /* initial statistical weight (deterministic mode) */
        if (status[i] == -4) { weight[i] = wi; continue; }
        if (variant == 3) boris_start(f, qm, r, v, t, dt);
        double s0 = det->normal[0] * (r[0] - det->origin[0]) + det->normal[1] * (r[1] - det->origin[1]) +
                    det->normal[2] * (r[2] - det->origin[2]);
        double nu0 = loss_rate(f, L, r);
        for (uint32_t step = 1; step <= steps[i]; ++step) {      /* the same steps orc_trace took */
            double rn[3], vn[3];
            solver_step(f, qm, variant, r, v, t, dt, rn, vn);
            double nu1 = loss_rate(f, L, rn);
            if (step == steps[i] && status[i] == 0) {
                double s1 = det->normal[0] * (rn[0] - det->origin[0]) + det->normal[1] * (rn[1] - det->origin[1]) +
                            det->normal[2] * (rn[2] - det->origin[2]);
                double lam = s0 / (s0 - s1);
                if (interp == 1) { double p[3]; lam = bezier_hit(r, v, rn, vn, dt, s0, s1, det, p); }
                double nuh = nu0 + lam * (nu1 - nu0);
                Lam += lam * dt * (nu0 + nuh) / 2.0;
                break;
            }
            if (step == steps[i] && status[i] == -3) break;      /* left the grid: the last step is not counted */
            Lam += dt * (nu0 + nu1) / 2.0;
            for (int c = 0; c < 3; ++c) { r[c] = rn[c]; v[c] = vn[c]; }
            t = t + dt;
            s0 = det->normal[0] * (r[0] - det->origin[0]) + det->normal[1] * (r[1] - det->origin[1]) +
                 det->normal[2] * (r[2] - det->origin[2]);
            nu0 = nu1;
        }
        weight[i] = wi * std::exp(-Lam);
    }
}

/* Weighted counters (L350: "weight ... by the secondary loss"): every plane-crossing ion adds its
 * weight in 32.32 fixed point, q = floor(w 2^32 + 1/2), so that sums are integers and independent
 * of the order of accumulation.  wcounts[n_hist][nw][nu] by segment; wsummary[n_hist][4] =
 * {sum q in segments, sum q of crossers outside the segments, sum floor(q^2 / 2^32) over all
 * crossers, number of crossers}.  cell[] as written by orc_histogram.                          */
extern "C" void orc_histogram_weighted(uint64_t n, const int32_t* cell, const double* weight, const uint16_t* group,
                                       const orc_detector* det, int n_hist, uint64_t* wcounts, uint64_t* wsummary) {
    const size_t ncell = (size_t)det->nu * det->nw;
    for (uint64_t i = 0; i < n; ++i) {
        int g = group ? (int)group[i] : 0;
        if (g >= n_hist || cell[i] < -1) continue;
        double wv = weight[i];
        if (!(wv >= 0.0)) wv = 0.0;                           /* negative / NaN weights count as 0 */
        if (wv > 1048576.0) wv = 1048576.0;
        uint64_t q = (uint64_t)std::floor(wv * 4294967296.0 + 0.5);
        if (cell[i] >= 0) { wcounts[(size_t)g * ncell + (size_t)cell[i]] += q; wsummary[g * 4 + 0] += q; }
        else wsummary[g * 4 + 1] += q;
        wsummary[g * 4 + 2] += (uint64_t)(((unsigned __int128)q * q) >> 32);
        wsummary[g * 4 + 3] += 1;
    }
}

/* O5  PAPER.md L330 (segments with optional non-uniform size and gaps on a perpendicular
 * grid), L344-350 (segment ID or error indicator per ion; atomically summed counters).
 * Brute-force linear scan over all segments; half-open [lo,hi) (A11).                      */
extern "C" void orc_histogram(uint64_t n, int32_t* cell_io, const double* hit_u, const double* hit_w,
                              const uint16_t* group, uint8_t* flags, const orc_detector* det, int n_hist,
                              uint64_t* counts, uint64_t* summary) {
    for (uint64_t i = 0; i < n; ++i) {
        int g = group ? (int)group[i] : 0;
        if (g >= n_hist) continue;
        uint64_t* sm = summary + (size_t)g * 6;
        int32_t st = cell_io[i];
        if (st >= -1) {
            double u = hit_u[i], w = hit_w[i];
            int iu = -1, iw = -1;
            for (int k = 0; k < det->nu; ++k) {
                if (det->u_lo[k] <= u && u < det->u_hi[k] && iu < 0) iu = k;
                if (std::fabs(u - det->u_lo[k]) < GRAZE || std::fabs(u - det->u_hi[k]) < GRAZE) flags[i] |= 1;
            }
            for (int k = 0; k < det->nw; ++k) {
                if (det->w_lo[k] <= w && w < det->w_hi[k] && iw < 0) iw = k;
                if (std::fabs(w - det->w_lo[k]) < GRAZE || std::fabs(w - det->w_hi[k]) < GRAZE) flags[i] |= 1;
            }
            if (iu >= 0 && iw >= 0) {
                cell_io[i] = iw * det->nu + iu;
                counts[((size_t)g * det->nw + iw) * det->nu + iu] += 1;
                sm[0] += 1;
            } else { cell_io[i] = -1; sm[1] += 1; }
        } else if (st == -2) sm[2] += 1;
        else if (st == -3) sm[3] += 1;
        else sm[4] += 1;
        if (flags[i]) sm[5] += 1;
    }
}

extern "C" int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
