/* TEST INFRASTRUCTURE -- NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the hot path of the ABP/TAIGA synthetic diagnostic
 * (arxiv/paper_2506_15812), written from PAPER.md and the readings listed in DESIGN.md
 * section 3 (= SURVEY.md 8(c) O0-O5, A1-A19).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call it.  It shares no code with the
 * CUDA path (paper_2506_15812_b200/csrc) and never includes anything from it.
 *
 * Parity pins (tests/test_oracle_pins.py): P1 Philox known answers; P2 RK4 amplification
 * factor in uniform B; P3 Larmor radius / gyro-period; P4 exact parabola in uniform E;
 * P5 kinetic-energy bound; P6 canonical momentum in axisymmetric fields; P7 step-halving
 * order; P8 magnetic moment / grad-B drift; P9 spline properties + scipy cross-check;
 * P10 CDF inversion exactness + statistics; P11 straight-line plane hit + brute-force
 * binning; P12 independent naive evaluator end to end; P13 RK4 (Eq. 4) amplification factor,
 * order and agreement with RKN; P14 Boris (Eq. 7-8) exact |v|, rotation angle 2 atan(z/2),
 * E x B drift, order of both position readings; P15 the three solvers agree as dt -> 0 (L294);
 * P16 Eq. 2 values and limits; P17 loss integral: constant rate -> exp(-nu t_hit) exactly,
 * order 2 under step halving, agreement with an independent quadrature; fixed-point counters;
 * P18 Bezier plane interpolation: exact on parabolas, order 3; P19 weighted-grid seeding:
 * weights sum to 1, marginals = CDF increments, weighted detector image = stochastic image;
 * P20 stage times in a time-linear uniform field (closed-form rotation), Boris B(t_n), trace vs an ODE
 * solution; P21 weight domain of the fixed-point counters; P23 gridded E: central-force invariants, constant grid = uniform E; P22 uniform-disc cross-section: radius bound,
 * r^2 law, uniform azimuth, second moments R^2/4, acceptance pi/4, retry counters.
 * Parity unpinned: nothing in this file; the paper's own figures that cannot be pinned
 * (Fig. 10 loss rate, Table 1, Fig. 12 curves) are listed in DESIGN.md.
 *
 * Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 */
#ifndef TAIGA_ORACLE_H
#define TAIGA_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* field kinds: 0,1,2 = spline tables (2-D static, time slices, toroidal planes);
 * >=10 analytic test fields used only by the pins (PAPER.md L274-282 scenarios). */
enum { ORC_F_RZ = 0, ORC_F_RZT = 1, ORC_F_RZPHI = 2,
       ORC_F_UNIFORM = 10,   /* B = (par0,par1,par2)                                   */
       ORC_F_GRADB   = 11,   /* B = (0,0,par0*(1+par1*x))                              */
       ORC_F_INVR    = 12,   /* B = (0,0,par0/sqrt(x^2+y^2))                           */
       ORC_F_SOLOVEV = 13 }; /* analytic axisymmetric: par = psi_a,R0,a,kappa,B_T      */

typedef struct {
    int kind, nR, nZ, nS;
    double Rmin, Rmax, Zmin, Zmax, s0, ds;
    const double* coef[3];   /* BR, BZ, Bphi per-cell power-basis tables (orc_build_tables) */
    double par[8];           /* analytic-field parameters */
    double E[3];             /* uniform electric field (Eq. 3; L175 "parametric modeling")  */
    const double* ecoef[3];  /* gridded E_R, E_Z, E_phi (Eq. 3 E(r); L177: given on the poloidal plane like B): per-cell
                              * power-basis tables of a static 2-D spline on the (R, Z) grid above, layout of kind 0
                              * (orc_build_tables with kind 0, one slice); all three null = none (reading E1)            */
} orc_field;

/* secondary-ionisation loss inputs (Eq. 2): psi spline table of ONE component in
 * the kind-0 layout [nR-1][nZ-1][16] (orc_build_tables), rate profile nu(psi0 + k dpsi) in 1/s */
typedef struct {
    const double* psi_coef;
    int n; double psi0, dpsi;
    const double* rate;
} orc_loss;

typedef struct {
    double origin[3], normal[3], eu[3], ew[3];
    int nu, nw;
    const double *u_lo, *u_hi, *w_lo, *w_hi;
} orc_detector;

typedef struct {
    double v0;                       /* sqrt(2 E e / m), computed by the caller           */
    double origin[3], axis[3], eT[3], eZ[3];
    const double* cdf_depth;  int n_depth;  double depth_max;
    const double* cdf_normal; int n_normal; double z_max;
    double sigma_pos, sigma_ang;
    int profile;                     /* cross-section: 0 = independent Gaussians (A7), 1 = uniform disc (A7') */
    double radius;                   /* disc radius [m] ("5 mm diameter")              */
} orc_beam;

/* O2.1  Philox4x32-10 */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* O2.1  five uniforms of ion `index` */
void orc_uniforms(uint64_t seed, uint64_t index, double U[5]);
/* O2.2  tabulated-CDF inversion; F has K+1 entries */
double orc_cdf_invert(const double* F, int K, double x_max, double U);
/* O2    seed ions first_index .. first_index+n-1 */
void orc_seed(const orc_beam* b, uint64_t seed, uint64_t first_index, uint64_t n,
              double* x, double* y, double* z, double* vx, double* vy, double* vz);

/* L314 deterministic initialisation (reading D1): weighted grid of nd x nT x nZ representative
 * ions, cross-section spanning +-z_lim sigma_pos; ion index i = (k nT + a) nZ + b */
void orc_seed_grid(const orc_beam* b, int nd, int nT, int nZ, double z_lim, uint64_t first_index, uint64_t n,
                   double* x, double* y, double* z, double* vx, double* vy, double* vz, double* w0);

/* O1  1-D splines on a unit-spaced grid: per-interval power coefficients c[i][0..3],
 *     S(i+p) = c0 + c1 p + c2 p^2 + c3 p^3.  not-a-knot: n>=4 nodes, n-1 intervals;
 *     periodic: n>=3 nodes, n intervals, y[n]==y[0] implied. */
int orc_spline_notaknot(int n, const double* y, double* c);
int orc_spline_periodic(int n, const double* y, double* c);
/* O1  tables of ONE component.  kind 0/1: coef[nS][nR-1][nZ-1][a][b] (16 per cell);
 *     kind 2: coef[nS][nR-1][nZ-1][c][a][b] (64 per cell).  nodal is [nS][nR][nZ]. */
int orc_build_tables(int kind, int nR, int nZ, int nS, const double* nodal, double* coef);
/* O0/O1 field at a Cartesian point and time: B Cartesian */
void orc_field_B(const orc_field* f, const double r[3], double t, double B[3]);
/* E(r) of Eq. 3 in Cartesian components: the uniform vector plus the gridded field (reading E1) */
void orc_field_E(const orc_field* f, const double r[3], double E[3]);
/* field components in the poloidal plane, (B_R,B_Z,B_phi), s = time or phi */
void orc_field_cyl(const orc_field* f, double R, double Z, double s, double Bc[3]);

/* O3  nsteps integrator steps of one ion, no termination tests (pins).  variant = solver code:
 *     0 = classical Nystrom (Eq. 5-6, A1 default), 1 = k3 position from k2 (the printed Eq. 6 k3),
 *     2 = linearised RK4 on y = (r, v) (Eq. 4), 3 = Boris-Verlet (Eq. 7-8 with r advanced by the
 *     NEW velocity, reading R2), 4 = Boris with Eq. 8 as printed (r advanced by the old velocity).
 *     f->E (uniform, "parametric" electric field, L175) enters every solver through Eq. 3. */
void orc_rkn_advance(const orc_field* f, double qm, int variant, double r[3], double v[3],
                     double* t, double dt, uint64_t nsteps);

/* O4  loop + termination + plane interpolation.  status: 0 crossed, -2 max_steps,
 *     -3 left the grid, -4 bad start.  flags: bit1 plane grazing, bit2 grid grazing. */
void orc_trace(const orc_field* f, double qm, int variant, uint64_t n,
               const double* x, const double* y, const double* z,
               const double* vx, const double* vy, const double* vz, const double* t0,
               double dt, uint32_t max_steps, const orc_detector* det,
               int32_t* status, double* hit_u, double* hit_w, double* hit_xyz /*[n][3] or 0*/,
               uint32_t* steps, uint8_t* flags, int nthreads);

/* O4 with the choice of plane interpolation (L338): interp 0 = linear, 1 = quadratic Bezier
 * (reading Z1); orc_trace is interp = 0. */
void orc_trace_interp(const orc_field* f, double qm, int variant, int interp, uint64_t n,
               const double* x, const double* y, const double* z,
               const double* vx, const double* vy, const double* vz, const double* t0,
               double dt, uint32_t max_steps, const orc_detector* det,
               int32_t* status, double* hit_u, double* hit_w, double* hit_xyz,
               uint32_t* steps, uint8_t* flags, int nthreads);

/* O5  binning + counting.  cell_io in: status from orc_trace; out: cell / -1 / error.
 *     counts[n_hist][nw][nu] and summary[n_hist][6] are accumulated into. */
void orc_histogram(uint64_t n, int32_t* cell_io, const double* hit_u, const double* hit_w,
                   const uint16_t* group, uint8_t* flags, const orc_detector* det, int n_hist,
                   uint64_t* counts, uint64_t* summary);

/* NEXT-1: Eq. 2 rate; O4 + loss integral (trapezoid over step end points, reading L2); weighted
 * counters in 32.32 fixed point. */
double orc_mcwhirter_rate(double ne_m3, double Te_eV, double E12_eV);
void orc_trace_loss(const orc_field* f, const orc_loss* L, double qm, int variant, uint64_t n,
                    const double* x, const double* y, const double* z,
                    const double* vx, const double* vy, const double* vz, const double* t0,
                    double dt, uint32_t max_steps, const orc_detector* det,
                    int32_t* status, double* hit_u, double* hit_w,
                    uint32_t* steps, uint8_t* flags, const double* w0 /* or 0 */, double* weight, int nthreads);
/* the same with the plane interpolation of orc_trace_interp (interp = 1: Bezier; the crossing step counts up to the curve
 * parameter of the hit, reading L2') */
void orc_trace_loss_interp(const orc_field* f, const orc_loss* L, double qm, int variant, int interp, uint64_t n,
                    const double* x, const double* y, const double* z,
                    const double* vx, const double* vy, const double* vz, const double* t0,
                    double dt, uint32_t max_steps, const orc_detector* det,
                    int32_t* status, double* hit_u, double* hit_w,
                    uint32_t* steps, uint8_t* flags, const double* w0 /* or 0 */, double* weight, int nthreads);
void orc_histogram_weighted(uint64_t n, const int32_t* cell, const double* weight, const uint16_t* group,
                            const orc_detector* det, int n_hist, uint64_t* wcounts, uint64_t* wsummary);

int orc_max_threads(void);
#ifdef __cplusplus
}
#endif
#endif
