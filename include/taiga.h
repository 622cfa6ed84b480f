/* taiga.h -- C ABI of the B200-native hot path of the ABP/TAIGA synthetic diagnostic
 * (arxiv/paper_2506_15812): field-coefficient precompute -> beam seeding -> Runge-Kutta-Nystrom
 * trajectory integration -> detector-plane crossing -> Faraday-cup histogram.
 *
 * Conventions
 *  - Every function returns 0 (TAIGA_OK) or a negative TAIGA_E_* code; nothing aborts or
 *    throws.  taiga_last_error(ctx) returns a NUL-terminated message owned by ctx.
 *  - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors);
 *    "host" pointers are ordinary host memory, read during the call only.  The ctx owns only
 *    its internal tables / scratch and frees them in taiga_destroy.
 *  - All kernels are enqueued on the ctx's stream and the caller synchronises.  Exceptions:
 *    taiga_load_field / taiga_load_efield / taiga_load_loss wait for the upload of HOST input arrays (so that the
 *    caller may reuse them on return; device inputs are not synchronised, and every table is built on the device);
 *    taiga_trace only enqueues (its counters reach the host when taiga_get_stats asks for them, which waits for the
 *    stream; the "stats" option = 1 makes taiga_trace itself wait, off by default);
 *    taiga_field_table and the taiga_measure_* calls always synchronise.  Small host tables (CDFs, detector edges) are staged
 *    through a pinned buffer of the ctx and never synchronise.
 *  - Coordinates: right-handed Cartesian (X,Y,Z), Z vertical, torus axis = Z,
 *    R = sqrt(X^2+Y^2); (R,phi,Z) right-handed; SI units.
 *  - There is no CPU fallback: every entry point needs an sm_100 device.
 */
#ifndef TAIGA_H
#define TAIGA_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TAIGA_OK        0
#define TAIGA_E_ARG    -1   /* null pointer, bad shape, non-monotone CDF, non-orthonormal frame */
#define TAIGA_E_STATE  -2   /* call order: e.g. trace before load_field                        */
#define TAIGA_E_CUDA   -3   /* a CUDA runtime call or kernel failed                            */
#define TAIGA_E_NOMEM  -4   /* device allocation failed                                        */

/* per-ion result codes written to taiga_ions.cell ("a segment ID
 * value or an error indicator") */
#define TAIGA_CELL_MISS      -1  /* crossed the plane, no segment (gap / outside); also the
                                    value taiga_trace leaves for every plane-crossing ion until
                                    taiga_detector_histogram assigns the segment              */
#define TAIGA_CELL_MAXSTEPS  -2  /* max_steps reached (trapped)                                */
#define TAIGA_CELL_OUT       -3  /* left the field grid                                        */
#define TAIGA_CELL_BADSTART  -4  /* starts on/behind the plane or outside the grid             */
/* taiga_ions.flags bits: results within 1e-9 m of a decision boundary */
#define TAIGA_FLAG_EDGE   1      /* hit within 1e-9 m of a segment edge                        */
#define TAIGA_FLAG_PLANE  2      /* |s| < 1e-9 m at an end of the crossing step                */
#define TAIGA_FLAG_GRID   4      /* within 1e-9 m of the grid boundary when leaving it         */

typedef struct taiga_ctx taiga_ctx;

/* device: CUDA ordinal; cuda_stream: a cudaStream_t (0 = default stream). */
int  taiga_create(taiga_ctx** out, int device, void* cuda_stream);
int  taiga_destroy(taiga_ctx* ctx);
const char* taiga_last_error(const taiga_ctx* ctx);

/* ---- a1: field tables (PAPER.md "bicubic B-spline fitted to the grid points ... the
 * coefficients are calculated and stored during the initialization"; L312; L65 toroidal
 * symmetry).  Interpolating tensor-product cubic spline with not-a-knot ends in R and Z
 * (reading A4), each of B_R, B_Z, B_phi separately (A5).
 *   kind 0: static (R,Z).  kind 1: nS time slices, linear in t, held outside [s0, s0+(nS-1)ds]
 *   (A16).  kind 2: nS toroidal planes spanning ONE period nS*ds, periodic cubic spline in phi
 *   (tricubic, A17).  Grids are uniform; node (i,j) sits at Rmin+i*hR, Zmin+j*hZ. */
typedef struct {
    int kind, nR, nZ, nS;            /* nR,nZ >= 4; nS = 1 (kind 0), >= 2 (kind 1), 3 ... 128 (kind 2) */
    double Rmin, Rmax, Zmin, Zmax;
    double s0, ds;                   /* first slice time, spacing [s]  |  phi0, dphi [rad]        */
} taiga_grid;

typedef struct {
    int form;        /* 0: nodal values [nS][nR][nZ] row-major -> the precompute kernel runs
                        1: ready per-cell power-basis coefficients, [nS][nR-1][nZ-1][16] (kind
                           0/1, index a*4+b of p^a w^b) or [...][64] (kind 2, c*16+a*4+b of
                           q^c p^a w^b): "read from the preprocessing database" mode (L312)   */
    const double *BR, *BZ, *Bphi;    /* three components, tesla                                  */
    int on_device;   /* 0: host pointers (copied inside the call)  1: dev pointers               */
} taiga_coeffs;

int taiga_load_field(taiga_ctx* ctx, const taiga_grid* grid, const taiga_coeffs* coeffs);

/* test / inspection hooks for a1: evaluate (B_R,B_Z,B_phi) at n points (dev arrays; s = time
 * or phi, may be null), and copy the internal per-cell table of one component back in the
 * form-1 layout above (host buffer of nS*(nR-1)*(nZ-1)*{16|64} doubles). */
int taiga_field_eval(taiga_ctx* ctx, uint64_t n, const double* R_dev, const double* Z_dev,
                     const double* s_dev, double* BR_dev, double* BZ_dev, double* Bphi_dev);
int taiga_field_table(taiga_ctx* ctx, int component, double* table_host);

/* ---- ion storage: SoA, dev, caller-owned, length n each.  x..vz are written by
 * taiga_seed_beam and only read by taiga_trace (so one seeding can be traced against several
 * detectors).  group/t0 may be null in taiga_trace / taiga_detector_histogram (=> 0). */
typedef struct {
    double *x, *y, *z, *vx, *vy, *vz;    /* initial position [m], velocity [m/s]              */
    double *hit_u, *hit_w;               /* detector-plane coordinates of the hit [m]          */
    int32_t *cell;                       /* segment iw*nu+iu, or TAIGA_CELL_*                  */
    uint32_t *steps;                     /* RKN steps taken                                    */
    uint8_t *flags;                      /* TAIGA_FLAG_*                                       */
    uint16_t *group;                     /* histogram index (energy / time slice)              */
    double *t0;                          /* birth time [s] (kind-1 fields)                     */
    double *weight;                      /* w0 x surviving fraction after secondary ionisation, written
                                            by taiga_trace when a loss model is loaded; may be null */
    double *w0;                          /* initial statistical weight (deterministic initialisation:
                                            written by taiga_seed_beam_grid); null = 1             */
    uint64_t n;                          /* < 2^32                                             */
} taiga_ions;

/* ---- a2: beam seeding (PAPER.md L314 stochastic initialisation: "the primary attenuation
 * profile as a cumulative distribution function ... randomly sampling it", on the GPU;
 * L128-134 linear beam model: ionisation depends on the position along the beam only).
 * Ion j (0 <= j < ions->n) uses Philox4x32-10 with key=(seed lo,hi), counters
 * (i lo, i hi, b, 0), b=0,1,2, i = first_index + j; five 52-bit uniforms; every draw is a
 * tabulated-CDF inversion with linear interpolation (bit-identical on any IEEE machine):
 *   depth d along `axis` from cdf_depth; cross-section offsets sigma_pos*(z1 eT + z2 eZ) and
 *   divergence angles sigma_ang*(z3, z4) from cdf_normal (table on [-z_max, z_max]);
 *   speed v0 = sqrt(2 energy_eV e / m) with e = charge_C.
 * profile = TAIGA_PROFILE_DISC ("a ... beam with a 5 mm diameter"): the cross-section
 *   offset is radius_m (a eT + c eZ) with (a, c) uniform over the unit disc, by rejection from the square:
 *   try 0 = (2 U_1 - 1, 2 U_2 - 1), try k >= 1 = two fresh uniforms from counter (i lo, i hi, 2 + k, 0),
 *   accepted when a^2 + c^2 <= 1 (64 tries at most, then the axis); depth and divergence as above.
 * CDF tables: host pointers, K+1 entries, F[0]=0, F[K]=1, non-decreasing; read during the call, the copy to the
 * device is enqueued on the context's stream from a context-owned staging buffer, so the caller may free or
 * change them as soon as the call returns. */
#define TAIGA_PROFILE_GAUSSIAN 0
#define TAIGA_PROFILE_DISC 1
typedef struct {
    double mass_kg, charge_C, energy_eV;
    double origin[3], axis[3], eT[3], eZ[3];       /* orthonormal (axis, eT, eZ)              */
    const double* cdf_depth;  int n_depth;  double depth_max;
    const double* cdf_normal; int n_normal; double z_max;
    double sigma_pos_m, sigma_ang_rad;
    uint64_t first_index;
    uint16_t group; double t0;                     /* written to ions->group / ions->t0       */
    int profile;                                   /* TAIGA_PROFILE_*                         */
    double radius_m;                               /* disc radius (TAIGA_PROFILE_DISC), > 0   */
} taiga_beam_params;

int taiga_seed_beam(taiga_ctx* ctx, const taiga_beam_params* params, uint64_t seed,
                    taiga_ions* ions);

/* Deterministic initialisation ("we define a grid with representative ions along the
 * beam, and each virtual ion gets a weight according to the ionization density function").
 * Reading D1: nd x nT x nZ cells -- depth cell k = depth_max [k, k+1]/nd along `axis`, cross-section
 * cells of width 2 z_lim/nT (2 z_lim/nZ) in units of sigma_pos spanning +-z_lim; the ion sits at the
 * cell centre, flies along `axis` (sigma_ang ignored) and gets ions->w0 = product of the increments
 * of the tabulated CDFs over the cell (linear between table points).  Ion j of the call is grid
 * index i = first_index + j = (k nT + a) nZ + b; first_index + ions->n <= nd nT nZ.  ions->w0 must
 * not be null.  No random numbers are drawn. */
typedef struct { int nd, nT, nZ; double z_lim; } taiga_seed_grid;
int taiga_seed_beam_grid(taiga_ctx* ctx, const taiga_beam_params* params, const taiga_seed_grid* grid,
                         taiga_ions* ions);

/* ---- detector (plane normal + perpendicular grid of segments with optional
 * non-uniform size and gaps; coordinate transformation to the plane).  u = (p-origin).eu,
 * w = (p-origin).ew.  Segment k of an axis is the half-open interval [lo[k], hi[k]); segments
 * must be ordered and non-overlapping.  Edge arrays are host pointers. */
typedef struct {
    double origin[3], normal[3], eu[3], ew[3];     /* orthonormal (normal, eu, ew)            */
    int nu, nw;
    const double *u_lo, *u_hi, *w_lo, *w_hi;
} taiga_detector;

/* ---- a3 + a4: integrator and termination (Eq. 3; Eq. 5-6 L218-235 with
 * readings A1-A3; L326 stop at the plane or at max_steps; L338 two-state storage and linear
 * interpolation to the plane; L318 error value).  charge_C/mass_kg of the LAST
 * taiga_seed_beam call is NOT implied: q/m is passed explicitly.
 * Writes hit_u, hit_w, cell (TAIGA_CELL_MISS for every plane-crossing ion, or an error code),
 * steps, flags.
 * solver: 0 = Runge-Kutta-Nystrom, classical stages (default reading A1; the production path),
 *         1 = RKN with the k3 position increment from k2 (Eq. 6 as printed),
 *         2 = linearised fourth-order Runge-Kutta on y = (r, v) (Eq. 4),
 *         3 = Boris-Verlet (Eq. 7-8) in its leap-frog form: r(t0+dt) = r(t0) + v' dt,
 *             v(t0) moved to t0 - dt/2 by one Boris push at the start (reading R2: "a
 *             second-order Verlet solver"),
 *         4 = Boris with Eq. 8 exactly as printed: r(t0+dt) = r(t0) + v(t0) dt (first order).
 * E of Eq. 3 is the uniform field set by taiga_set_efield (default 0) plus the gridded field of taiga_load_efield (default none). */
int taiga_trace(taiga_ctx* ctx, taiga_ions* ions, double q_over_m, double dt,
                uint32_t max_steps, const taiga_detector* det, int solver);

/* Uniform electric field E [V/m] of Eq. 3 ("we can use parametric modeling
 * for it"; verification scenarios 2 and 5, L279, L282).  Host pointer, copied.  Applies to all
 * later taiga_trace calls of this ctx; (0,0,0) restores the E = 0 production kernels. */
int taiga_set_efield(taiga_ctx* ctx, const double E_V_per_m[3]);

/* Gridded electric field E(R, Z) [V/m] of Eq. 3 (E(r); L177: the Cartesian coordinates "are mapped to a
 * poloidal cross-section plane in each iteration step.  That is how the local magnetic and electric field is given"; L175:
 * a parametric model of E near the wall is tabulated on the grid by the caller).  Reading E1: nodal values
 * E_R, E_Z, E_phi on the (R, Z) nodes of the LOADED magnetic field's grid, c->form = 0, arrays [nR][nZ] (one static slice
 * whatever the kind of B) in c->BR, c->BZ, c->Bphi, host or device (c->on_device); interpolated by the same not-a-knot
 * bicubic spline as B (a1's kernels), the boundary cell extrapolating outside the grid, rotated to Cartesian components like
 * B and ADDED to the uniform field of taiga_set_efield at every stage of every solver (Boris: at r(t0), as B).  c == NULL
 * removes it.  Must follow taiga_load_field (TAIGA_E_STATE otherwise); a later taiga_load_field removes it.  The table is
 * gathered per evaluation (48 coefficients through L1, no register cache): meant for edge studies, not for the production
 * E = 0 path, whose kernels are unchanged.  fp64 only, like the uniform E: taiga_trace refuses "precision" = 32 while either is set. */
int taiga_load_efield(taiga_ctx* ctx, const taiga_coeffs* c);

/* ---- a5: binning + histogram (segment ID per ion; atomically summed
 * per-segment counters; only the compact counter array is returned).
 * counts_dev [n_hist][nw][nu] and summary_dev [n_hist][6] = {hit, miss, maxsteps, out,
 * badstart, flagged} are ACCUMULATED into (caller zeroes).  Rewrites ions->cell for plane
 * crossers (segment id or TAIGA_CELL_MISS) and ORs TAIGA_FLAG_EDGE into ions->flags. */
int taiga_detector_histogram(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det,
                             int n_hist, unsigned long long* counts_dev,
                             unsigned long long* summary_dev);

/* The same binning for callers that are not allowed to allocate GPU or pinned memory.  taiga_detector_histogram keeps a
 * device copy of the segment edges in a buffer of the context that it creates on first use and replaces when a larger
 * detector arrives (cudaMalloc / cudaFree), and stages the edges through a pinned buffer (cudaMallocHost).  That rules it
 * out in two places this library is meant for: a between-shot or in-shot evaluation loop that shares the GPU with other
 * streams and must never stall them (cudaMalloc and cudaFree make the whole device wait), and a process whose memory pool
 * -- torch's caching allocator, a control system's fixed partition -- already owns the device's memory, where a late
 * cudaMalloc just fails.  This entry point calls no cudaMalloc, cudaMallocHost, cudaFree or any other allocating routine:
 * its edge table is a fixed array inside the library image, TAIGA_STATIC_MAX_SEGMENTS * 2 doubles = 32 KB, which every GPU
 * that loads libtaiga.so holds until the process exits.  Arguments, outputs, accumulation and results are exactly those of
 * taiga_detector_histogram (same kernel); ions, counts_dev and summary_dev remain the caller's.
 *  - Limit: det->nu + det->nw <= TAIGA_STATIC_MAX_SEGMENTS, else TAIGA_E_ARG with a message naming the limit (nothing
 *    is enqueued).
 *  - First call on a device: looks up the device address of the array (cudaGetSymbolAddress, no allocation).  Make that
 *    first call during set-up, before any stream capture is begun.
 *  - The edge arrays are copied from the caller's host memory by four cudaMemcpyAsync on the ctx's stream; ordinary
 *    (pageable) arrays have been read when the call returns, pinned ones must stay valid until the stream reaches the copy.
 *  - The array is shared by every context and every call on that GPU and keeps what the last call wrote.  Nothing in
 *    it has to start at zero -- each call rewrites every entry its kernel reads -- but two calls that overlap on the GPU
 *    (different streams, or host threads with different contexts on one device) race on it: keep all calls on one
 *    device in one stream, or order them with events. */
#define TAIGA_STATIC_MAX_SEGMENTS 2048
int taiga_detector_histogram_static(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det,
                                    int n_hist, unsigned long long* counts_dev,
                                    unsigned long long* summary_dev);

/* ---- secondary-ionisation loss (PAPER.md III.C, Eq. 2; L177: "numerically integrated with
 * every step using the one-dimensional secondary ionization profile"; L350 weighting).
 * taiga_load_loss builds (i) the bicubic spline table of the poloidal flux psi(R,Z) from nodal values
 * [nR][nZ] on the (R,Z) grid of the field loaded before (any kind; psi is static and axisymmetric),
 * (ii) the rate profile nu_k = n_e,k sqrt(t) exp(-1/t) / (E12^1.5 (6+t)) 1e-11 [1/s], t = T_e,k/E12
 * (Eq. 2) at psi0 + k dpsi, k < n; nu(psi) is linear in between and held constant outside.
 * While a loss model is loaded and ions->weight is not null, taiga_trace (every solver, with or without E; fp64)
 * also writes weight = w0 exp(-integral of nu dt) (w0 = 1 when ions->w0 is null), the integral taken
 * by the trapezoidal rule over the step end points, the crossing step counted up to the plane with nu
 * interpolated linearly
 * (reading L2); ions that do not cross keep the weight of their completed steps (1 for bad starts).
 * psi_nodal = NULL unloads the model.  ne / Te: host pointers; psi_nodal host or dev. */
typedef struct {
    int n;                               /* >= 2 profile points                                   */
    double psi0, dpsi;                   /* psi of point 0 and spacing (dpsi > 0), same unit as psi_nodal */
    const double *ne_m3, *Te_eV;         /* electron density [m^-3] and temperature [eV]          */
    double E12_eV;                       /* second ionisation energy of the beam species           */
} taiga_loss_profile;
int taiga_load_loss(taiga_ctx* ctx, const double* psi_nodal, int psi_on_device,
                    const taiga_loss_profile* profile);

/* Weighted counters (L350): every plane-crossing ion adds q = floor(weight 2^32 + 1/2) (32.32 fixed
 * point: integer sums, independent of the order of the atomics) to wcounts_dev[n_hist][nw][nu] at
 * its segment (weight = ions->weight if not null, else ions->w0); wsummary_dev[n_hist][4] = {sum q in
 * segments, sum q of crossers outside the segments, sum floor(q^2 / 2^32) over crossers, number of
 * crossers}.  Both are ACCUMULATED into.  Weights outside [0, 2^20] (reading L3': weights are probability masses
 * or counts) are clamped: negative and NaN count as 0, larger ones as 2^20; ions whose group is >= n_hist are
 * skipped (as in taiga_detector_histogram).
 * Call after taiga_detector_histogram (uses ions->cell); needs ions->weight or ions->w0.  A non-null
 * ions->weight must lie inside a weight array that one of the 16 most recent taiga_trace calls of this context wrote
 * (a loss model loaded) and that no later trace without a loss model has gone over, else TAIGA_E_STATE: weights of
 * your own go in w0, with weight = NULL. */
int taiga_detector_histogram_weighted(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det,
                                      int n_hist, unsigned long long* wcounts_dev,
                                      unsigned long long* wsummary_dev);

/* Mean and spread of the secondary-ionisation loss 1 - weight/w0... over the plane-crossing ions of one histogram,
 * the form of PAPER.md Table 1 (L147-158), from its four fixed-point sums wsummary_host[4] (HOST memory, read
 * back by the caller): mean weight mu = (s0 + s1) / 2^32 / N, variance s2 / 2^32 / N - mu^2 (>= 0), N = s3
 * (the division by N the paper does on the CPU, L350).  out_host[0] = 1 - mu, out_host[1] = sqrt(variance),
 * out_host[2] = N.  No device work. */
int taiga_loss_statistics(const unsigned long long wsummary_host[4], double out_host[3]);

/* ---- tuning / measurement hooks (not part of the method) */
/* integer options: "sort" (1: order the ion queue by birth cell before tracing, default 1),
 * "sort_sub" (sort bins per grid cell and axis, default 16), "min_active" (a warp refills its
 * free lanes from the queue when at least this many are free; 32 = whole tiles, default),
 * "ctas_per_sm", "variant" (kernel variant: 0 register cell cache with rolling predictive refill,
 * 8 warps/SM in 32-thread CTAs (default); 4 predictive refill after each evaluation; 5 refill on demand only; 3 the
 * same at 12 warps/SM; 1 / 2 no cache at 8 / 16 warps/SM; 7 the same in 128-thread CTAs at 223 registers; time-sliced fields: 0 time-blended cell
 * cache in registers with the slice difference in per-lane shared-memory slots (default), 6 the same
 * with the difference gathered through L1, 4 slice cache with rolling refill), "stats" (1: taiga_trace waits for its
 * counters itself; default 0: taiga_get_stats does), "precision" (64 default; 32 = the fp32 variant of BASELINE config 5: kind-2 fields
 * with the RKN solver only, tricubic evaluation and its table in fp32, cell location and the ion
 * state in fp64; offered for that accuracy statement, not for speed: it is slower than fp64 on the cooperative tracer (8.5 s against 6.7 s on BASELINE config 5); hit coordinates then agree with fp64 to 1e-5 m, integer outputs are not
 * bit-exact; taiga_trace returns TAIGA_E_ARG for other kinds / solvers), "plane_interp" (0 default:
 * linear interpolation to the detector plane; 1: quadratic Bezier through r_n, r_n+1 with the
 * control point at the mean of r_n + v_n dt/2 and r_n+1 - v_n+1 dt/2, reading Z1;
 * RKN solvers (the Boris velocities live at half steps), with or without E and the loss model (whose crossing step then
 * counts up to the curve parameter of the hit)), "mma" (kinds 1 and 2, fp64: 1 = warp-cooperative evaluation on the FP64
 * tensor pipe (trace_mma.cu; default for kind 2; kind-2 tables with planes more than 0.04 rad apart always take the other path), 0 = one lane evaluates its own ion (trace.cu; default for kind 1),
 * -1 = the default of the kind), "regroup" (kinds 1 / 2: the CTA re-sorts its 128 ions over its lanes by field cell
 * every this many steps, so that the lanes of a warp / of an 8-ion group share cells; default 8; with mma = 0, 0 = off:
 * per-warp tiles), "refill_cta" (mma: the CTA refills its finished lanes from the queue at a re-sort point once this
 * many are free; default: all of them, i.e. whole tiles of consecutive queue entries, which keeps the ions of a CTA
 * in few cells -- 9.4e9 against 7.5e9 ion-steps/s with 16 on BASELINE config 5), "mma_geom" (mma, plain RKN kernel: threads per
 * CTA x register cap: 0 = 128 x 128, four CTAs per SM (default); 1 = 128 x 168; 2 = 64 x 144; 3 = 32 x 144; 4 = 32 x 128;
 * 5 = 64 x 128).  Values out of range are refused with TAIGA_E_ARG when set. */
int taiga_set_option(taiga_ctx* ctx, const char* key, long long value);
/* counters of the last taiga_trace; waits for the ctx's stream when that trace has not been collected yet: [0] ion-steps, [1] warp-steps*32
 * (lane slots issued), [2] 1, [3] kernel launches, [4] cell refills, [5..7] 0. */
int taiga_get_stats(taiga_ctx* ctx, unsigned long long stats_host[8]);
/* register-resident DFMA microkernel: measured FP64 FMA instructions per second (thread-level,
 * i.e. lanes x instr) over ~`ms` milliseconds; the roofline denominator. */
int taiga_measure_fp64_peak(taiga_ctx* ctx, double ms, double* dfma_per_s);
/* the same for the FP64 tensor pipe: DMMA.8x8x4 chains, FMA per second (256 per warp instruction); the
 * denominator of the warp-cooperative tracer of kinds 1 and 2. */
int taiga_measure_dmma_peak(taiga_ctx* ctx, double ms, double* fma_per_s);
/* DFMA and DMMA chains interleaved 1 : 1 in FMA count: total FMA per second.  It does not exceed the DFMA rate (one
 * FP64 datapath per SM serves both), which is why every kernel is reported against 148 x 64 FMA/clk. */
int taiga_measure_mixed_fp64_peak(taiga_ctx* ctx, double ms, double* fma_per_s);
/* L1-resident gather microkernel shaped like the uncached field evaluation (8 warps/SM, 48 x 256-bit
 * loads of a 1536-B cell per lane): bytes per second delivered to registers; `spread` = distinct cells
 * read by the lanes of a warp (1 ... 32).  The roofline denominator of the kind-1 / kind-2 kernels. */
int taiga_measure_l1_gather_peak(taiga_ctx* ctx, double ms, int spread, double* bytes_per_s);

#ifdef __cplusplus
}
#endif
#endif
