// a3 + a4 for the (R, Z, phi) tables of kind 2 (the default there) and, on request ("mma" = 1), the time slices of
// kind 1, which default to k_trace (trace.cu): the field evaluation as a small FP64 tensor-core product,
// coefficients delivered ONCE PER WARP instead of once per lane.
//
// PAPER.md L63 (stored spline coefficients), L177 (field interpolated at every stage), Eq. 5-6; L47 and
// L406-408 (perturbed, non-axisymmetric fields are what the GPU solver is for).
//
// Why.  B_m = sum_{a,b,c} C_m[c][a][b] p^a w^b q^c needs 192 coefficients per evaluation (kind 2; 96 for the
// two slices of kind 1).  With one lane evaluating its own ion, every lane receives its own copy of them
// through the L1 data pipe even when the whole warp sits in one cell: 1536 B per lane and evaluation against a
// 128 B/clk/SM register write-back port, 4x the time the FP64 pipe needs (profiles/r1d_other_configs.md: L1
// data pipe 78 % busy, FP64 pipe 18 %).  DMMA.8x8x4 runs at the DFMA rate on B200 (measured 0.994 of 148 x 64
// FMA/clk, profiles/r2a_microbench.md) but reads each operand register for 8 FMAs, and its B operand is
// shared by 8 ions.  So:
//
//   per group of 8 ions (rows) in one cell:   D[ion][(a, c0)] = sum_{b, c1} (w^b q^(2 c1)) C_m[2 c1 + c0][a][b]
//       A[ion][k = b]      = w^b                  k-step 0   (kind 2 adds k-step 1: w^b q^2)
//       B[k = b][n = 2a+c0] = coefficient          one 8x8x4 DMMA per component m and k-step: 6 (kind 2) / 3 (kind 1)
//   the lane (ion r, t) of the quad that holds row r gets D[r][2t], D[r][2t+1] = the a = t terms for c0 = 0, 1,
//   forms f_m[t] = D0 + q D1 (kind 1: c0 is the slice, q = tau, D1 the slice difference) and hands the three
//   f_m[t] to the ion's own lane through shared memory; that lane finishes with the Horner sum in p over t.
//
// The warp holds 32 ions, one per lane (state in registers, as in trace.cu); ion (g, r) = group g, row r sits in
// lane 4r + g, i.e. inside the quad that receives its results.  The coefficients of a cell are 6 (3) coalesced
// 256-B loads per WARP from a copy of the table in B-fragment order; lanes of a warp in different cells are
// served cell by cell (warp-uniform loop, ballot + leader), so the cost is one DMMA set per (cell, group) pair.
// To keep that number near 4 per evaluation the CTA re-sorts its ions over its lanes by field cell every few
// steps through shared memory (as trace.cu's REGROUP), and at the same points refills finished lanes from the
// birth-cell-ordered queue, so all warps stay full through the tail.
#include "trace_common.cuh"

#define TG_IDX(L) ((L) + 2 * ((L) >> 4))          // skewed slot of lane L: quad-strided 64-bit reads hit distinct banks
#define TG_ROW 35                                 // row stride of the per-warp buffer: 34 slots; 35 = 3 mod 16 keeps the 16 lanes
                                                  // of a half-warp (rows r = 0..3 or 4..7, t = 0..3) on distinct 8-byte banks
#define TG_ROWB (TG_ROW * 8)                      // ... in bytes

// Per-warp exchange buffer, rows of TG_ROW doubles indexed by the slot of an ion's own lane:
//   rows 0..7   A operands [s * 4 + t] = w^t q^(2s)        row 8   q (kind 2) / tau (kind 1)
//   rows 9..20  results f[m * 4 + t]
// followed by the work list of the current evaluation: 32 descriptors {cell, member lanes, 8 g, -}.
#define TG_LIST_OFF ((21 * TG_ROW + 1) * 8)
struct __align__(16) TgWarpBuf { double v[21 * TG_ROW + 1]; int4 list[32]; };

// Shared-memory addresses of one lane, computed once per kernel: ptxas otherwise rematerialises them from
// %tid / the CTA's window base inside the item loop (60 integer instructions per 6 DMMAs in the r2a profile).
struct TgLane {
    unsigned own;                                 // &v[slot of my lane]                  (my ion's column)
    unsigned quad;                                // &v[t * TG_ROW + slot of lane 4r]     (+ 8 g: column of ion (g, r), row t)
    unsigned qrow;                                // &v[8 * TG_ROW + slot of lane 4r]
    unsigned bit0;                                // 1 << 4r: bit of ion (0, r) in a lane mask
    unsigned list;                                // the warp's work list
    unsigned lane;
    const double* frag;                           // fragment table + lane
};

__device__ __forceinline__ double tg_lds(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ void tg_sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void tg_lds4(unsigned a, int& x, unsigned& y, unsigned& z) {
    [[maybe_unused]] int w;                   // fourth word of the descriptor: padding
    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(w) : "r"(a));
}
__device__ __forceinline__ void tg_sts4(unsigned a, int x, unsigned y, unsigned z) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%3};" ::"r"(a), "r"(x), "r"(y), "r"(z) : "memory");
}

__device__ __forceinline__ void tg_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// cell id (index into the fragment table) and in-cell coordinates; same arithmetic as tg_field_cyl
template <int KIND>
__device__ __forceinline__ int tg_locate_cell(const FieldDev& f, double X, double Y, double Z, double R, double t,
                                              double& p, double& w, double& q) {
    int i = tg_locate(R, f.inv_hR, f.offR, f.cR, p);
    int j = tg_locate(Z, f.inv_hZ, f.offZ, f.cZ, w);
    if constexpr (KIND == 2) {
        double xs = (atan2(Y, X) - f.s0) * f.inv_ds;
        xs = xs - (double)f.nS * floor(xs / (double)f.nS);
        int k = tg_clampi(__double2int_rd(xs), 0, f.nS - 1);
        q = xs - (double)k;
        return (k * f.cR + i) * f.cZ + j;
    } else {
        double xs = (t - f.s0) * f.inv_ds;
        int k = tg_clampi(__double2int_rd(xs), 0, f.nS - 2);
        q = fmin(fmax(xs - (double)k, 0.0), 1.0);
        return (i * f.cZ + j) * (f.nS - 1) + k;
    }
}

// Kind 2 without atan2.  The ion carries K, the global index of the toroidal cell it is in (K ds <= phi - s0 < (K+1) ds,
// NK = 2 pi / ds cells around the torus), and (c0, s0) = (cos, sin) of that cell's lower plane from a table (k_phi_tab).
// For a point (X, Y) the angle past the plane is small, delta = asin((Y c0 - X s0) / R) with |delta| <~ ds, so
// q = delta / ds is a 4-term series in s = (Y c0 - X s0) / R (1/R is needed anyway): 10 FP64 instructions instead of the
// ~65 of atan2 + modulo.  A point beyond the cell moves K (and the frame) by floor(q) and is evaluated again.
struct TgTor { int K, k; double c0, s0; };       // k = K mod nS: plane index of the table

__device__ __forceinline__ void tg_tor_set(const TraceParams& P, TgTor& T, int K) {
    T.K = K; T.k = K % P.f.nS;
    const double2 cs = __ldg(P.phi_tab + K);
    T.c0 = cs.x; T.s0 = cs.y;
}
// K of a point from scratch (ion load): the definition, with atan2
__device__ __forceinline__ int tg_tor_K(const TraceParams& P, double X, double Y) {
    double xs = (atan2(Y, X) - P.f.s0) * P.f.inv_ds;
    xs = xs - (double)P.phi_n * floor(xs / (double)P.phi_n);
    return tg_clampi(__double2int_rd(xs), 0, P.phi_n - 1);
}
__device__ __forceinline__ int tg_locate_tor(const TraceParams& P, TgTor& T, double X, double Y, double Z, double R, double rinv,
                                             double& p, double& w, double& q) {
    const FieldDev& f = P.f;
    int i = tg_locate(R, f.inv_hR, f.offR, f.cR, p);
    int j = tg_locate(Z, f.inv_hZ, f.offZ, f.cZ, w);
#pragma unroll 1
    for (int it = 0;; ++it) {
        const double s = fma(Y, T.c0, -(X * T.s0)) * rinv, s2 = s * s;
        q = (s * fma(s2, fma(s2, fma(s2, 15.0 / 336.0, 3.0 / 40.0), 1.0 / 6.0), 1.0)) * f.inv_ds;   // asin(s) / ds
        if (tg_in01(q)) break;
        if (it == 3) { q = fmin(fmax(q, 0.0), 0x1.fffffffffffffp-1); break; }   // on a plane to rounding: either side evaluates the same (C2 spline)
        if (!(fabs(q) < 4.0)) { tg_tor_set(P, T, tg_tor_K(P, X, Y)); continue; }  // far off (never for steps shorter than a cell): from scratch
        int K = T.K + __double2int_rd(q);
        K = K < 0 ? K + P.phi_n : (K >= P.phi_n ? K - P.phi_n : K);
        tg_tor_set(P, T, K);
    }
    return (T.k * f.cR + i) * f.cZ + j;
}

// Warp-collective evaluation: every lane calls it; cell < 0 = this lane has no ion to evaluate.
// Work items = (cell, group) pairs: the ions of one group (lanes 4r + g) that sit in one cell.  The whole list of an
// evaluation is built up front from one match.any (lanes in the same cell) and one ballot (the lowest lane of each
// pair writes its descriptor), so the DMMA loop carries no vote / shuffle chain; descriptors and operands are fetched
// one item ahead, into the registers the issued DMMAs have already read.
template <int KIND>
__device__ __forceinline__ void tg_eval_mma(const TgLane& L, int cell, double p, double w, double q,
                                            double& BR, double& BZ, double& Bp, unsigned& sets) {
    constexpr int KS = (KIND == 2) ? 2 : 1;
    const unsigned FULL = 0xffffffffu;
    {                                             // my ion's monomials and q into the warp buffer
        const double w2 = w * w, w3 = w2 * w;
        tg_sts(L.own, 1.0); tg_sts(L.own + TG_ROWB, w); tg_sts(L.own + 2 * TG_ROWB, w2); tg_sts(L.own + 3 * TG_ROWB, w3);
        if constexpr (KS == 2) {
            const double q2 = q * q;
            tg_sts(L.own + 4 * TG_ROWB, q2); tg_sts(L.own + 5 * TG_ROWB, w * q2);
            tg_sts(L.own + 6 * TG_ROWB, w2 * q2); tg_sts(L.own + 7 * TG_ROWB, w3 * q2);
        }
        tg_sts(L.own + 8 * TG_ROWB, q);
    }
    const unsigned mine_g = __match_any_sync(FULL, cell) & (0x11111111u << (L.lane & 3));   // my (cell, group) pair
    const bool lead = cell >= 0 && (mine_g & (0u - mine_g)) == (1u << L.lane);            // its lowest lane
    const unsigned leaders = __ballot_sync(FULL, lead);
    if (lead) tg_sts4(L.list + 16 * __popc(leaders & ((1u << L.lane) - 1u)), cell, mine_g, (L.lane & 3) * 8);
    __syncwarp();
    const int n_items = __popc(leaders);
    sets += n_items;
    double b[KS][3], a[KS], qg = 0.0;
    int cs = 0;
    unsigned mem = 0, gofs = 0;
    auto operands = [&]() {
        const double* src = L.frag + (size_t)cs * (KS * 96);
#pragma unroll
        for (int s = 0; s < KS; ++s)
#pragma unroll
            for (int m = 0; m < 3; ++m) b[s][m] = __ldg(src + (s * 3 + m) * 32);
#pragma unroll
        for (int s = 0; s < KS; ++s) a[s] = tg_lds(L.quad + gofs + s * 4 * TG_ROWB);
        qg = tg_lds(L.qrow + gofs);
    };
    if (n_items) { tg_lds4(L.list, cs, mem, gofs); operands(); }
    for (int i = 0; i < n_items; ++i) {           // warp-uniform
        int cs2 = 0; unsigned mem2 = 0, gofs2 = 0;
        if (i + 1 < n_items) tg_lds4(L.list + 16 * (i + 1), cs2, mem2, gofs2);
        double d[3][2];
#pragma unroll
        for (int m = 0; m < 3; ++m) { d[m][0] = 0.0; d[m][1] = 0.0; }
#pragma unroll
        for (int s = 0; s < KS; ++s)
#pragma unroll
            for (int m = 0; m < 3; ++m) tg_dmma(d[m][0], d[m][1], a[s], b[s][m]);
        const double qc = qg;
        const bool mine = mem & (L.bit0 << (gofs >> 3));       // the ion of my row is served by this item
        const unsigned o = L.quad + 9 * TG_ROWB + gofs;
        cs = cs2; mem = mem2; gofs = gofs2;
        if (i + 1 < n_items) operands();
        if (mine) {
#pragma unroll
            for (int m = 0; m < 3; ++m) tg_sts(o + m * 4 * TG_ROWB, fma(qc, d[m][1], d[m][0]));
        }
        __syncwarp();                             // the next DMMA is warp-collective
    }
    __syncwarp();
    if (cell >= 0) {
        const unsigned o = L.own + 9 * TG_ROWB;
        BR = fma(fma(fma(tg_lds(o + 3 * TG_ROWB), p, tg_lds(o + 2 * TG_ROWB)), p, tg_lds(o + TG_ROWB)), p, tg_lds(o));
        BZ = fma(fma(fma(tg_lds(o + 7 * TG_ROWB), p, tg_lds(o + 6 * TG_ROWB)), p, tg_lds(o + 5 * TG_ROWB)), p, tg_lds(o + 4 * TG_ROWB));
        Bp = fma(fma(fma(tg_lds(o + 11 * TG_ROWB), p, tg_lds(o + 10 * TG_ROWB)), p, tg_lds(o + 9 * TG_ROWB)), p, tg_lds(o + 8 * TG_ROWB));
    }
}

#define TG_KEY_DEAD 0x7fffff

// SOLVER / HAS_E / LOSS / BEZ as in trace.cu's k_trace.
template <int KIND, int THREADS, int MAXREG, int SOLVER, bool HAS_E, bool LOSS, bool BEZ>
__global__ void __launch_bounds__(THREADS) __maxnreg__(MAXREG) k_trace_mma(const TraceParams P) {
    constexpr int NW = THREADS / 32;
    constexpr int ND = LOSS ? 10 : 8;
    const unsigned FULL = 0xffffffffu;
    // the warp buffers (evaluation) and the exchange arrays of the CTA sync point (refill + re-sort) are never live at
    // the same time: one allocation, so that more of the SM's 256 KB stays L1 for the fragment table
    constexpr size_t EXCH_BYTES = (size_t)ND * THREADS * 8 + (size_t)(KIND == 2 ? 4 : 3) * THREADS * 4 + (size_t)THREADS * 4;
    constexpr size_t SMEM_BYTES = sizeof(TgWarpBuf) * NW > EXCH_BYTES ? sizeof(TgWarpBuf) * NW : EXCH_BYTES;
    __shared__ __align__(16) unsigned char s_raw[SMEM_BYTES];
    TgWarpBuf* s_wb = reinterpret_cast<TgWarpBuf*>(s_raw);
    double (*sh_d)[THREADS] = reinterpret_cast<double (*)[THREADS]>(s_raw);
    uint32_t (*sh_u)[THREADS] = reinterpret_cast<uint32_t (*)[THREADS]>(s_raw + (size_t)ND * THREADS * 8);
    int* sh_key = reinterpret_cast<int*>(s_raw + (size_t)ND * THREADS * 8 + (size_t)(KIND == 2 ? 4 : 3) * THREADS * 4);
    __shared__ unsigned long long s_base;
    __shared__ int s_wcnt[NW];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    TgLane L;
    {
        const unsigned wb = (unsigned)__cvta_generic_to_shared(&s_wb[warp]);
        const int t4 = lane & 3, slot0 = TG_IDX(lane & ~3);
        L.own = wb + TG_IDX(lane) * 8;
        L.quad = wb + t4 * TG_ROWB + slot0 * 8;
        L.qrow = wb + 8 * TG_ROWB + slot0 * 8;
        L.bit0 = 1u << (lane & ~3);
        L.list = wb + TG_LIST_OFF;
        L.lane = (unsigned)lane;
        L.frag = P.frag + lane;
    }

    double X = 0, Y = 0, Z = 0, Ux = 0, Uy = 0, Uz = 0, t = 0, s0 = -1.0;
    double Lam = 0.0, nu0 = 0.0;
    uint32_t idx = 0, nst = 0;
    bool alive = false, exhausted = false;
    [[maybe_unused]] TgTor T = {0, 0, 1.0, 0.0};
    unsigned sets = 0, ion_steps = 0;
    unsigned long long warp_steps = 0;
    int since = 0;

    // collective: Cartesian B at (Xs, Ys, Zs, ts) for the lanes with `alive`; Rs = cylindrical radius of the point
    auto field = [&](double Xs, double Ys, double Zs, double ts, double& bx, double& by, double& bz, double& Rs) {
        double p = 0.0, w = 0.0, q = 0.0, rinv = 0.0, BR = 0.0, BZ = 0.0, Bp = 0.0;
        int cell = -1;
        if (alive) {
            double R2 = fma(Xs, Xs, Ys * Ys);
            rinv = tg_rsqrt(R2); Rs = R2 * rinv;
            if constexpr (KIND == 2) cell = tg_locate_tor(P, T, Xs, Ys, Zs, Rs, rinv, p, w, q);
            else cell = tg_locate_cell<KIND>(P.f, Xs, Ys, Zs, Rs, ts, p, w, q);
        }
        tg_eval_mma<KIND>(L, cell, p, w, q, BR, BZ, Bp, sets);
        if (alive) { tg_rotate(Xs, Ys, rinv, BR, Bp, bx, by); bz = BZ; }
    };

    while (true) {
        if (since == 0) {                      // CTA sync point: refill finished lanes, re-sort the ions over the lanes by cell
            int nalive = __syncthreads_count(alive);
            if (nalive == 0 && exhausted) break;
            const int nfree = THREADS - nalive;
            if (!exhausted && nfree >= (P.refill_cta < THREADS ? P.refill_cta : THREADS)) {
                unsigned dm = __ballot_sync(FULL, !alive);
                if (lane == 0) s_wcnt[warp] = __popc(dm);
                if (tid == 0) s_base = atomicAdd(&P.counters[0], (unsigned long long)nfree);
                __syncthreads();
                int off = 0;
                for (int k = 0; k < warp; ++k) off += s_wcnt[k];
                unsigned long long q = s_base + off + __popc(dm & ((1u << lane) - 1u));
                if (s_base + nfree >= P.n) exhausted = true;
                if (!alive && q < P.n) {
                    idx = P.order ? P.order[q] : (uint32_t)q;
                    X = P.x[idx]; Y = P.y[idx]; Z = P.z[idx];
                    Ux = P.qm * P.vx[idx]; Uy = P.qm * P.vy[idx]; Uz = P.qm * P.vz[idx];
                    t = P.t0 ? P.t0[idx] : 0.0;
                    nst = 0;
                    if constexpr (LOSS) Lam = 0.0;
                    s0 = fma(P.det.normal[0], X, fma(P.det.normal[1], Y, fma(P.det.normal[2], Z, -P.nrD)));
                    alive = true;
                    if constexpr (KIND == 2) tg_tor_set(P, T, tg_tor_K(P, X, Y));
                    if (!(s0 < 0.0)) {             // O4: must start in front of the plane
                        P.hit_u[idx] = 0.0; P.hit_w[idx] = 0.0; P.cell[idx] = TAIGA_CELL_BADSTART; P.steps[idx] = 0;
                        P.flags[idx] = (fabs(s0) < TG_GRAZE) ? TAIGA_FLAG_PLANE : 0;
                        if constexpr (LOSS) P.weight[idx] = P.w0 ? P.w0[idx] : 1.0;
                        alive = false;
                    }
                }
            }
            // sort key: the field cell (unique keys: cell << 8 | tid), finished lanes last
            int key = TG_KEY_DEAD;
            if (alive) {
                double p_, w_, q_;
                int c;
                if constexpr (KIND == 2) {         // the toroidal cell the ion carries (at most one evaluation old)
                    const int ci = tg_locate(sqrt(fma(X, X, Y * Y)), P.f.inv_hR, P.f.offR, P.f.cR, p_);
                    const int cj = tg_locate(Z, P.f.inv_hZ, P.f.offZ, P.f.cZ, w_);
                    c = ((T.k * P.f.cR + ci) * P.f.cZ + cj) >> P.key_shift;
                } else c = tg_locate_cell<KIND>(P.f, X, Y, Z, sqrt(fma(X, X, Y * Y)), t, p_, w_, q_) >> P.key_shift;
                key = c < TG_KEY_DEAD - 1 ? c : TG_KEY_DEAD - 1;
            }
            const int mykey = (key << 8) | tid;
            sh_key[tid] = mykey;
            __syncthreads();
            int rank = 0;
#pragma unroll 4
            for (int o = 0; o < THREADS; o += 4) {
                int4 k4 = *reinterpret_cast<const int4*>(&sh_key[o]);
                rank += (k4.x < mykey) + (k4.y < mykey) + (k4.z < mykey) + (k4.w < mykey);
            }
            // sorted position -> lane: consecutive ions fill one group (lanes 4r + g, r = 0..7) after the other
            const int rho = rank & 31;
            const int dst = (rank & ~31) | ((rho & 7) << 2) | (rho >> 3);
            sh_d[0][dst] = X; sh_d[1][dst] = Y; sh_d[2][dst] = Z; sh_d[3][dst] = Ux; sh_d[4][dst] = Uy; sh_d[5][dst] = Uz;
            sh_d[6][dst] = t; sh_d[7][dst] = s0;
            if constexpr (LOSS) { sh_d[8][dst] = Lam; sh_d[9][dst] = nu0; }
            sh_u[0][dst] = idx; sh_u[1][dst] = nst; sh_u[2][dst] = alive ? 1u : 0u;
            if constexpr (KIND == 2) sh_u[3][dst] = (uint32_t)T.K;
            __syncthreads();
            X = sh_d[0][tid]; Y = sh_d[1][tid]; Z = sh_d[2][tid]; Ux = sh_d[3][tid]; Uy = sh_d[4][tid]; Uz = sh_d[5][tid];
            t = sh_d[6][tid]; s0 = sh_d[7][tid];
            if constexpr (LOSS) { Lam = sh_d[8][tid]; nu0 = sh_d[9][tid]; }
            idx = sh_u[0][tid]; nst = sh_u[1][tid]; alive = sh_u[2][tid] != 0u;
            if constexpr (KIND == 2) tg_tor_set(P, T, (int)sh_u[3][tid]);
            __syncthreads();                   // the exchange arrays share their memory with the warp buffers
        }
        since = (since + 1 >= P.regroup_every) ? 0 : since + 1;
        if (__ballot_sync(FULL, alive) == 0) continue;        // this warp idles until the next sync point
        ++warp_steps;

        // ---- stage 1 at (r, u); its grid test is the out-of-grid test of the previous step (O4)
        double Bx = 0, By = 0, Bz = 0, R = 0;
        field(X, Y, Z, t, Bx, By, Bz, R);
        double Xn = 0, Yn = 0, Zn = 0, nu1 = 0.0;
        double c1x = 0.0, c1y = 0.0, c1z = 0.0;          // BEZ: r_n + v_n dt/2
        if (alive) {
            bool outside = (R < P.f.Rmin) | (R > P.f.Rmax) | (Z < P.f.Zmin) | (Z > P.f.Zmax);
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
            }
            if constexpr (BEZ) { c1x = fma(Ux, P.a1, X); c1y = fma(Uy, P.a1, Y); c1z = fma(Uz, P.a1, Z); }
        }
        if constexpr (SOLVER == 0) {
            // Eq. 5-6 (readings A1-A3)
            double k1x = 0, k1y = 0, k1z = 0, k2x = 0, k2y = 0, k2z = 0, k3x = 0, k3y = 0, k3z = 0;
            double Xm = 0, Ym = 0, Zm = 0, ux = 0, uy = 0, uz = 0, Rd;
            if (alive) {
                k1x = fma(Uy, Bz, -(Uz * By)); k1y = fma(Uz, Bx, -(Ux * Bz)); k1z = fma(Ux, By, -(Uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, X, Y, Z, k1x, k1y, k1z);
                Xm = fma(k1x, P.a2, fma(Ux, P.a1, X)); Ym = fma(k1y, P.a2, fma(Uy, P.a1, Y)); Zm = fma(k1z, P.a2, fma(Uz, P.a1, Z));
                ux = fma(k1x, P.b1, Ux); uy = fma(k1y, P.b1, Uy); uz = fma(k1z, P.b1, Uz);
            }
            const double tm = t + 0.5 * P.dt;
            field(Xm, Ym, Zm, tm, Bx, By, Bz, Rd);             // stage 2 (and 3, classical: same position)
            if (alive) {
                k2x = fma(uy, Bz, -(uz * By)); k2y = fma(uz, Bx, -(ux * Bz)); k2z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xm, Ym, Zm, k2x, k2y, k2z);
                ux = fma(k2x, P.b1, Ux); uy = fma(k2y, P.b1, Uy); uz = fma(k2z, P.b1, Uz);
            }
            if (P.variant) {                   // printed Eq. 6: k3 position increment from k2 (kernel-uniform)
                if (alive) { Xm = fma(k2x, P.a2, fma(Ux, P.a1, X)); Ym = fma(k2y, P.a2, fma(Uy, P.a1, Y)); Zm = fma(k2z, P.a2, fma(Uz, P.a1, Z)); }
                field(Xm, Ym, Zm, tm, Bx, By, Bz, Rd);
            }
            double Xe = 0, Ye = 0, Ze = 0;
            if (alive) {
                k3x = fma(uy, Bz, -(uz * By)); k3y = fma(uz, Bx, -(ux * Bz)); k3z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xm, Ym, Zm, k3x, k3y, k3z);
                Xe = fma(k3x, 4.0 * P.a2, fma(Ux, 2.0 * P.a1, X)); Ye = fma(k3y, 4.0 * P.a2, fma(Uy, 2.0 * P.a1, Y));
                Ze = fma(k3z, 4.0 * P.a2, fma(Uz, 2.0 * P.a1, Z));
                ux = fma(k3x, 2.0 * P.b1, Ux); uy = fma(k3y, 2.0 * P.b1, Uy); uz = fma(k3z, 2.0 * P.b1, Uz);
            }
            field(Xe, Ye, Ze, t + P.dt, Bx, By, Bz, Rd);       // stage 4
            if (alive) {
                double k4x = fma(uy, Bz, -(uz * By)), k4y = fma(uz, Bx, -(ux * Bz)), k4z = fma(ux, By, -(uy * Bx));
                if constexpr (HAS_E) tg_add_qE(P, Xe, Ye, Ze, k4x, k4y, k4z);
                double Tx = k2x + k3x, Ty = k2y + k3y, Tz = k2z + k3z;
                Xn = fma(k1x + Tx, P.c6, fma(Ux, P.dtq, X)); Yn = fma(k1y + Ty, P.c6, fma(Uy, P.dtq, Y));
                Zn = fma(k1z + Tz, P.c6, fma(Uz, P.dtq, Z));
                Ux = fma(fma(2.0, Tx, k1x + k4x), P.d6, Ux);
                Uy = fma(fma(2.0, Ty, k1y + k4y), P.d6, Uy);
                Uz = fma(fma(2.0, Tz, k1z + k4z), P.d6, Uz);
            }
        } else if constexpr (SOLVER == 2) {
            // Eq. 4: classical RK4 on y = (r, v); see trace.cu
            double k1x = 0, k1y = 0, k1z = 0, k2x = 0, k2y = 0, k2z = 0, k3x = 0, k3y = 0, k3z = 0;
            double Xs = 0, Ys = 0, Zs = 0, ux = 0, uy = 0, uz = 0, Rd;
            if (alive) {
                k1x = fma(Uy, Bz, -(Uz * By)); k1y = fma(Uz, Bx, -(Ux * Bz)); k1z = fma(Ux, By, -(Uy * Bx));
                tg_add_qE(P, X, Y, Z, k1x, k1y, k1z);
                ux = fma(k1x, P.b1, Ux); uy = fma(k1y, P.b1, Uy); uz = fma(k1z, P.b1, Uz);
                Xs = fma(Ux, P.a1, X); Ys = fma(Uy, P.a1, Y); Zs = fma(Uz, P.a1, Z);
            }
            field(Xs, Ys, Zs, t + 0.5 * P.dt, Bx, By, Bz, Rd);
            if (alive) {
                k2x = fma(uy, Bz, -(uz * By)); k2y = fma(uz, Bx, -(ux * Bz)); k2z = fma(ux, By, -(uy * Bx));
                tg_add_qE(P, Xs, Ys, Zs, k2x, k2y, k2z);
                ux = fma(k2x, P.b1, Ux); uy = fma(k2y, P.b1, Uy); uz = fma(k2z, P.b1, Uz);
                Xs = fma(k1x, 2.0 * P.a2, fma(Ux, P.a1, X)); Ys = fma(k1y, 2.0 * P.a2, fma(Uy, P.a1, Y)); Zs = fma(k1z, 2.0 * P.a2, fma(Uz, P.a1, Z));
            }
            field(Xs, Ys, Zs, t + 0.5 * P.dt, Bx, By, Bz, Rd);
            if (alive) {
                k3x = fma(uy, Bz, -(uz * By)); k3y = fma(uz, Bx, -(ux * Bz)); k3z = fma(ux, By, -(uy * Bx));
                tg_add_qE(P, Xs, Ys, Zs, k3x, k3y, k3z);
                ux = fma(k3x, 2.0 * P.b1, Ux); uy = fma(k3y, 2.0 * P.b1, Uy); uz = fma(k3z, 2.0 * P.b1, Uz);
                Xs = fma(k2x, 4.0 * P.a2, fma(Ux, 2.0 * P.a1, X)); Ys = fma(k2y, 4.0 * P.a2, fma(Uy, 2.0 * P.a1, Y)); Zs = fma(k2z, 4.0 * P.a2, fma(Uz, 2.0 * P.a1, Z));
            }
            field(Xs, Ys, Zs, t + P.dt, Bx, By, Bz, Rd);
            if (alive) {
                double k4x = fma(uy, Bz, -(uz * By)), k4y = fma(uz, Bx, -(ux * Bz)), k4z = fma(ux, By, -(uy * Bx));
                tg_add_qE(P, Xs, Ys, Zs, k4x, k4y, k4z);
                double Tx = k2x + k3x, Ty = k2y + k3y, Tz = k2z + k3z;
                Xn = fma(k1x + Tx, P.c6, fma(Ux, P.dtq, X)); Yn = fma(k1y + Ty, P.c6, fma(Uy, P.dtq, Y));
                Zn = fma(k1z + Tz, P.c6, fma(Uz, P.dtq, Z));
                Ux = fma(fma(2.0, Tx, k1x + k4x), P.d6, Ux);
                Uy = fma(fma(2.0, Ty, k1y + k4y), P.d6, Uy);
                Uz = fma(fma(2.0, Tz, k1z + k4z), P.d6, Uz);
            }
        } else {
            // Eq. 7-8: Boris push with B, E at r(t0); see trace.cu
            if (alive) {
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
        // ---- a4: plane test, interpolation (L326, L338)
        bool crossed = false;
        double lam = 0.0, s1 = 0.0;
        if (alive) {
            ++nst; ++ion_steps;
            s1 = fma(P.det.normal[0], Xn, fma(P.det.normal[1], Yn, fma(P.det.normal[2], Zn, -P.nrD)));
            crossed = s1 >= 0.0;
        }
        if (crossed) {                         // O4: s0 < 0 <= s1
            lam = s0 / (s0 - s1);
            [[maybe_unused]] double frac = lam;     // fraction of the crossing step up to the plane (Bezier: its tau)
            double px = fma(lam, Xn - X, X) - P.det.origin[0], py = fma(lam, Yn - Y, Y) - P.det.origin[1],
                   pz = fma(lam, Zn - Z, Z) - P.det.origin[2];
            if constexpr (BEZ) {
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
        if (alive) {
            X = Xn; Y = Yn; Z = Zn; t += P.dt; s0 = s1;
            if constexpr (LOSS) nu0 = nu1;
        }
    }
    unsigned long long rl = sets, is = ion_steps;
    for (int o = 16; o > 0; o >>= 1) {
        rl += __shfl_down_sync(FULL, rl, o);
        is += __shfl_down_sync(FULL, is, o);
    }
    if (lane == 0) {
        atomicAdd(&P.counters[1], warp_steps);
        atomicAdd(&P.counters[2], rl >> 5);        // every lane counted the warp's items
        atomicAdd(&P.counters[3], is);
    }
}

// The table in B-fragment order.  Per cell (kind 2: (k, i, j); kind 1: ((i, j), slice pair k)) and component m one
// 4 x 8 operand per k-step s, element [b][n = 2a + c0] held by lane l = 4n + b:
//   kind 2:  C_m[c = 2s + c0][a][b]                       192 doubles per cell
//   kind 1:  c0 = 0: slice k,  c0 = 1: slice k+1 - slice k     96 doubles per (cell, k)
__global__ void k_table_to_frag(const double* __restrict__ T, double* __restrict__ F, int kind, long long ncell, int nS) {
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int per = (kind == 2) ? 192 : 96;
    const long long tot = (kind == 2) ? ncell * nS * per : ncell * (nS - 1) * per;
    if (e >= tot) return;
    const long long c = e / per;
    const int r = (int)(e % per), l = r & 31, sm = r >> 5;
    const int b = l & 3, n = l >> 2, a = n >> 1, c0 = n & 1;
    if (kind == 2) {
        const int s = sm / 3, m = sm % 3;
        F[e] = T[c * 192 + m * 64 + (2 * s + c0) * 16 + a * 4 + b];
    } else {
        const long long cell = c / (nS - 1);
        const int k = (int)(c % (nS - 1)), m = sm;
        const double* lo = T + (cell * nS + k) * 48 + m * 16 + a * 4 + b;
        F[e] = c0 ? lo[48] - lo[0] : lo[0];
    }
}

int tg_build_frag(taiga_ctx* ctx) {
    const FieldDev& f = ctx->field;
    if (ctx->frag_valid) return TAIGA_OK;
    const long long ncell = (long long)f.cR * f.cZ;
    const size_t n = (f.kind == 2) ? (size_t)ncell * f.nS * 192 : (size_t)ncell * (f.nS - 1) * 96;
    int rc = tg_reserve(ctx, &ctx->frag, &ctx->cap_frag, n);
    if (rc) return rc;
    k_table_to_frag<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(ctx->table, ctx->frag, f.kind, ncell, f.nS);
    TG_CUDA(ctx, cudaGetLastError());
    ctx->frag_valid = true;
    return TAIGA_OK;
}

// Number of toroidal cells around the torus, NK = 2 pi / ds, when the planes close on themselves (NK an integer multiple
// of nS: the period nS ds divides 2 pi); 0 otherwise (then phi has a seam at +-pi and the kernel is not offered).
static int tg_phi_cells(const FieldDev& f) {
    const double nk = 6.283185307179586476925286766559 * f.inv_ds;
    const long long r = llround(nk);
    if (r < f.nS || r > (1 << 20) || fabs(nk - (double)r) > 1e-9 * nk || r % f.nS != 0) return 0;
    return (int)r;
}

// Plane spacing up to which tg_locate_tor's four-term asin series is exact to rounding: the first dropped term of
// q = asin(s) / ds is (35 / 1152) s^9 / ds <= 0.0304 ds^8 = 2.0e-13 of a cell at ds = 0.04 (|s| <= ds once K has settled);
// 2.6e-10 at ds = 2 pi / 64 and 6.5e-8 at 2 pi / 32 would break the 1e-9 m parity.  Coarser plane sets (full-torus tables
// with a few dozen planes) go to the per-lane kernel, which takes the angle from atan2 (tg_locate_cell<2>).
#define TG_MMA_MAX_DS 0.04

// Is the cooperative kernel offered for this field?  (cell ids are 32-bit; 2 slices / planes at least)
bool tg_mma_supported(const taiga_ctx* ctx) {
    const FieldDev& f = ctx->field;
    if (f.kind != 1 && f.kind != 2) return false;
    const long long ncell = (long long)f.cR * f.cZ * f.nS;
    if (f.kind == 2 && (tg_phi_cells(f) == 0 || !(f.inv_ds * TG_MMA_MAX_DS >= 1.0))) return false;
    return ncell < (1ll << 31) && f.nS >= 2;
}

// (cos, sin) of the lower plane of every toroidal cell, built on the device
__global__ void k_phi_tab(double* __restrict__ tab, int nk, double s0, double ds) {
    const int K = blockIdx.x * blockDim.x + threadIdx.x;
    if (K >= nk) return;
    double sn, cs;
    sincos(s0 + (double)K * ds, &sn, &cs);
    tab[2 * K] = cs; tab[2 * K + 1] = sn;
}

static int tg_build_phi_tab(taiga_ctx* ctx, int nk) {
    if (ctx->phi_tab_n == nk && ctx->phi_tab_s0 == ctx->field.s0 && ctx->phi_tab) return TAIGA_OK;
    int rc = tg_reserve(ctx, &ctx->phi_tab, &ctx->cap_phi_tab, (size_t)2 * nk);
    if (rc) return rc;
    k_phi_tab<<<(nk + 127) / 128, 128, 0, ctx->stream>>>(ctx->phi_tab, nk, ctx->field.s0, 1.0 / ctx->field.inv_ds);
    TG_CUDA(ctx, cudaGetLastError());
    ctx->phi_tab_n = nk; ctx->phi_tab_s0 = ctx->field.s0;
    return TAIGA_OK;
}

// Launch geometry: THREADS per CTA (the pool the CTA re-sorts; 32 = every warp on its own, no CTA barrier) and the
// register cap.  The kernel is latency-bound: throughput follows the resident warps, and 4 CTAs of 128 threads at 128
// registers (40 B of spills) beat 3 at 148 registers by 6 % on BASELINE config 5 (profiles/r2_experiments.md), so the
// production RKN kernel is capped at 128; the grid is one persistent CTA per resident slot.
template <int KIND, int SOLVER, bool HAS_E, bool LOSS, bool BEZ, int THREADS = 128, int MAXREG = 168>
static int tg_launch_mma_t(taiga_ctx* ctx, const TraceParams& P, int per_sm, uint64_t n, cudaStream_t st) {
    auto kern = k_trace_mma<KIND, THREADS, MAXREG, SOLVER, HAS_E, LOSS, BEZ>;
    int resident = 0;
    TG_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, kern, THREADS, 0));
    if (resident < 1) resident = 1;
    if (per_sm > 0 && per_sm < resident) resident = per_sm;
    unsigned grid = (unsigned)ctx->sm_count * (unsigned)resident;
    unsigned need = (unsigned)((n + THREADS - 1) / THREADS);
    if (grid > need) grid = need;
    kern<<<grid, THREADS, 0, st>>>(P);
    return TAIGA_OK;
}

// solver: 0 RKN (P.variant 0 / 1), 2 RK4, 3 Boris (P.variant 3 / 4).  bez: RKN only; loss: any solver (as trace.cu).
int tg_trace_mma(taiga_ctx* ctx, TraceParams& P, int solver, bool hasE, bool loss, bool bez, uint64_t n) {
    int rc = tg_build_frag(ctx);
    if (rc) return rc;
    const FieldDev& f = ctx->field;
    P.frag = ctx->frag;
    P.phi_tab = nullptr; P.phi_n = 0;
    if (f.kind == 2) {
        P.phi_n = tg_phi_cells(f);
        rc = tg_build_phi_tab(ctx, P.phi_n);
        if (rc) return rc;
        P.phi_tab = (const double2*)ctx->phi_tab;
    }
    long long ncell = (f.kind == 2) ? (long long)f.cR * f.cZ * f.nS : (long long)f.cR * f.cZ * (f.nS - 1);
    P.key_shift = 0;
    while ((ncell >> P.key_shift) >= TG_KEY_DEAD - 1) ++P.key_shift;
    if (P.regroup_every < 1) P.regroup_every = 8;
    P.refill_cta = ctx->opt_refill_cta > 0 ? ctx->opt_refill_cta : 1024;      // default: whole-CTA tiles (clamped to THREADS in the kernel)
    const int per_sm = ctx->opt_ctas_per_sm;
    cudaStream_t st = ctx->stream;
#define TG_MMA(K, S, E, L, B, ...) rc = tg_launch_mma_t<K, S, E, L, B, ##__VA_ARGS__>(ctx, P, per_sm, n, st)
#define TG_MMA_KIND(K)                                                        \
    do {                                                                      \
        if (bez && loss && hasE) TG_MMA(K, 0, true, true, true);              \
        else if (bez && loss) TG_MMA(K, 0, false, true, true);                \
        else if (bez && hasE) TG_MMA(K, 0, true, false, true);                \
        else if (bez) TG_MMA(K, 0, false, false, true);                       \
        else if (loss && solver == 2) TG_MMA(K, 2, true, true, false);        \
        else if (loss && solver == 3) TG_MMA(K, 3, true, true, false);        \
        else if (loss && hasE) TG_MMA(K, 0, true, true, false);               \
        else if (loss) TG_MMA(K, 0, false, true, false);                      \
        else if (solver == 0 && hasE) TG_MMA(K, 0, true, false, false);       \
        else if (solver == 0) {                                               \
            switch (ctx->opt_mma_geom) {                                      \
                case 1: TG_MMA(K, 0, false, false, false, 128, 168); break;   \
                case 2: TG_MMA(K, 0, false, false, false, 64, 144); break;    \
                case 3: TG_MMA(K, 0, false, false, false, 32, 144); break;    \
                case 4: TG_MMA(K, 0, false, false, false, 32, 128); break;    \
                case 5: TG_MMA(K, 0, false, false, false, 64, 128); break;    \
                default: TG_MMA(K, 0, false, false, false, 128, 128); break;  \
            }                                                                 \
        } else if (solver == 2) TG_MMA(K, 2, true, false, false);             \
        else TG_MMA(K, 3, true, false, false);                                \
    } while (0)
    if (f.kind == 2) TG_MMA_KIND(2); else TG_MMA_KIND(1);
#undef TG_MMA_KIND
#undef TG_MMA
    if (rc) return rc;
    TG_CUDA(ctx, cudaGetLastError());
    return TAIGA_OK;
}
