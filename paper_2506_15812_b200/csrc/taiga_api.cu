// C ABI entry points: argument validation, context lifetime, dispatch (include/taiga.h).
#include <math.h>
#include <new>

#include "taiga_internal.h"

static bool orthonormal(const double a[3], const double b[3], const double c[3]) {
    auto dot = [](const double* p, const double* q) { return p[0] * q[0] + p[1] * q[1] + p[2] * q[2]; };
    const double tol = 1e-12;
    return fabs(dot(a, a) - 1) < tol && fabs(dot(b, b) - 1) < tol && fabs(dot(c, c) - 1) < tol &&
           fabs(dot(a, b)) < tol && fabs(dot(a, c)) < tol && fabs(dot(b, c)) < tol;
}

static bool cdf_ok(const double* F, int K) {
    if (!F || K < 1 || F[0] != 0.0 || F[K] != 1.0) return false;
    for (int i = 0; i < K; ++i) if (!(F[i] <= F[i + 1])) return false;
    return true;
}

extern "C" int taiga_create(taiga_ctx** out, int device, void* cuda_stream) {
    if (!out) return TAIGA_E_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return TAIGA_E_CUDA;
    taiga_ctx* ctx = new (std::nothrow) taiga_ctx();
    if (!ctx) return TAIGA_E_NOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(device) != cudaSuccess) { delete ctx; return TAIGA_E_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete ctx; return TAIGA_E_CUDA; }
    if (prop.major < 10) { delete ctx; return TAIGA_E_CUDA; }     // sm_100a code only
    ctx->sm_count = prop.multiProcessorCount;
    if (cudaMalloc((void**)&ctx->counters, 16 * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMallocHost((void**)&ctx->counters_host, 16 * sizeof(unsigned long long)) != cudaSuccess) {
        if (ctx->counters) cudaFree(ctx->counters);
        delete ctx; return TAIGA_E_NOMEM;
    }
    if (cudaEventCreateWithFlags(&ctx->stage_done, cudaEventDisableTiming) != cudaSuccess) {
        cudaFree(ctx->counters); cudaFreeHost(ctx->counters_host); delete ctx; return TAIGA_E_CUDA;
    }
    ctx->opt_sort = 1; ctx->opt_sort_sub = 16;
    ctx->opt_min_active = 32;
    ctx->opt_ctas_per_sm = 0; ctx->opt_variant = 0; ctx->opt_stats = 0; ctx->opt_precision = 64; ctx->opt_plane_interp = 0; ctx->opt_regroup = 8;
    ctx->opt_mma = -1; ctx->opt_refill_cta = 0;
    strcpy(ctx->err, "ok");
    *out = ctx;
    return TAIGA_OK;
}

extern "C" int taiga_destroy(taiga_ctx* ctx) {
    if (!ctx) return TAIGA_E_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    void* bufs[] = {ctx->table, ctx->scratch, ctx->band[0], ctx->band[1], ctx->cdf_depth, ctx->cdf_normal, ctx->edges, ctx->order,
                    ctx->bins, ctx->counters, ctx->table32, ctx->psi_table, ctx->loss_rate, ctx->dtable, ctx->frag, ctx->phi_tab, ctx->etable};
    for (void* b : bufs) if (b) cudaFree(b);
    if (ctx->counters_host) cudaFreeHost(ctx->counters_host);
    if (ctx->stage) cudaFreeHost(ctx->stage);
    if (ctx->stage_done) cudaEventDestroy(ctx->stage_done);
    delete ctx;
    return TAIGA_OK;
}

extern "C" const char* taiga_last_error(const taiga_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" int taiga_load_field(taiga_ctx* ctx, const taiga_grid* g, const taiga_coeffs* c) {
    if (!ctx) return TAIGA_E_ARG;
    if (!g || !c || !c->BR || !c->BZ || !c->Bphi) { TG_SET_ERR(ctx, "load_field: null argument"); return TAIGA_E_ARG; }
    if (g->kind < 0 || g->kind > 2 || g->nR < 4 || g->nZ < 4 || !(g->Rmax > g->Rmin) || !(g->Zmax > g->Zmin) ||
        !(g->Rmin > 0.0) || (g->kind == 0 && g->nS != 1) || (g->kind == 1 && g->nS < 2) ||
        (g->kind == 2 && g->nS < 3) || (g->kind != 0 && !(g->ds > 0.0)) || (c->form != 0 && c->form != 1)) {
        TG_SET_ERR(ctx, "load_field: bad grid (kind=%d nR=%d nZ=%d nS=%d form=%d)", g->kind, g->nR, g->nZ, g->nS, c->form);
        return TAIGA_E_ARG;
    }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->field_loaded = false; ctx->table32_valid = false; ctx->frag_valid = false; ctx->dtable_valid = false; ctx->loss.psi = nullptr;   // a new grid invalidates psi
    int rc = tg_precompute(ctx, g, c);
    if (rc == TAIGA_OK) ctx->field_loaded = true;
    return rc;
}

extern "C" int taiga_field_eval(taiga_ctx* ctx, uint64_t n, const double* R, const double* Z, const double* s,
                                double* BR, double* BZ, double* Bp) {
    if (!ctx) return TAIGA_E_ARG;
    if (!ctx->field_loaded) { TG_SET_ERR(ctx, "field_eval before load_field"); return TAIGA_E_STATE; }
    if (n && (!R || !Z || !BR || !BZ || !Bp)) { TG_SET_ERR(ctx, "field_eval: null argument"); return TAIGA_E_ARG; }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return n ? tg_field_eval(ctx, n, R, Z, s, BR, BZ, Bp) : TAIGA_OK;
}

extern "C" int taiga_field_table(taiga_ctx* ctx, int comp, double* host) {
    if (!ctx) return TAIGA_E_ARG;
    if (!ctx->field_loaded) { TG_SET_ERR(ctx, "field_table before load_field"); return TAIGA_E_STATE; }
    if (comp < 0 || comp > 2 || !host) { TG_SET_ERR(ctx, "field_table: bad argument"); return TAIGA_E_ARG; }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_field_table(ctx, comp, host);
}

static int check_ions(taiga_ctx* ctx, const taiga_ions* ions, bool need_out) {
    if (!ions) { TG_SET_ERR(ctx, "null ions"); return TAIGA_E_ARG; }
    if (ions->n >= (1ull << 32)) { TG_SET_ERR(ctx, "ions->n must be < 2^32"); return TAIGA_E_ARG; }
    if (ions->n == 0) return TAIGA_OK;
    if (!ions->x || !ions->y || !ions->z || !ions->vx || !ions->vy || !ions->vz) { TG_SET_ERR(ctx, "null ion state array"); return TAIGA_E_ARG; }
    if (need_out && (!ions->hit_u || !ions->hit_w || !ions->cell || !ions->steps || !ions->flags)) {
        TG_SET_ERR(ctx, "null ion result array"); return TAIGA_E_ARG;
    }
    return TAIGA_OK;
}

static int seed_common(taiga_ctx* ctx, const taiga_beam_params* p, uint64_t seed, taiga_ions* ions, const taiga_seed_grid* g) {
    if (!ctx) return TAIGA_E_ARG;
    if (!p) { TG_SET_ERR(ctx, "seed_beam: null params"); return TAIGA_E_ARG; }
    int rc = check_ions(ctx, ions, false);
    if (rc) return rc;
    if (!(p->mass_kg > 0) || !(p->charge_C != 0) || !(p->energy_eV > 0) || !(p->depth_max > 0) || !(p->z_max > 0) ||
        p->sigma_pos_m < 0 || p->sigma_ang_rad < 0 || (p->profile != TAIGA_PROFILE_GAUSSIAN && p->profile != TAIGA_PROFILE_DISC) ||
        (p->profile == TAIGA_PROFILE_DISC && !(p->radius_m > 0))) { TG_SET_ERR(ctx, "seed_beam: bad beam parameters"); return TAIGA_E_ARG; }
    if (g && p->profile != TAIGA_PROFILE_GAUSSIAN) { TG_SET_ERR(ctx, "seed_beam_grid: the weighted grid is defined for the Gaussian profile"); return TAIGA_E_ARG; }
    if (!orthonormal(p->axis, p->eT, p->eZ)) { TG_SET_ERR(ctx, "seed_beam: (axis,eT,eZ) not orthonormal"); return TAIGA_E_ARG; }
    if (!cdf_ok(p->cdf_depth, p->n_depth) || !cdf_ok(p->cdf_normal, p->n_normal)) {
        TG_SET_ERR(ctx, "seed_beam: CDF table must have F[0]=0, F[K]=1 and be non-decreasing"); return TAIGA_E_ARG;
    }
    if (g) {
        if (g->nd < 1 || g->nT < 1 || g->nZ < 1 || !(g->z_lim > 0) || !(g->z_lim <= p->z_max)) { TG_SET_ERR(ctx, "seed_beam_grid: bad grid (0 < z_lim <= z_max)"); return TAIGA_E_ARG; }
        unsigned long long tot = (unsigned long long)g->nd * (unsigned long long)g->nT * (unsigned long long)g->nZ;
        if (p->first_index > tot || ions->n > tot - p->first_index) { TG_SET_ERR(ctx, "seed_beam_grid: first_index + n exceeds nd*nT*nZ"); return TAIGA_E_ARG; }
        if (ions->n && !ions->w0) { TG_SET_ERR(ctx, "seed_beam_grid: ions->w0 is null"); return TAIGA_E_ARG; }
    }
    if (ions->n == 0) return TAIGA_OK;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    double v0 = sqrt(2.0 * p->energy_eV * fabs(p->charge_C) / p->mass_kg);   // IEEE sqrt, host
    return tg_seed(ctx, p, seed, ions, v0, g);
}

extern "C" int taiga_seed_beam(taiga_ctx* ctx, const taiga_beam_params* p, uint64_t seed, taiga_ions* ions) {
    return seed_common(ctx, p, seed, ions, nullptr);
}

extern "C" int taiga_seed_beam_grid(taiga_ctx* ctx, const taiga_beam_params* p, const taiga_seed_grid* g, taiga_ions* ions) {
    if (!ctx) return TAIGA_E_ARG;
    if (!g) { TG_SET_ERR(ctx, "seed_beam_grid: null grid"); return TAIGA_E_ARG; }
    return seed_common(ctx, p, 0, ions, g);
}

static int check_det(taiga_ctx* ctx, const taiga_detector* d, bool need_edges) {
    if (!d) { TG_SET_ERR(ctx, "null detector"); return TAIGA_E_ARG; }
    if (!orthonormal(d->normal, d->eu, d->ew)) { TG_SET_ERR(ctx, "detector: (normal,eu,ew) not orthonormal"); return TAIGA_E_ARG; }
    if (!need_edges) return TAIGA_OK;
    if (d->nu < 1 || d->nw < 1 || d->nu > 4096 || d->nw > 4096 || !d->u_lo || !d->u_hi || !d->w_lo || !d->w_hi) {
        TG_SET_ERR(ctx, "detector: bad segment arrays"); return TAIGA_E_ARG;
    }
    for (int ax = 0; ax < 2; ++ax) {
        const double *lo = ax ? d->w_lo : d->u_lo, *hi = ax ? d->w_hi : d->u_hi;
        int n = ax ? d->nw : d->nu;
        for (int k = 0; k < n; ++k)
            if (!(lo[k] < hi[k]) || (k + 1 < n && !(hi[k] <= lo[k + 1]))) {
                TG_SET_ERR(ctx, "detector: segments must be ordered and non-overlapping"); return TAIGA_E_ARG;
            }
    }
    return TAIGA_OK;
}

extern "C" int taiga_trace(taiga_ctx* ctx, taiga_ions* ions, double qm, double dt, uint32_t max_steps,
                           const taiga_detector* det, int variant) {
    if (!ctx) return TAIGA_E_ARG;
    if (!ctx->field_loaded) { TG_SET_ERR(ctx, "trace before load_field"); return TAIGA_E_STATE; }
    int rc = check_ions(ctx, ions, true);
    if (rc) return rc;
    rc = check_det(ctx, det, false);
    if (rc) return rc;
    if (!(dt > 0) || !isfinite(qm) || qm == 0 || variant < 0 || variant > 4) { TG_SET_ERR(ctx, "trace: bad dt / q_over_m / solver"); return TAIGA_E_ARG; }
    if (ions->n == 0) return TAIGA_OK;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    DetDev dd;
    for (int c = 0; c < 3; ++c) { dd.origin[c] = det->origin[c]; dd.normal[c] = det->normal[c]; dd.eu[c] = det->eu[c]; dd.ew[c] = det->ew[c]; }
    return tg_trace(ctx, ions, qm, dt, max_steps, dd, variant);
}

extern "C" int taiga_load_loss(taiga_ctx* ctx, const double* psi_nodal, int on_device, const taiga_loss_profile* prof) {
    if (!ctx) return TAIGA_E_ARG;
    if (!psi_nodal) { ctx->loss.psi = nullptr; return TAIGA_OK; }
    if (!ctx->field_loaded) { TG_SET_ERR(ctx, "load_loss before load_field (psi lives on the field's (R,Z) grid)"); return TAIGA_E_STATE; }
    if (!prof || prof->n < 2 || prof->n > (1 << 20) || !prof->ne_m3 || !prof->Te_eV || !(prof->dpsi > 0) || !isfinite(prof->psi0) ||
        !(prof->E12_eV > 0)) { TG_SET_ERR(ctx, "load_loss: bad profile"); return TAIGA_E_ARG; }
    for (int k = 0; k < prof->n; ++k)
        if (!(prof->ne_m3[k] >= 0) || !isfinite(prof->ne_m3[k]) || !isfinite(prof->Te_eV[k])) { TG_SET_ERR(ctx, "load_loss: negative / non-finite profile value"); return TAIGA_E_ARG; }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_load_loss(ctx, psi_nodal, on_device, prof);
}

extern "C" int taiga_detector_histogram_weighted(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                                                 unsigned long long* wcounts, unsigned long long* wsummary) {
    if (!ctx) return TAIGA_E_ARG;
    int rc = check_ions(ctx, ions, true);
    if (rc) return rc;
    rc = check_det(ctx, det, true);
    if (rc) return rc;
    if (n_hist < 1 || n_hist > 65536 || !wcounts || !wsummary) { TG_SET_ERR(ctx, "histogram_weighted: bad n_hist / null output"); return TAIGA_E_ARG; }
    if (ions->n == 0) return TAIGA_OK;
    if (!ions->weight && !ions->w0) { TG_SET_ERR(ctx, "histogram_weighted: ions->weight and ions->w0 are null"); return TAIGA_E_ARG; }
    if (ions->weight) {
        bool known = false;
        for (int q = 0; q < ctx->n_wranges && !known; ++q)
            known = ctx->wranges[q].p <= ions->weight && ions->weight + ions->n <= ctx->wranges[q].p + ctx->wranges[q].n;
        if (!known) {
            TG_SET_ERR(ctx, "histogram_weighted: ions->weight is set but no recent taiga_trace of this context wrote these weights "
                            "(no loss model loaded, or other ions traced); pass your own weights as w0 with weight = null");
            return TAIGA_E_STATE;
        }
    }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_histogram_weighted(ctx, ions, det, n_hist, wcounts, wsummary);
}

extern "C" int taiga_set_efield(taiga_ctx* ctx, const double E[3]) {
    if (!ctx || !E) return TAIGA_E_ARG;
    for (int c = 0; c < 3; ++c) if (!isfinite(E[c])) { TG_SET_ERR(ctx, "set_efield: non-finite component"); return TAIGA_E_ARG; }
    for (int c = 0; c < 3; ++c) ctx->E[c] = E[c];
    return TAIGA_OK;
}

extern "C" int taiga_load_efield(taiga_ctx* ctx, const taiga_coeffs* c) {
    if (!ctx) return TAIGA_E_ARG;
    if (!ctx->field_loaded) { TG_SET_ERR(ctx, "load_efield: no magnetic field loaded (its grid carries E)"); return TAIGA_E_STATE; }
    if (c && (c->form != 0 || !c->BR || !c->BZ || !c->Bphi)) {
        TG_SET_ERR(ctx, "load_efield: nodal values (form 0) of E_R, E_Z, E_phi on the (R, Z) grid");
        return TAIGA_E_ARG;
    }
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_load_efield(ctx, c);
}

extern "C" int taiga_detector_histogram(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                                        unsigned long long* counts, unsigned long long* summary) {
    if (!ctx) return TAIGA_E_ARG;
    int rc = check_ions(ctx, ions, true);
    if (rc) return rc;
    rc = check_det(ctx, det, true);
    if (rc) return rc;
    if (n_hist < 1 || n_hist > 65536 || !counts || !summary) { TG_SET_ERR(ctx, "histogram: bad n_hist / null output"); return TAIGA_E_ARG; }
    if (ions->n == 0) return TAIGA_OK;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_histogram(ctx, ions, det, n_hist, counts, summary);
}

// The binning of taiga_detector_histogram for callers that must not allocate (include/taiga.h): same checks, same kernel,
// the edge table in a fixed device array of the library instead of a buffer of the context.
extern "C" int taiga_detector_histogram_static(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                                               unsigned long long* counts, unsigned long long* summary) {
    if (!ctx) return TAIGA_E_ARG;
    int rc = check_ions(ctx, ions, true);
    if (rc) return rc;
    rc = check_det(ctx, det, true);
    if (rc) return rc;
    if (n_hist < 1 || n_hist > 65536 || !counts || !summary) { TG_SET_ERR(ctx, "histogram_static: bad n_hist / null output"); return TAIGA_E_ARG; }
    if (det->nu + det->nw > TAIGA_STATIC_MAX_SEGMENTS) {
        TG_SET_ERR(ctx, "histogram_static: nu + nw = %d segments exceed TAIGA_STATIC_MAX_SEGMENTS = %d (the fixed edge table); "
                        "use taiga_detector_histogram, which allocates", det->nu + det->nw, TAIGA_STATIC_MAX_SEGMENTS);
        return TAIGA_E_ARG;
    }
    if (ions->n == 0) return TAIGA_OK;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_histogram_static(ctx, ions, det, n_hist, counts, summary);
}

extern "C" int taiga_set_option(taiga_ctx* ctx, const char* key, long long v) {
    if (!ctx || !key) return TAIGA_E_ARG;
    struct { const char* k; int* p; long long lo, hi; } tab[] = {
        {"sort", &ctx->opt_sort, 0, 1}, {"sort_sub", &ctx->opt_sort_sub, 1, 64},
        {"precision", &ctx->opt_precision, 32, 64}, {"plane_interp", &ctx->opt_plane_interp, 0, 1},
        {"regroup", &ctx->opt_regroup, 0, 1 << 20}, {"min_active", &ctx->opt_min_active, 0, 32},
        {"ctas_per_sm", &ctx->opt_ctas_per_sm, 0, 32}, {"variant", &ctx->opt_variant, 0, 7}, {"stats", &ctx->opt_stats, 0, 1},
        {"mma", &ctx->opt_mma, -1, 1}, {"refill_cta", &ctx->opt_refill_cta, 0, 1024},
        {"mma_geom", &ctx->opt_mma_geom, 0, 5}};
    for (auto& t : tab) if (!strcmp(key, t.k)) {
        if (v < t.lo || v > t.hi || (t.p == &ctx->opt_precision && v != 32 && v != 64)) {
            TG_SET_ERR(ctx, "set_option: %s = %lld out of range [%lld, %lld]", key, v, t.lo, t.hi);
            return TAIGA_E_ARG;
        }
        *t.p = (int)v;
        return TAIGA_OK;
    }
    TG_SET_ERR(ctx, "set_option: unknown key '%s'", key);
    return TAIGA_E_ARG;
}

extern "C" int taiga_get_stats(taiga_ctx* ctx, unsigned long long out[8]) {
    if (!ctx || !out) return TAIGA_E_ARG;
    if (ctx->stats_pending) {                   // the one place the trace path waits for the device
        TG_CUDA(ctx, cudaSetDevice(ctx->device));
        int rc = tg_collect_stats(ctx);
        if (rc) return rc;
    }
    for (int i = 0; i < 8; ++i) out[i] = ctx->stats[i];
    return TAIGA_OK;
}

extern "C" int taiga_measure_l1_gather_peak(taiga_ctx* ctx, double ms, int spread, double* bytes_per_s) {
    if (!ctx || !bytes_per_s || !(ms > 0)) return TAIGA_E_ARG;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_l1_gather_peak(ctx, ms, spread, bytes_per_s);
}

extern "C" int taiga_measure_fp64_peak(taiga_ctx* ctx, double ms, double* rate) {
    if (!ctx || !rate || !(ms > 0)) return TAIGA_E_ARG;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_fp64_peak(ctx, ms, rate);
}

extern "C" int taiga_measure_dmma_peak(taiga_ctx* ctx, double ms, double* rate) {
    if (!ctx || !rate || !(ms > 0)) return TAIGA_E_ARG;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_dmma_peak(ctx, ms, rate);
}

extern "C" int taiga_measure_mixed_fp64_peak(taiga_ctx* ctx, double ms, double* rate) {
    if (!ctx || !rate || !(ms > 0)) return TAIGA_E_ARG;
    TG_CUDA(ctx, cudaSetDevice(ctx->device));
    return tg_mixed_peak(ctx, ms, rate);
}

extern "C" int taiga_loss_statistics(const unsigned long long ws[4], double out[3]) {
    if (!ws || !out) return TAIGA_E_ARG;
    const double n = ws[3] ? (double)ws[3] : 1.0;
    const double mu = ((double)ws[0] + (double)ws[1]) / 4294967296.0 / n;
    double var = (double)ws[2] / 4294967296.0 / n - mu * mu;
    if (!(var > 0.0)) var = 0.0;
    out[0] = 1.0 - mu; out[1] = sqrt(var); out[2] = (double)ws[3];
    return TAIGA_OK;
}
