// Internal declarations of libtaiga (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/taiga.h"

// Grid geometry as the kernels want it (derived once in taiga_load_field).
struct FieldDev {
    int kind, nR, nZ, nS;            // nodes
    int cR, cZ;                      // cells
    double Rmin, Rmax, Zmin, Zmax;
    double inv_hR, inv_hZ;           // 1/h
    double offR, offZ;               // Rmin/hR, Zmin/hZ   (p_total = R*inv_hR - offR)
    double s0, inv_ds;
    // kind 0: [iR][iZ][comp][16]            (384 B per cell, one 128-B line per component)
    // kind 1: [iR][iZ][slice][comp][16]     (the two slices of a cell are adjacent)
    // kind 2: [iphi][iR][iZ][comp][64]
    const double* table;
    const double* dtable;            // kind 1: slice differences [iR][iZ][k < nS-1][comp][16] = table[k+1] - table[k]
    const float* table32;            // kind 2, "precision" = 32: the same table rounded to fp32 (else null)
    const double* etable;            // gridded E (taiga_load_efield): [iR][iZ][comp E_R, E_Z, E_phi][16], else null
};

// secondary-ionisation loss model (taiga_load_loss); psi == nullptr: none
struct LossDev {
    const double* psi;               // [iR][iZ][48]: 16 coefficients used (kind-0 cell layout)
    const double* rate;              // nu_k [1/s]
    int n;
    double psi0, inv_dpsi;
};

struct DetDev {
    double origin[3], normal[3], eu[3], ew[3];
};

struct taiga_ctx {
    int device;
    cudaStream_t stream;
    char err[512];
    int sm_count;

    // field
    bool field_loaded;
    FieldDev field;
    double* table;            size_t table_bytes;
    double* scratch;          size_t scratch_bytes;     // precompute work arrays
    double* dtable;           size_t cap_dtable;   bool dtable_valid;    // kind 1: slice differences (built on first use)
    double* phi_tab;          size_t cap_phi_tab;  int phi_tab_n; double phi_tab_s0;   // kind 2: plane directions (trace_mma.cu)
    double* frag;             size_t cap_frag;     bool frag_valid;      // kinds 1, 2: table in DMMA B-fragment order (trace_mma.cu)
    float* table32;           size_t cap_table32;  bool table32_valid;   // fp32 copy of a kind-2 table
    double* band[2];          size_t band_cap[2]; int band_n[2];   // y -> y'' band operators (Z, R)

    double E[3];                                         // uniform electric field (taiga_set_efield), V/m
    double* etable;           size_t cap_etable;         // gridded electric field (taiga_load_efield); field.etable = null: none

    // loss model
    LossDev loss;
    double* psi_table;        size_t cap_psi;
    double* loss_rate;        size_t cap_rate;

    // seeding tables
    double *cdf_depth, *cdf_normal;  int cap_depth, cap_normal;

    // pinned staging buffer for small host tables (CDFs, detector edges): reused once `stage_done` has passed
    void* stage;              size_t stage_cap;    cudaEvent_t stage_done;

    // detector edges (histogram)
    double* edges;            int cap_edges;

    // trace scratch
    uint32_t* order;          size_t cap_order;          // permutation (sorted by birth cell)
    uint32_t* bins;           size_t cap_bins;           // counting-sort bins
    unsigned long long* counters;                        // device counters (16)
    unsigned long long* counters_host;                   // pinned mirror
    unsigned long long stats[8];
    bool stats_pending;  int stats_launches;             // the last trace's counters are on their way to counters_host

    // options
    int opt_sort, opt_min_active, opt_ctas_per_sm, opt_variant, opt_stats;
    int opt_sort_sub, opt_precision, opt_plane_interp, opt_regroup;
    int opt_mma, opt_refill_cta, opt_mma_geom;
    // ions->weight ranges written by recent taiga_trace calls with a loss model (newest last); a trace without one drops
    // the ranges it overlaps (their weights are stale).  taiga_detector_histogram_weighted accepts a weight array inside one.
    struct { const double* p; uint64_t n; } wranges[16];
    int n_wranges;
};

#define TG_SET_ERR(ctx, ...) snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__)

#define TG_CUDA(ctx, call)                                                            \
    do {                                                                              \
        cudaError_t e_ = (call);                                                      \
        if (e_ != cudaSuccess) {                                                      \
            TG_SET_ERR(ctx, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? TAIGA_E_NOMEM : TAIGA_E_CUDA;  \
        }                                                                             \
    } while (0)

// grow-only device buffer
template <typename T>
static inline int tg_reserve(taiga_ctx* ctx, T** p, size_t* cap, size_t need) {
    if (*cap >= need && *p) return TAIGA_OK;
    if (*p) cudaFree(*p);
    *p = nullptr; *cap = 0;
    cudaError_t e = cudaMalloc((void**)p, need * sizeof(T));
    if (e != cudaSuccess) { TG_SET_ERR(ctx, "cudaMalloc(%zu B): %s", need * sizeof(T), cudaGetErrorString(e)); return TAIGA_E_NOMEM; }
    *cap = need;
    return TAIGA_OK;
}

// Pinned staging for small host tables: waits until the previous staged copy has left the buffer, grows it if needed.
static inline int tg_stage(taiga_ctx* ctx, size_t bytes) {
    if (ctx->stage_done) cudaEventSynchronize(ctx->stage_done);
    if (ctx->stage_cap < bytes) {
        if (ctx->stage) cudaFreeHost(ctx->stage);
        ctx->stage = nullptr; ctx->stage_cap = 0;
        size_t cap = bytes < 65536 ? 65536 : bytes;
        if (cudaMallocHost(&ctx->stage, cap) != cudaSuccess) { TG_SET_ERR(ctx, "cudaMallocHost(%zu B) failed", cap); return TAIGA_E_NOMEM; }
        ctx->stage_cap = cap;
    }
    return TAIGA_OK;
}

// implemented in the per-kernel translation units
int tg_precompute(taiga_ctx* ctx, const taiga_grid* g, const taiga_coeffs* c);
int tg_seed(taiga_ctx* ctx, const taiga_beam_params* p, uint64_t seed, taiga_ions* ions, double v0,
            const taiga_seed_grid* grid /* null: stochastic */);
int tg_build_order(taiga_ctx* ctx, const taiga_ions* ions);      // queue_sort.cu: fills ctx->order
int tg_trace(taiga_ctx* ctx, taiga_ions* ions, double qm, double dt, uint32_t max_steps,
             const DetDev& det, int variant);
int tg_collect_stats(taiga_ctx* ctx);                            // trace.cu: waits for the stream, fills ctx->stats
struct TraceParams;
int tg_trace_mma(taiga_ctx* ctx, TraceParams& P, int solver, bool hasE, bool loss, bool bez, uint64_t n);   // trace_mma.cu
bool tg_mma_supported(const taiga_ctx* ctx);
int tg_build_dtable(taiga_ctx* ctx);                             // field_precompute.cu
int tg_histogram(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                 unsigned long long* counts, unsigned long long* summary);
int tg_histogram_static(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                        unsigned long long* counts, unsigned long long* summary);       // histogram.cu: no allocation
int tg_field_eval(taiga_ctx* ctx, uint64_t n, const double* R, const double* Z, const double* s,
                  double* BR, double* BZ, double* Bp);
int tg_field_table(taiga_ctx* ctx, int comp, double* host);
int tg_load_loss(taiga_ctx* ctx, const double* psi_nodal, int on_device, const taiga_loss_profile* prof);
int tg_load_efield(taiga_ctx* ctx, const taiga_coeffs* c);        // field_precompute.cu
int tg_histogram_weighted(taiga_ctx* ctx, const taiga_ions* ions, const taiga_detector* det, int n_hist,
                          unsigned long long* wcounts, unsigned long long* wsummary);
int tg_fp64_peak(taiga_ctx* ctx, double ms, double* rate);
int tg_dmma_peak(taiga_ctx* ctx, double ms, double* rate);
int tg_mixed_peak(taiga_ctx* ctx, double ms, double* rate);
int tg_l1_gather_peak(taiga_ctx* ctx, double ms, int spread, double* bytes_per_s);
