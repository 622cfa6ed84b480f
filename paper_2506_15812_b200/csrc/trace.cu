// a3 + a4: host side of taiga_trace and the k_trace instantiations of the production path (RKN, E = 0), with the loss
// integral and the Bezier interpolation; the variants with an electric field / the other solvers live in
// trace_variants.cu, the kernel template in trace_kernel.cuh.
#include "trace_kernel.cuh"

__global__ void k_table_to_f32(const double* __restrict__ src, float* __restrict__ dst, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) dst[i] = (float)src[i];
}

static const TgVariant tg_variants_a[] = {
    // 32-thread CTAs (warps are independent: any block size), register cap 224: 8 warps per SM as before (the register
    // file is allocated in steps that put 210 registers at 256 per lane); 10 warps at 192 registers were slower
    // (profiles/r2_experiments.md)
    TG_VT(0, 1, 224, 2, 32),
    // production path: RKN, E = 0
    TG_V(0, 1, 255, 2, 0, 0, 0, 0, 0), TG_V(0, 1, 255, 1, 0, 0, 0, 0, 0), TG_V(0, 1, 255, 0, 0, 0, 0, 0, 0), TG_V(0, 1, 168, 0, 0, 0, 0, 0, 0),
    TG_V(0, 0, 128, 0, 0, 0, 0, 0, 0), TG_V(0, 0, 255, 0, 0, 0, 0, 0, 0),
    TG_V(1, 1, 255, 4, 0, 0, 0, 0, 0), TG_V(1, 1, 255, 3, 0, 0, 0, 0, 0), TG_V(1, 1, 255, 2, 0, 0, 0, 0, 0), TG_V(1, 0, 255, 0, 0, 0, 0, 0, 0), TG_V(1, 0, 128, 0, 0, 0, 0, 0, 0),
    TG_V(2, 0, 255, 0, 0, 0, 0, 0, 1), TG_V(2, 0, 255, 0, 0, 0, 0, 0, 0), TG_V(2, 0, 128, 0, 0, 0, 0, 0, 0),
    // quadratic Bezier plane interpolation
    TG_V(0, 1, 255, 2, 0, 0, 0, 1, 0), TG_V(0, 1, 255, 0, 0, 0, 0, 1, 0), TG_V(1, 1, 255, 4, 0, 0, 0, 1, 0), TG_V(1, 0, 255, 0, 0, 0, 0, 1, 0),
    TG_V(2, 0, 255, 0, 0, 0, 0, 1, 0),
    // Eq. 2 loss integral
    TG_V(0, 1, 255, 2, 0, 0, 1, 0, 0), TG_V(0, 1, 255, 0, 0, 0, 1, 0, 0), TG_V(1, 1, 255, 4, 0, 0, 1, 0, 0), TG_V(1, 0, 255, 0, 0, 0, 1, 0, 0),
    TG_V(2, 0, 255, 0, 0, 0, 1, 0, 0),
    // the loss integral with the Bezier interpolation (reading L2')
    TG_V(0, 1, 255, 2, 0, 0, 1, 1, 0), TG_V(0, 1, 255, 0, 0, 0, 1, 1, 0), TG_V(1, 1, 255, 4, 0, 0, 1, 1, 0), TG_V(1, 0, 255, 0, 0, 0, 1, 1, 0),
    TG_V(2, 0, 255, 0, 0, 0, 1, 1, 0),
};

const TgVariant* tg_trace_variants_b(int* n);       // trace_variants.cu

int tg_collect_stats(taiga_ctx* ctx) {
    if (!ctx->stats_pending) return TAIGA_OK;
    TG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->stats[0] = ctx->counters_host[3];
    ctx->stats[1] = ctx->counters_host[1] * 32ull;
    ctx->stats[2] = 1;
    ctx->stats[3] = (unsigned long long)ctx->stats_launches;
    ctx->stats[4] = ctx->counters_host[2];
    ctx->stats[5] = 0;
    ctx->stats_pending = false;
    return TAIGA_OK;
}

int tg_trace(taiga_ctx* ctx, taiga_ions* ions, double qm, double dt, uint32_t max_steps, const DetDev& det, int variant) {
    cudaStream_t st = ctx->stream;
    const int kind = ctx->field.kind;
    const bool loss = ctx->loss.psi != nullptr && ions->weight != nullptr;
    const bool bez = ctx->opt_plane_interp == 1;
    const bool f32 = ctx->opt_precision == 32;
    bool hasE = false;
    for (int c = 0; c < 3; ++c) hasE |= ctx->E[c] != 0.0;
    hasE |= ctx->field.etable != nullptr;          // gridded E (taiga_load_efield)
    // ---- what is offered (checked before anything is enqueued)
    if (f32 && (kind != 2 || variant > 1)) {
        TG_SET_ERR(ctx, "precision=32 is offered for kind-2 (R,Z,phi) fields with the RKN solver only");
        return TAIGA_E_ARG;
    }
    if (bez && (variant > 1 || f32)) {
        TG_SET_ERR(ctx, "plane_interp=1 (Bezier) is offered with the RKN solvers (Boris velocities live at half steps), fp64");
        return TAIGA_E_ARG;
    }
    if (loss && f32) {
        TG_SET_ERR(ctx, "the loss model is offered in fp64");
        return TAIGA_E_ARG;
    }
    if (hasE && f32) {
        TG_SET_ERR(ctx, "precision=32 is offered without an electric field (the uniform and the gridded E are fp64 only)");
        return TAIGA_E_ARG;
    }
    TraceParams P;
    P.f = ctx->field; P.det = det;
    P.loss = ctx->loss; P.hdt = 0.5 * dt; P.weight = ions->weight; P.w0 = ions->w0;
    P.frag = nullptr; P.key_shift = 0; P.refill_cta = 0; P.phi_tab = nullptr; P.phi_n = 0;
    if (f32) {                                 // fp32 field evaluation (BASELINE config 5 "fp32 variant")
        if (!ctx->table32_valid) {
            size_t n = (size_t)ctx->field.nS * ctx->field.cR * ctx->field.cZ * 192;
            int rc = tg_reserve(ctx, &ctx->table32, &ctx->cap_table32, n);
            if (rc) return rc;
            k_table_to_f32<<<ctx->sm_count * 8, 256, 0, st>>>(ctx->table, ctx->table32, n);
            TG_CUDA(ctx, cudaGetLastError());
            ctx->table32_valid = true;
        }
        P.f.table32 = ctx->table32;
    }
    P.nrD = det.normal[0] * det.origin[0] + det.normal[1] * det.origin[1] + det.normal[2] * det.origin[2];
    P.qm = qm; P.dt = dt;
    P.a1 = dt / (2.0 * qm); P.a2 = dt * dt / 8.0; P.b1 = qm * dt / 2.0;
    P.c6 = dt * dt / 6.0; P.d6 = qm * dt / 6.0; P.dtq = dt / qm;
    for (int c = 0; c < 3; ++c) { P.qE[c] = qm * ctx->E[c]; P.eh[c] = qm * qm * ctx->E[c] * dt * 0.5; }
    P.pa1R = P.a1 * ctx->field.inv_hR; P.pa1Z = P.a1 * ctx->field.inv_hZ;
    P.max_steps = max_steps; P.n = (uint32_t)ions->n; P.variant = variant;
    P.regroup_every = ctx->opt_regroup > 0 ? ctx->opt_regroup : 0;
    P.refill_min = ctx->opt_min_active > 0 ? (ctx->opt_min_active > 32 ? 32 : ctx->opt_min_active) : 1;
    P.x = ions->x; P.y = ions->y; P.z = ions->z; P.vx = ions->vx; P.vy = ions->vy; P.vz = ions->vz; P.t0 = ions->t0;
    P.hit_u = ions->hit_u; P.hit_w = ions->hit_w; P.cell = ions->cell; P.steps = ions->steps; P.flags = ions->flags;
    P.counters = ctx->counters;
    P.order = nullptr;
    int launches = 0;
    if (ctx->opt_sort && ions->n > 64) {
        int rc = tg_build_order(ctx, ions);
        if (rc) return rc;
        P.order = ctx->order;
        launches += 5;
    }
    TG_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, 8 * sizeof(unsigned long long), st));
    const int S = variant <= 1 ? 0 : (variant == 2 ? 2 : 3);
    const int use_mma = ctx->opt_mma < 0 ? (kind == 2) : ctx->opt_mma;      // default: kind 2 (kind 1: 3 DMMAs per set do not pay)
    if (kind >= 1 && use_mma && !f32 && tg_mma_supported(ctx)) {
        // kinds 1, 2: warp-cooperative evaluation on the FP64 tensor pipe (trace_mma.cu), every solver and option
        int rc = tg_trace_mma(ctx, P, S, hasE || S != 0, loss, bez, ions->n);
        if (rc) return rc;
    } else {
        // option "variant", kind 0 with the classical RKN: 0 rolling predictive refill (default), 4 predictive refill after
        // each Horner, 5 refill on demand, 3 on demand at 168 registers, 1 no cache, 2 no cache at 128 registers
        const int kv = ctx->opt_variant;
        const bool special = bez || loss || hasE || S != 0;       // these run at 2 CTAs/SM on the full-register kernels
        TgVariant k = {kind, 0, 255, 0, S, (hasE || S != 0) ? 1 : 0, loss ? 1 : 0, bez ? 1 : 0, 0, nullptr};
        if (kind == 0) {
            if (special) { k.cached = 1; k.pred = (variant == 0) ? 2 : 0; }
            else if (variant != 0) { k.cached = (kv != 1 && kv != 2); k.regs = (kv == 2) ? 128 : 255; }     // printed k3: 4th evaluation, on demand
            else switch (kv) {
                case 0: k.cached = 1; k.pred = 2; k.regs = 224; break;     // 8 x 32-thread CTAs per SM, 210 registers: 31.3 against 31.5 ms
                case 7: k.cached = 1; k.pred = 2; break;                   // 8 warps/SM (2 x 128 threads), the round-1 geometry
                case 4: k.cached = 1; k.pred = 1; break;
                case 5: k.cached = 1; break;
                case 3: k.cached = 1; k.regs = 168; break;
                case 2: k.regs = 128; break;
                default: break;
            }
        } else if (kind == 1) {
            if (variant == 0 && (special || kv == 0)) { k.cached = 1; k.pred = 4; }   // blended cell cache, slice difference in per-lane shared-memory slots
            else if (variant == 0 && kv == 6) { k.cached = 1; k.pred = 3; }           // blended cell cache, slice difference gathered through L1 (r2a)
            else if (variant == 0 && kv == 4) { k.cached = 1; k.pred = 2; }           // slice cache + rolling refill, difference gathered per evaluation (r1e)
            else if (!special && (kv == 2 || kv == 3)) k.regs = 128;
        } else {
            if (!special && (kv == 2 || kv == 3)) k.regs = 128;
            else if (!special && P.regroup_every > 0 && ions->n >= 128) k.regroup = 1;
        }
        if (kind == 1 && k.cached) { int rc = tg_build_dtable(ctx); if (rc) return rc; P.f.dtable = ctx->dtable; }
        const TgVariant* sel = nullptr;
        int nb = 0;
        const TgVariant* vb = tg_trace_variants_b(&nb);
        const int na = (int)(sizeof(tg_variants_a) / sizeof(tg_variants_a[0]));
        for (int q = 0; q < na + nb && !sel; ++q) {
            const TgVariant& v = q < na ? tg_variants_a[q] : vb[q - na];
            if (v.kind == k.kind && v.cached == k.cached && v.regs == k.regs && v.pred == k.pred && v.solver == k.solver &&
                v.hasE == k.hasE && v.loss == k.loss && v.bez == k.bez && v.regroup == k.regroup) sel = &v;
        }
        if (!sel) { TG_SET_ERR(ctx, "trace: no kernel for kind %d solver %d with these options", kind, variant); return TAIGA_E_ARG; }
        const int threads = sel->threads;
        int per_sm = ctx->opt_ctas_per_sm > 0 ? ctx->opt_ctas_per_sm : (k.regs == 128 ? 4 : (k.regs == 168 ? 3 : 2));
        if (threads != 128 && ctx->opt_ctas_per_sm <= 0) {     // other CTA shapes: as many CTAs as fit
            TG_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)sel->fn, threads, 0));
            if (per_sm < 1) per_sm = 1;
        }
        unsigned grid = (unsigned)(ctx->sm_count * per_sm);
        unsigned need = (unsigned)((ions->n + threads - 1) / threads);
        if (grid > need) grid = need;
        size_t smem = 0;
        if (k.kind == 1 && k.pred == 4) {          // per-lane slice-difference slots: above the 48 KB static limit
            smem = (size_t)threads * TG_SLOT;
            TG_CUDA(ctx, cudaFuncSetAttribute((const void*)sel->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        }
        sel->fn<<<grid, threads, smem, st>>>(P);
        cudaError_t le = cudaGetLastError();
        if (le != cudaSuccess) {
            cudaFuncAttributes fa;
            memset(&fa, 0, sizeof(fa));
            cudaFuncGetAttributes(&fa, (const void*)sel->fn);
            TG_SET_ERR(ctx, "trace launch (%u x %d threads, %zu B dynamic smem; kernel: %d registers, max %d threads per block, %zu B static smem): %s",
                       grid, threads, smem, fa.numRegs, fa.maxThreadsPerBlock, fa.sharedSizeBytes, cudaGetErrorString(le));
            return TAIGA_E_CUDA;
        }
    }
    ++launches;
    TG_CUDA(ctx, cudaGetLastError());
    if (ions->weight) {        // bookkeeping for taiga_detector_histogram_weighted: which weight arrays hold this context's results
        const double *lo = ions->weight, *hi = ions->weight + ions->n;
        int m = 0;
        for (int q = 0; q < ctx->n_wranges; ++q)
            if (ctx->wranges[q].p + ctx->wranges[q].n <= lo || hi <= ctx->wranges[q].p) ctx->wranges[m++] = ctx->wranges[q];
        if (loss) {
            if (m == 16) { for (int q = 1; q < 16; ++q) ctx->wranges[q - 1] = ctx->wranges[q]; m = 15; }
            ctx->wranges[m].p = lo; ctx->wranges[m].n = ions->n; ++m;
        }
        ctx->n_wranges = m;
    }
    // counters of this trace: copied to the pinned mirror in stream order; taiga_get_stats waits for the stream and reads
    // them ("stats" = 1: wait here, as the library did before round 3)
    TG_CUDA(ctx, cudaMemcpyAsync(ctx->counters_host, ctx->counters, 8 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    ctx->stats_launches = launches;
    ctx->stats_pending = true;
    if (ctx->opt_stats) return tg_collect_stats(ctx);
    return TAIGA_OK;
}
