// a3 + a4, second translation unit of the k_trace instantiations (compiled in parallel with trace.cu): the variants with
// an electric field (uniform and / or gridded, Eq. 3) and the other solvers (Eq. 4, Eq. 7-8), alone and combined with the
// loss integral and the Bezier interpolation.
#include "trace_kernel.cuh"

static const TgVariant tg_variants_b[] = {
    // uniform / gridded E and / or the other solvers (Eq. 4, Eq. 7-8)
    TG_V(0, 1, 255, 2, 0, 1, 0, 0, 0), TG_V(0, 1, 255, 0, 0, 1, 0, 0, 0), TG_V(0, 1, 255, 0, 2, 1, 0, 0, 0), TG_V(0, 1, 255, 0, 3, 1, 0, 0, 0),
    TG_V(1, 1, 255, 4, 0, 1, 0, 0, 0), TG_V(1, 0, 255, 0, 0, 1, 0, 0, 0), TG_V(1, 0, 255, 0, 2, 1, 0, 0, 0), TG_V(1, 0, 255, 0, 3, 1, 0, 0, 0),
    TG_V(2, 0, 255, 0, 0, 1, 0, 0, 0), TG_V(2, 0, 255, 0, 2, 1, 0, 0, 0), TG_V(2, 0, 255, 0, 3, 1, 0, 0, 0),
    // the loss integral with an electric field and with the other solvers
    TG_V(0, 1, 255, 2, 0, 1, 1, 0, 0), TG_V(0, 1, 255, 0, 0, 1, 1, 0, 0), TG_V(0, 1, 255, 0, 2, 1, 1, 0, 0), TG_V(0, 1, 255, 0, 3, 1, 1, 0, 0),
    TG_V(1, 1, 255, 4, 0, 1, 1, 0, 0), TG_V(1, 0, 255, 0, 0, 1, 1, 0, 0), TG_V(1, 0, 255, 0, 2, 1, 1, 0, 0), TG_V(1, 0, 255, 0, 3, 1, 1, 0, 0),
    TG_V(2, 0, 255, 0, 0, 1, 1, 0, 0), TG_V(2, 0, 255, 0, 2, 1, 1, 0, 0), TG_V(2, 0, 255, 0, 3, 1, 1, 0, 0),
    // the Bezier interpolation with an electric field, alone and with the loss integral
    TG_V(0, 1, 255, 2, 0, 1, 0, 1, 0), TG_V(0, 1, 255, 0, 0, 1, 0, 1, 0), TG_V(1, 1, 255, 4, 0, 1, 0, 1, 0), TG_V(1, 0, 255, 0, 0, 1, 0, 1, 0),
    TG_V(2, 0, 255, 0, 0, 1, 0, 1, 0),
    TG_V(0, 1, 255, 2, 0, 1, 1, 1, 0), TG_V(0, 1, 255, 0, 0, 1, 1, 1, 0), TG_V(1, 1, 255, 4, 0, 1, 1, 1, 0), TG_V(1, 0, 255, 0, 0, 1, 1, 1, 0),
    TG_V(2, 0, 255, 0, 0, 1, 1, 1, 0),
};

const TgVariant* tg_trace_variants_b(int* n) {
    *n = (int)(sizeof(tg_variants_b) / sizeof(tg_variants_b[0]));
    return tg_variants_b;
}
