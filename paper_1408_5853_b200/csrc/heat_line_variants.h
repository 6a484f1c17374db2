// heat_line_variants.h -- tables of the compiled heat_line_kernel<M, G> / heat_line_persist_kernel<M, G>
// instances (heat_line_a.cu: M = 4, 8; heat_line_b.cu: M = 16) and of the heat_tma_kernel<G, CL>
// instances (heat_tma.cu).  The kernels live in translation units of their own so that the library
// builds in parallel.
#pragma once
#include <cstddef>

#include "heat_device.cuh"
#include "heat_tma_kernel.cuh"

namespace heat {

typedef void (*kernel_fn)(const KParams);
struct Variant {
    int M, G, tpb, lpb;
    kernel_fn fn, fn_persist, fn_iter;
    const char *name;
    size_t smem_fixed; // bytes without the layer table
};
extern const Variant k_variants_a[];
extern const int k_nvariants_a;
extern const Variant k_variants_b[];
extern const int k_nvariants_b;

#define HEAT_VARIANT(M_, G_)                                                                      \
    {                                                                                             \
        M_, G_, LineCfg<M_, G_>::TPB, LineCfg<M_, G_>::LPB, heat_line_kernel<M_, G_>,             \
            heat_line_persist_kernel<M_, G_>, heat_line_iter_kernel<M_, G_>,                      \
            "line<M=" #M_ ",G=" #G_ ">", LineCfg<M_, G_>::smem_bytes(0)                           \
    }

typedef void (*tma_kernel_fn)(const TParams);
struct TmaVariant {
    int G, CL;
    tma_kernel_fn fn;
    const char *name;
    size_t smem_fixed; // bytes without the layer table
};
extern const TmaVariant k_tma_variants[];
extern const int k_ntma_variants;

#define HEAT_TMA_VARIANT(G_, CL_)                                                                 \
    {                                                                                             \
        G_, CL_, heat_tma_kernel<G_, CL_>, "tma<G=" #G_ ",CL=" #CL_ ">", TmaCfg<G_, CL_>::smem_bytes(0) \
    }

} // namespace heat
