// heat_tband_variants.h -- table of the compiled heat_tband_kernel<WL, NW, DEGK> instances
// (heat_tband2.cu, heat_tband4.cu: lambda polynomials of degree <= 2 / <= 4).
#pragma once
#include <cstddef>

#include "heat_wband_params.cuh"

namespace heat {

typedef void (*tband_kernel_fn)(const WParams);
struct TBandVariant {
    int WL, NW, DEGK, CL, LPB;
    tband_kernel_fn fn;
    const char *name;
    size_t smem_fixed; // bytes without the layer table
};
extern const TBandVariant k_tband_variants2[];
extern const int k_ntband_variants2;
extern const TBandVariant k_tband_variants4[];
extern const int k_ntband_variants4;

#define HEAT_TBAND_VARIANT(WL_, NW_, D_)                                                          \
    {                                                                                             \
        WL_, NW_, D_, TBandCfg<WL_, NW_>::CL, TBandCfg<WL_, NW_>::LPB, heat_tband_kernel<WL_, NW_, D_>, \
            "tband<WL=" #WL_ ",NW=" #NW_ ",DEGK=" #D_ ">", TBandCfg<WL_, NW_>::smem_bytes(0)       \
    }
// warps per line 1..16 (nr = 512..8192) in CTAs of 4 warps (four CTAs per SM); for nr = 4096 and 8192
// also CTAs of 8 and 16 warps (a whole line per CTA: no cluster; these are the defaults)
#define HEAT_TBAND_VARIANTS(D_)                                                                   \
    HEAT_TBAND_VARIANT(1, 4, D_), HEAT_TBAND_VARIANT(2, 4, D_), HEAT_TBAND_VARIANT(4, 4, D_),     \
        HEAT_TBAND_VARIANT(8, 4, D_), HEAT_TBAND_VARIANT(8, 8, D_), HEAT_TBAND_VARIANT(16, 4, D_), \
        HEAT_TBAND_VARIANT(16, 8, D_), HEAT_TBAND_VARIANT(16, 16, D_)

} // namespace heat
