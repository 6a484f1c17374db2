// heat_wband_variants.h -- table of the compiled heat_wband_kernel<WL, NW, DEGK> instances.
// The instances live in their own translation units (heat_wband2.cu, heat_wband4.cu: lambda
// polynomials of degree <= 2 / <= 4) so that the library compiles in parallel.
#pragma once
#include <cstddef>

#include "heat_wband_params.cuh"

namespace heat {

typedef void (*wband_kernel_fn)(const WParams);
struct WBandVariant {
    int WL, NW, DEGK, CL, LPB;
    wband_kernel_fn fn;
    const char *name;
    size_t smem_fixed; // bytes without the layer table
};
extern const WBandVariant k_wband_variants2[];
extern const int k_nwband_variants2;
extern const WBandVariant k_wband_variants4[];
extern const int k_nwband_variants4;

#define HEAT_WBAND_VARIANT(WL_, NW_, D_)                                                          \
    {                                                                                             \
        WL_, NW_, D_, WBandCfg<WL_, NW_>::CL, WBandCfg<WL_, NW_>::LPB, heat_wband_kernel<WL_, NW_, D_>, \
            "wband<WL=" #WL_ ",NW=" #NW_ ",DEGK=" #D_ ">", WBandCfg<WL_, NW_>::smem_bytes(0)       \
    }
// warps per line 1..16 (nr = 512..8192) in CTAs of 4 warps (two CTAs per SM); for nr = 8192 also
// CTAs of 2 and 8 warps (clusters of 8 and 2)
#define HEAT_WBAND_VARIANTS(D_)                                                                   \
    HEAT_WBAND_VARIANT(1, 4, D_), HEAT_WBAND_VARIANT(2, 4, D_), HEAT_WBAND_VARIANT(4, 4, D_),     \
        HEAT_WBAND_VARIANT(8, 4, D_), HEAT_WBAND_VARIANT(16, 4, D_), HEAT_WBAND_VARIANT(16, 2, D_), \
        HEAT_WBAND_VARIANT(16, 8, D_)

} // namespace heat
