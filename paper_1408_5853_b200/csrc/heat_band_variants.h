// heat_band_variants.h -- table of the compiled heat_band_kernel<G, CL, DEGK> instances.
// The instances live in their own translation unit (heat_band.cu) so that the two halves of
// the library compile in parallel; heat_api.cu only needs the launch table.
#pragma once
#include <cstddef>

#include "heat_band_params.cuh"

namespace heat {

typedef void (*band_kernel_fn)(const BParams);
struct BandVariant {
    int G, CL, DEGK, NT;
    band_kernel_fn fn;
    const char *name;
    size_t smem_fixed; // bytes without the layer table
};
extern const BandVariant k_band_variants[];
extern const int k_nband_variants;

} // namespace heat
