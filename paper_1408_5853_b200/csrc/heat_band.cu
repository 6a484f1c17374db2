// heat_band.cu -- instances of the band kernel (heat_band_kernel.cuh) and their launch table.
#include "heat_band_kernel.cuh"
#include "heat_band_variants.h"

namespace heat {

#define HEAT_BAND_VARIANT(G_, CL_, D_, NT_)                                                       \
    {                                                                                             \
        G_, CL_, D_, NT_, heat_band_kernel<G_, CL_, D_, NT_>,                                     \
            "band<G=" #G_ ",CL=" #CL_ ",DEGK=" #D_ ",NT=" #NT_ ">", BandCfg<G_, CL_, NT_>::smem_bytes(0) \
    }
#define HEAT_BAND_VARIANTS(D_)                                                                    \
    HEAT_BAND_VARIANT(64, 1, D_, 256), HEAT_BAND_VARIANT(128, 1, D_, 256), HEAT_BAND_VARIANT(256, 1, D_, 256), \
        HEAT_BAND_VARIANT(256, 2, D_, 256), HEAT_BAND_VARIANT(256, 4, D_, 256), HEAT_BAND_VARIANT(64, 1, D_, 128), \
        HEAT_BAND_VARIANT(128, 1, D_, 128), HEAT_BAND_VARIANT(128, 2, D_, 128), HEAT_BAND_VARIANT(128, 4, D_, 128), \
        HEAT_BAND_VARIANT(128, 8, D_, 128)
const BandVariant k_band_variants[] = {HEAT_BAND_VARIANTS(2), HEAT_BAND_VARIANTS(4)};
const int k_nband_variants = (int)(sizeof(k_band_variants) / sizeof(k_band_variants[0]));

} // namespace heat
