// heat_band.cu -- instances of the band kernel (heat_band_kernel.cuh) and their launch table.
#include "heat_band_kernel.cuh"
#include "heat_band_variants.h"

namespace heat {

#define HEAT_BAND_VARIANT(G_, CL_, D_)                                                            \
    {                                                                                             \
        G_, CL_, D_, heat_band_kernel<G_, CL_, D_>, "band<G=" #G_ ",CL=" #CL_ ",DEGK=" #D_ ">",    \
            BandCfg<G_, CL_>::smem_bytes(0)                                                       \
    }
const BandVariant k_band_variants[] = {
    HEAT_BAND_VARIANT(64, 1, 2),  HEAT_BAND_VARIANT(128, 1, 2), HEAT_BAND_VARIANT(256, 1, 2),
    HEAT_BAND_VARIANT(256, 2, 2), HEAT_BAND_VARIANT(256, 4, 2), HEAT_BAND_VARIANT(64, 1, 4),
    HEAT_BAND_VARIANT(128, 1, 4), HEAT_BAND_VARIANT(256, 1, 4), HEAT_BAND_VARIANT(256, 2, 4),
    HEAT_BAND_VARIANT(256, 4, 4),
};
const int k_nband_variants = (int)(sizeof(k_band_variants) / sizeof(k_band_variants[0]));

} // namespace heat
