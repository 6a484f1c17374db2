// heat_wband2.cu -- instances of the warp-autonomous band kernel for lambda polynomials of degree <= 2.
#include "heat_wband_kernel.cuh"
#include "heat_wband_variants.h"

namespace heat {
const WBandVariant k_wband_variants2[] = {HEAT_WBAND_VARIANTS(2)};
const int k_nwband_variants2 = (int)(sizeof(k_wband_variants2) / sizeof(k_wband_variants2[0]));
} // namespace heat
