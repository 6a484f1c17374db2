// heat_wband4.cu -- instances of the warp-autonomous band kernel for lambda polynomials of degree <= 4.
#include "heat_wband_kernel.cuh"
#include "heat_wband_variants.h"

namespace heat {
const WBandVariant k_wband_variants4[] = {HEAT_WBAND_VARIANTS(4)};
const int k_nwband_variants4 = (int)(sizeof(k_wband_variants4) / sizeof(k_wband_variants4[0]));
} // namespace heat
