// heat_tband2.cu -- instances of the tensor-memory band kernel for lambda polynomials of degree <= 2.
#include "heat_tband_kernel.cuh"
#include "heat_tband_variants.h"

namespace heat {
const TBandVariant k_tband_variants2[] = {HEAT_TBAND_VARIANTS(2)};
const int k_ntband_variants2 = (int)(sizeof(k_tband_variants2) / sizeof(k_tband_variants2[0]));
} // namespace heat
