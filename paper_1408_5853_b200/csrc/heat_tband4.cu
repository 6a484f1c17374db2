// heat_tband4.cu -- instances of the tensor-memory band kernel for lambda polynomials of degree <= 4.
#include "heat_tband_kernel.cuh"
#include "heat_tband_variants.h"

namespace heat {
const TBandVariant k_tband_variants4[] = {HEAT_TBAND_VARIANTS(4)};
const int k_ntband_variants4 = (int)(sizeof(k_tband_variants4) / sizeof(k_tband_variants4[0]));
} // namespace heat
