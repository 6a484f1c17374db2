// heat_line_b.cu -- instances of the general line kernel with 16 rows per thread.
#include "heat_line_kernel.cuh"
#include "heat_line_variants.h"

namespace heat {
const Variant k_variants_b[] = {
    HEAT_VARIANT(16, 32), HEAT_VARIANT(16, 64), HEAT_VARIANT(16, 128), HEAT_VARIANT(16, 256), HEAT_VARIANT(16, 512),
};
const int k_nvariants_b = (int)(sizeof(k_variants_b) / sizeof(k_variants_b[0]));
} // namespace heat
