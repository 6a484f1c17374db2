// heat_line_a.cu -- instances of the general line kernel with 4 and 8 rows per thread.
#include "heat_line_kernel.cuh"
#include "heat_line_variants.h"

namespace heat {
const Variant k_variants_a[] = {
    HEAT_VARIANT(4, 8),  HEAT_VARIANT(4, 16),  HEAT_VARIANT(4, 32),  HEAT_VARIANT(8, 32),   HEAT_VARIANT(8, 64),
    HEAT_VARIANT(8, 128), HEAT_VARIANT(8, 256), HEAT_VARIANT(8, 512), HEAT_VARIANT(8, 1024),
};
const int k_nvariants_a = (int)(sizeof(k_variants_a) / sizeof(k_variants_a[0]));
} // namespace heat
