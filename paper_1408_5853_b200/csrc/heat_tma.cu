// heat_tma.cu -- instances of the TMA line kernel.
#include "heat_tma_kernel.cuh"
#include "heat_line_variants.h"

namespace heat {
const TmaVariant k_tma_variants[] = {
    HEAT_TMA_VARIANT(8, 1),   HEAT_TMA_VARIANT(16, 1),  HEAT_TMA_VARIANT(32, 1),  HEAT_TMA_VARIANT(64, 1),
    HEAT_TMA_VARIANT(128, 1), HEAT_TMA_VARIANT(128, 2), HEAT_TMA_VARIANT(128, 4),
};
const int k_ntma_variants = (int)(sizeof(k_tma_variants) / sizeof(k_tma_variants[0]));
} // namespace heat
