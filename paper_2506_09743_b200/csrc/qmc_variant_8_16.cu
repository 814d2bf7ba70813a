// The (NS, NMO, exact) = (8, 16, false) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_8_16
#define QMC_VARIANT_ARGS 8, 16, false
#include "qmc_variant.cuh"
