// The (NS, NMO, exact) = (3, 8, true) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_3_8
#define QMC_VARIANT_ARGS 3, 8, true
#include "qmc_variant.cuh"
