// The (NS, NMO, exact) = (1, 2, true) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_1_2
#define QMC_VARIANT_ARGS 1, 2, true
#include "qmc_variant.cuh"
