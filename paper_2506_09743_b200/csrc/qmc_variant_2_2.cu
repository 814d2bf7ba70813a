// The (NS, NMO, exact) = (2, 2, true) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_2_2
#define QMC_VARIANT_ARGS 2, 2, true
#include "qmc_variant.cuh"
