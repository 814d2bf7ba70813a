// The (NS, NMO, exact) = (4, 8, false) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_4_8
#define QMC_VARIANT_ARGS 4, 8, false
#include "qmc_variant.cuh"
