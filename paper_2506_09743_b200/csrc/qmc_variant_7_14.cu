// The (NS, NMO, exact) = (7, 14, true) instantiation of the template kernels (see qmc_variant.cuh).
#define QMC_VARIANT_TU
#define QMC_VARIANT_NAME variant_7_14
#define QMC_VARIANT_ARGS 7, 14, true
#include "qmc_variant.cuh"
