// lookup_f16.cu -- instantiates the fused gather-and-pool kernel (lookup_kernels.cuh) for f16 tables.
#include "lookup_kernels.cuh"
#define DPI_TRAITS F16Traits
#define DPI_SUFFIX f16
#include "lookup_dispatch.inc"
