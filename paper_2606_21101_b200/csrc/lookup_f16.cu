// lookup_f16.cu -- instantiates the fused gather-and-pool kernel (lookup_kernels.cuh) for f16 tables
// (output in f16, or in fp32 when the plan asks for it).
#include "lookup_kernels.cuh"
#define DPI_TRAITS F16Traits
#define DPI_SUFFIX f16
#define DPI_HAS_OUT32 1
#include "lookup_dispatch.inc"
