// lookup_f32.cu -- instantiates the fused gather-and-pool kernel (lookup_kernels.cuh) for f32 tables.
#include "lookup_kernels.cuh"
#define DPI_TRAITS F32Traits
#define DPI_SUFFIX f32
#include "lookup_dispatch.inc"
