// lookup_bf16.cu -- instantiates the fused gather-and-pool kernel (lookup_kernels.cuh) for bf16 tables.
#include "lookup_kernels.cuh"
#define DPI_TRAITS BF16Traits
#define DPI_SUFFIX bf16
#include "lookup_dispatch.inc"
