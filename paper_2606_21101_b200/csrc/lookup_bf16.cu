// lookup_bf16.cu -- instantiates the fused gather-and-pool kernel (lookup_kernels.cuh) for bf16 tables
// (output in bf16, or in fp32 when the plan asks for it).
#include "lookup_kernels.cuh"
#define DPI_TRAITS BF16Traits
#define DPI_SUFFIX bf16
#define DPI_HAS_OUT32 1
#include "lookup_dispatch.inc"
