// ablation_input_first.cu -- the paper's strawman thread mapping, kept as a measured ablation (SURVEY.md §8(f)
// NEXT-1): "The input-first scheme involves maximizing the allocation of different input samples among
// threads": one THREAD per sample walks that sample's T bags and their entries serially.
// "Even though the input reads have a sequentially addressed pattern, the table lookups and output writes
// will involve random reads and writes": the lanes of a warp touch 32 different table rows and
// 32 different output rows at every step, so every 128-bit access of a warp is its own 32-byte sector.
// Same arithmetic and same results as lookup_kernel (fp32 accumulate, one RNE cast at the store); only the
// workload allocation differs. Fig. 11 of the paper reports output-first up to 10.3x faster.
#include "lookup_kernels.cuh"

namespace dpi {
namespace {

// Column slices are walked kGroup 16-byte vectors at a time (128 B of row), so a bag's index entries are read once for rows
// up to 128 B and once per 128-byte slice beyond that (the accumulators of a whole 512-byte row do not fit in registers).
template <class Tr, bool OUT32>
__global__ void __launch_bounds__(128) input_first_kernel(const LookupArgs a, const uint32_t B) {
    constexpr int kAcc = Tr::kAcc;
    constexpr uint32_t kGroup = 8;
    constexpr size_t kOutVec = (OUT32 && kAcc == 8) ? 32 : 16;
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const size_t row_bytes = static_cast<size_t>(a.nvec) * 16;
    char* const out = static_cast<char*>(a.out);
    for (uint32_t t = 0; t < a.T; ++t) {
        const size_t g = static_cast<size_t>(b) * a.T + t;
        const int lo = __ldg(a.offsets + g), hi = __ldg(a.offsets + g + 1);
        const char* tab = static_cast<const char*>(a.tables[t]);
        const bool mean = ((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1;
        for (uint32_t v0 = 0; v0 < a.nvec; v0 += kGroup) {
            float2 acc[kGroup][kAcc / 2];
#pragma unroll
            for (uint32_t v = 0; v < kGroup; ++v) zero_acc(acc[v]);
            for (int j = lo; j < hi; ++j) {
                const char* row = tab + static_cast<size_t>(static_cast<uint32_t>(__ldg(a.indices + j))) * row_bytes + v0 * 16;
#pragma unroll
                for (uint32_t v = 0; v < kGroup; ++v) Tr::add(acc[v], ld_row16(row + v * 16, v0 + v < a.nvec));
            }
#pragma unroll
            for (uint32_t v = 0; v < kGroup; ++v) {
                if (v0 + v < a.nvec) {
                    if (mean) scale_mean(acc[v], hi - lo);
                    store_pooled<Tr, OUT32>(out + (g * a.nvec + v0 + v) * kOutVec, acc[v]);
                }
            }
        }
    }
}

}  // namespace

cudaError_t launch_input_first(const LookupArgs& a, uint32_t B, int dtype, bool out32, cudaStream_t stream) {
    // one thread per sample is the scheme itself; small batches get 32-thread CTAs so that they still spread over the SMs
    const unsigned bt = B >= 148u * 128u ? 128u : 32u;
    const dim3 block(bt), grid((B + bt - 1) / bt);
    count_launch();
    switch (dtype) {
        case DPI_F32: input_first_kernel<F32Traits, false><<<grid, block, 0, stream>>>(a, B); break;
        case DPI_F16:
            if (out32) input_first_kernel<F16Traits, true><<<grid, block, 0, stream>>>(a, B);
            else input_first_kernel<F16Traits, false><<<grid, block, 0, stream>>>(a, B);
            break;
        default:
            if (out32) input_first_kernel<BF16Traits, true><<<grid, block, 0, stream>>>(a, B);
            else input_first_kernel<BF16Traits, false><<<grid, block, 0, stream>>>(a, B);
            break;
    }
    return cudaGetLastError();
}

}  // namespace dpi
