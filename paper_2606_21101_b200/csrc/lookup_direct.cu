// lookup_direct.cu -- short-bag variant of step a3 (DPI_OPT_MODE = 6, and the automatic choice when the plan's capacity
// says bags are short: max_indices <= 4 * G). Algorithm 1's division of labour (every thread fills its own
// piece of the output matrix, no shared control flow) carried over to CSR bags: lane group q (W lanes = one row) owns bags
// q, q + n_groups, ...; for each it reads offsets[g], offsets[g+1] straight from the plan, gathers and pools the bag's rows
// in registers and stores the pooled vector. U bags per lane group are processed side by side (independent chains).
// No segments, no staging, no per-task pipeline: the planned kernel spends ~36 warp instructions per 1-3-row bag on that
// machinery; this one spends what the bag itself needs. Long bags would serialise inside one lane group,
// which is why the balanced-segment kernel stays the default whenever bags can be long.
// Same arithmetic as lookup_kernel: fp32 accumulation in entry order, one RNE cast at the store, mean by reciprocal,
// bags of length <= 1 bit-exact, empty bags +0.0.
#include "lookup_kernels.cuh"

namespace dpi {
namespace {

template <class Tr, int W, int U, bool OUT32>
__global__ void __launch_bounds__(256) direct_kernel(const LookupArgs a) {
    constexpr int kAcc2 = Tr::kAcc / 2;
    constexpr int kOutVec = (OUT32 && Tr::kAcc == 8) ? 32 : 16;
    extern __shared__ const char* s_tab_direct[];
    for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) s_tab_direct[t] = static_cast<const char*>(a.tables[t]);
    __syncthreads();
    griddep_wait();  // PDL: the planner's offsets are visible past this point (no-op otherwise)
    const uint32_t lane_id = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t q = lane_id / W, sl = lane_id % W;
    const uint32_t n_groups = (gridDim.x * blockDim.x) / W;
    const bool vec_ok = sl < a.nvec;
    const uint32_t row_bytes = a.nvec * 16;
    const uint32_t t_step = n_groups % a.T;
    char* const out = static_cast<char*>(a.out);
    uint32_t t = q % a.T;
    for (uint32_t g0 = q; g0 < a.G; g0 += n_groups * U) {
        int lo[U], len[U];
        uint32_t tt[U];
        int max_len = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            const bool ok = g < a.G;
            tt[u] = t;
            lo[u] = ok ? __ldg(a.offsets + g) : 0;
            len[u] = ok ? __ldg(a.offsets + g + 1) - lo[u] : 0;
            max_len = max(max_len, len[u]);
            t += t_step;
            if (t >= a.T) t -= a.T;
        }
        float2 acc[U][kAcc2];
#pragma unroll
        for (int u = 0; u < U; ++u) zero_acc(acc[u]);
        for (int j = 0; j < max_len; ++j) {
            uint4 v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool ok = vec_ok && j < len[u];
                // int64 ids are read through their low words (little-endian, rows < 2^31): idx_shift = 1
                const uint32_t r = ok ? static_cast<uint32_t>(__ldg(a.indices + (static_cast<size_t>(lo[u] + j) << a.idx_shift))) : 0u;
                v[u] = ld_row16(s_tab_direct[tt[u]] + static_cast<uint64_t>(r) * row_bytes + sl * 16, ok);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) Tr::add(acc[u], v[u]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            if (vec_ok && g < a.G) {
                if (((a.pool.w[tt[u] >> 5] >> (tt[u] & 31)) & 1u) && len[u] > 1) scale_mean(acc[u], len[u]);
                store_pooled<Tr, OUT32>(out + (static_cast<size_t>(g) * a.nvec + sl) * kOutVec, acc[u]);
            }
        }
    }
}

template <class Tr, bool OUT32>
cudaError_t launch_direct_t(const LookupArgs& a, int lanes, int num_sms, bool pdl, cudaStream_t stream) {
    constexpr int U = 2;
    const unsigned long long lanes_needed = (static_cast<unsigned long long>(a.G) * lanes + U - 1) / U;
    unsigned long long ctas = (lanes_needed + 255) / 256;
    if (ctas < 1) ctas = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(static_cast<unsigned>(ctas));
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = static_cast<size_t>(a.T) * sizeof(const char*);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    count_launch();
    // One resident wave at most: CTAs beyond SMs x occupancy would only queue behind the first wave and leave a ragged tail
    // (c3: 1.6 waves at a fixed cap of 8 per SM cost 9 %); the kernel strides over the bags instead.
    switch (lanes) {
#define DPI_DIRECT(w)                                                                                                         \
    case w: {                                                                                                                 \
        static int occ = 0;                                                                                                   \
        if (occ == 0 && (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, direct_kernel<Tr, w, U, OUT32>, 256,             \
                                                                       cfg.dynamicSmemBytes) != cudaSuccess || occ < 1)) {    \
            (void)cudaGetLastError();                                                                                         \
            occ = 4;                                                                                                          \
        }                                                                                                                     \
        const unsigned long long cap = static_cast<unsigned long long>(num_sms > 0 ? num_sms : 148) * occ;                    \
        cfg.gridDim = dim3(static_cast<unsigned>(ctas > cap ? cap : ctas));                                                   \
        return cudaLaunchKernelEx(&cfg, direct_kernel<Tr, w, U, OUT32>, a);                                                   \
    }
        DPI_DIRECT(1) DPI_DIRECT(2) DPI_DIRECT(4) DPI_DIRECT(8) DPI_DIRECT(16) DPI_DIRECT(32)
#undef DPI_DIRECT
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_direct(const LookupArgs& a, int dtype, bool out32, int lanes, int num_sms, bool pdl, cudaStream_t stream) {
    switch (dtype) {
        case DPI_F32: return launch_direct_t<F32Traits, false>(a, lanes, num_sms, pdl, stream);
        case DPI_F16: return out32 ? launch_direct_t<F16Traits, true>(a, lanes, num_sms, pdl, stream)
                                   : launch_direct_t<F16Traits, false>(a, lanes, num_sms, pdl, stream);
        default: return out32 ? launch_direct_t<BF16Traits, true>(a, lanes, num_sms, pdl, stream)
                              : launch_direct_t<BF16Traits, false>(a, lanes, num_sms, pdl, stream);
    }
}

}  // namespace dpi
