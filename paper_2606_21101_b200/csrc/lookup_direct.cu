// lookup_direct.cu -- the short-bag variant of step a3 as its own launch: one lane group per bag straight from the
// plan's offsets (short_bag_body in lookup_kernels.cuh, which also documents the mapping).
// Chosen on the HOST: DPI_OPT_MODE = 6, or DPI_OPT_MAX_BAG_HINT = L with L <= 8 (a caller's optional promise, checked
// off the hot path by dpi_check_indices). Without either, dpi_lookup launches lookup_kernel, which reads a1's max_len
// on the DEVICE and branches into the same body -- no promise needed; this separate launch only buys the smaller
// register footprint (40-46 registers, 5-6 resident CTAs per SM instead of 4) and is kept for A/B measurements.
// Long bags would serialise inside one lane group, which is why the balanced-segment kernel is the default whenever
// bags can be long.
#include "lookup_kernels.cuh"

namespace dpi {
namespace {

constexpr int kDirectU = 2;   // bags side by side per lane group (U = 1 / 4 measured slower on c3: 23.2 / 28.7 us vs 20.8)

template <class Tr, int W, bool OUT32>
__global__ void __launch_bounds__(256) direct_kernel(const LookupArgs a) {
    extern __shared__ const char* s_tab_direct[];
    griddep_wait();  // PDL: nothing (table pointers included) is read before the preceding grid has completed
    const int S = ld_plan(a.meta + META_S);   // S == 0 marks an overflowed plan (N > max_indices): its offsets may point past indices
    for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) s_tab_direct[t] = static_cast<const char*>(a.tables[t]);
    __syncthreads();
    if (S == 0) return;
    const uint32_t lane_id = blockIdx.x * blockDim.x + threadIdx.x;
    short_bag_body<Tr, W, kDirectU, OUT32>(a, s_tab_direct, lane_id / W, lane_id % W, (gridDim.x * blockDim.x) / W);
}

template <class Tr, bool OUT32, class F>
auto for_lanes(int lanes, F&& f) {
    switch (lanes) {
        case 1: return f(direct_kernel<Tr, 1, OUT32>);
        case 2: return f(direct_kernel<Tr, 2, OUT32>);
        case 4: return f(direct_kernel<Tr, 4, OUT32>);
        case 8: return f(direct_kernel<Tr, 8, OUT32>);
        case 16: return f(direct_kernel<Tr, 16, OUT32>);
        case 32: return f(direct_kernel<Tr, 32, OUT32>);
        default: return f(static_cast<void (*)(const LookupArgs)>(nullptr));
    }
}

template <class F>
auto for_kernel(int dtype, bool out32, int lanes, F&& f) {
    switch (dtype) {
        case DPI_F32: return for_lanes<F32Traits, false>(lanes, f);
        case DPI_F16: return out32 ? for_lanes<F16Traits, true>(lanes, f) : for_lanes<F16Traits, false>(lanes, f);
        default: return out32 ? for_lanes<BF16Traits, true>(lanes, f) : for_lanes<BF16Traits, false>(lanes, f);
    }
}

}  // namespace

// Resident CTAs per SM of the instantiation (per plan, never per lookup); >= 1.
int direct_occupancy(int dtype, bool out32, int lanes, uint32_t T) {
    return for_kernel(dtype, out32, lanes, [&](void (*k)(const LookupArgs)) -> int {
        int occ = 0;
        if (!k || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, 256, static_cast<size_t>(T) * sizeof(const char*)) != cudaSuccess || occ < 1) {
            (void)cudaGetLastError();
            occ = 4;
        }
        return occ;
    });
}

cudaError_t launch_direct(const LookupArgs& a, int dtype, bool out32, int lanes, int grid_cap, bool pdl, cudaStream_t stream) {
    return for_kernel(dtype, out32, lanes, [&](void (*k)(const LookupArgs)) -> cudaError_t {
        if (!k) return cudaErrorInvalidValue;
        const unsigned long long lanes_needed = (static_cast<unsigned long long>(a.G) * lanes + kDirectU - 1) / kDirectU;
        unsigned long long ctas = (lanes_needed + 255) / 256;
        // One resident wave at most: CTAs beyond SMs x occupancy would only queue behind the first wave and leave a ragged
        // tail (c3: 1.6 waves at a fixed cap of 8 per SM cost 9 %); the kernel strides over the bags instead.
        if (grid_cap > 0 && ctas > static_cast<unsigned long long>(grid_cap)) ctas = grid_cap;
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
        return cudaLaunchKernelEx(&cfg, k, a);
    });
}

}  // namespace dpi
