// lookup_onehot.cu -- Algorithm 1 itself: the one-hot multi-table lookup, where the workload is
// pure arithmetic ("deterministic and known in advance") and needs no plan: IDs[b x k] in, the
// concatenated EmbedOut[b x (k*d)] out, one launch, no offsets, no segments, no accumulation -- a row copy.
//
// Granularity is the one of lookup_kernel (one lane per 16-byte vector, W lanes per row, R15), the mapping
// the paper's output-first one: consecutive lanes fill consecutive output addresses. Lane group
// q of the grid owns bags q, q + n_groups, ... ; it first issues U id loads, then U row loads, then U stores, so a
// lane has U independent request chains in flight and the kernel is two dependent memory round trips deep
// (id -> row) instead of the planned path's three (segment -> staged ids -> row).
// The table id of a bag is g mod k computed once; later bags of the same lane group step it by (stride mod k).
#include "dpi_internal.cuh"

namespace dpi {
namespace {

struct OnehotArgs {
    const void* const* __restrict__ tables;
    const int32_t* __restrict__ ids;   // [G], g = b*T + t, or int64 read through its low word (idx_shift = 1)
    char* __restrict__ out;            // [G * nvec * 16] bytes
    uint32_t G, T, nvec, idx_shift;
};

template <int W, int U>
__global__ void __launch_bounds__(256) onehot_kernel(const OnehotArgs a) {
    extern __shared__ const char* s_tab[];
    for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) s_tab[t] = static_cast<const char*>(a.tables[t]);
    __syncthreads();
    const uint32_t lane_id = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t q = lane_id / W, sl = lane_id % W;
    const uint32_t n_groups = (gridDim.x * blockDim.x) / W;
    const bool vec_ok = sl < a.nvec;
    const uint32_t row_bytes = a.nvec * 16;
    const uint32_t t_step = n_groups % a.T;
    uint32_t t = q % a.T;
    for (uint32_t g0 = q; g0 < a.G; g0 += n_groups * U) {
        uint32_t r[U], tt[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            tt[u] = t;
            r[u] = g < a.G ? static_cast<uint32_t>(__ldg(a.ids + (static_cast<size_t>(g) << a.idx_shift))) : 0u;
            t += t_step;
            if (t >= a.T) t -= a.T;
        }
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            v[u] = make_uint4(0u, 0u, 0u, 0u);
            if (vec_ok && g < a.G)
                v[u] = __ldg(reinterpret_cast<const uint4*>(s_tab[tt[u]] + static_cast<uint64_t>(r[u]) * row_bytes + sl * 16));
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            if (vec_ok && g < a.G) {
                char* po = a.out + (static_cast<size_t>(g) * a.nvec + sl) * 16;
                asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(po), "r"(v[u].x), "r"(v[u].y), "r"(v[u].z),
                             "r"(v[u].w) : "memory");
            }
        }
    }
}

}  // namespace

cudaError_t launch_onehot(const void* const* tables, const void* ids, uint32_t idx_shift, void* out, uint32_t G, uint32_t T,
                          uint32_t nvec, int lanes, int num_sms, cudaStream_t stream) {
    OnehotArgs a{tables, static_cast<const int32_t*>(ids), static_cast<char*>(out), G, T, nvec, idx_shift};
    constexpr int U = 4;
    const unsigned long long lanes_needed = (static_cast<unsigned long long>(G) * lanes + U - 1) / U;  // U bags per lane group
    unsigned long long ctas = (lanes_needed + 255) / 256;
    const unsigned long long cap = static_cast<unsigned long long>(num_sms > 0 ? num_sms : 148) * 8;
    if (ctas > cap) ctas = cap;
    if (ctas < 1) ctas = 1;
    const size_t smem = static_cast<size_t>(T) * sizeof(const char*);
    count_launch();
    switch (lanes) {
#define DPI_OH(w) case w: onehot_kernel<w, U><<<static_cast<unsigned>(ctas), 256, smem, stream>>>(a); break;
        DPI_OH(1) DPI_OH(2) DPI_OH(4) DPI_OH(8) DPI_OH(16) DPI_OH(32)
#undef DPI_OH
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace dpi
