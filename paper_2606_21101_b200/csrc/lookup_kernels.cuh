// lookup_kernels.cuh -- step a3: the fused multi-table gather-and-pool (Alg. 1, generalised
// to CSR bags per PAPER.md:168).  One persistent launch covers every table and every sample.
//
// Mapping (output-first): warp-task s owns the contiguous bags [seg_bag[s], seg_bag[s+1])
// -> adjacent warps own adjacent output addresses, and out[b, t*D + c] == out[g*D + c] for g = b*T + t, so
// the concatenated [B, T*D] block is written once, in place, with no per-table intermediates.
//
// A row is NV = D*sizeof(elt)/16 128-bit vectors; W = pow2ceil(NV) lanes hold one row (lane sl < NV loads
// vector sl), P = 32/W sub-warps per warp.  Three warp-uniform shapes per segment:
//   one-hot   (every bag in the segment has length 1): pure row copy, P*U rows in flight per warp (Alg. 1)
//   sub-warp  (short bags): sub-warp q pools bags g_lo+q, g_lo+q+P, ... with U loads in flight per lane
//   warp      (long bags) : all P sub-warps stride the entries of one bag, U loads in flight per lane, then
//                           log2(P) __shfl_xor steps combine the partial sums
// fp32 accumulation in registers; one RNE cast at the store (fp16/bf16 tables).
#pragma once

#include "dpi_internal.cuh"

namespace dpi {

// ---- memory helpers ----------------------------------------------------------------------------------
__device__ __forceinline__ uint4 ld_row16(const void* p, int no_alloc) {
    uint4 r;
    if (no_alloc) {
        asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
            : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    } else {
        asm("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];"
            : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    }
    return r;
}
__device__ __forceinline__ void st_out16(void* p, const uint4& v) {
    // streaming store: the output block is consumed by the next layer, not re-read here
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- per-dtype arithmetic ----------------------------------------------------------------------------
struct F32Traits {
    static constexpr int kAcc = 4;
    __device__ static __forceinline__ void add(float (&acc)[4], const uint4& v) {
        acc[0] += __uint_as_float(v.x); acc[1] += __uint_as_float(v.y);
        acc[2] += __uint_as_float(v.z); acc[3] += __uint_as_float(v.w);
    }
    __device__ static __forceinline__ uint4 pack(const float (&acc)[4]) {
        return make_uint4(__float_as_uint(acc[0]), __float_as_uint(acc[1]), __float_as_uint(acc[2]),
                          __float_as_uint(acc[3]));
    }
};
struct F16Traits {
    static constexpr int kAcc = 8;
    __device__ static __forceinline__ void add(float (&acc)[8], const uint4& v) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
            acc[2 * i] += f.x; acc[2 * i + 1] += f.y;
        }
    }
    __device__ static __forceinline__ uint4 pack(const float (&acc)[8]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __half2 h = __floats2half2_rn(acc[2 * i], acc[2 * i + 1]);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};
struct BF16Traits {
    static constexpr int kAcc = 8;
    __device__ static __forceinline__ void add(float (&acc)[8], const uint4& v) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {  // bf16 -> fp32 is a 16-bit shift
            acc[2 * i] += __uint_as_float(w[i] << 16);
            acc[2 * i + 1] += __uint_as_float(w[i] & 0xffff0000u);
        }
    }
    __device__ static __forceinline__ uint4 pack(const float (&acc)[8]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(acc[2 * i], acc[2 * i + 1]);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

template <int N>
__device__ __forceinline__ void scale_mean(float (&acc)[N], int len) {
    const float L = static_cast<float>(len);
#pragma unroll
    for (int i = 0; i < N; ++i) acc[i] = __fdiv_rn(acc[i], L);
}

constexpr int kLookupMaxThreads = 512;

template <class Tr, int W, int U>
__global__ void __launch_bounds__(kLookupMaxThreads) lookup_kernel(const LookupArgs a) {
    constexpr int P = 32 / W;
    constexpr int kAcc = Tr::kAcc;
    const int lane = threadIdx.x & 31;
    const int sub = lane / W;
    const int sl = lane % W;
    const bool vec_ok = static_cast<uint32_t>(sl) < a.nvec;
    const uint32_t warps_per_cta = blockDim.x >> 5;
    const uint32_t n_warps = gridDim.x * warps_per_cta;
    const uint32_t warp_id = blockIdx.x * warps_per_cta + (threadIdx.x >> 5);
    const size_t row_bytes = static_cast<size_t>(a.nvec) * 16;
    const char* const out_lane = static_cast<char*>(a.out) + sl * 16;
    const int no_alloc = a.row_no_alloc;

    griddep_wait();  // PDL: the planner's writes are visible past this point (no-op otherwise)
    const uint32_t S = static_cast<uint32_t>(a.meta[META_S]);

    for (uint32_t s = warp_id; s < S; s += n_warps) {
        const uint32_t g_lo = __ldg(a.seg_bag + s), g_hi = __ldg(a.seg_bag + s + 1);
        if (g_lo >= g_hi) continue;  // a long bag spanning several quanta leaves empty tasks behind it
        const uint32_t nb = g_hi - g_lo;
        const int e_lo = __ldg(a.offsets + g_lo), e_hi = __ldg(a.offsets + g_hi);
        const uint32_t ne = static_cast<uint32_t>(e_hi - e_lo);

        if (ne == nb && a.mode != 2) {
            // ---------------- one-hot segment: Alg. 1, a pure row copy -------------------------------
            // (a segment with ne == nb could also mix empty and longer bags; verify per batch below)
            bool all_one = true;
            for (uint32_t i0 = 0; i0 < nb; i0 += 32) {
                const uint32_t i = i0 + lane;
                if (i < nb) all_one &= (__ldg(a.offsets + g_lo + i + 1) - __ldg(a.offsets + g_lo + i)) == 1;
            }
            if (__all_sync(0xffffffffu, all_one)) {
                for (uint32_t i0 = 0; i0 < nb; i0 += P * U) {
                    uint4 v[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        v[u] = make_uint4(0, 0, 0, 0);
                        if (i < nb && vec_ok) {
                            const uint32_t g = g_lo + i;
                            const char* tab = static_cast<const char*>(a.tables[g % a.T]) + sl * 16;
                            const int r = __ldg(a.indices + e_lo + i);
                            v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, no_alloc);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        if (i < nb && vec_ok)
                            st_out16(const_cast<char*>(out_lane) + static_cast<size_t>(g_lo + i) * row_bytes, v[u]);
                    }
                }
                continue;
            }
        }

        const bool warp_per_bag = (P > 1) && (a.mode == 2 || (a.mode == 0 && (nb < P || ne >= 2u * P * nb)));
        if (!warp_per_bag) {
            // ---------------- sub-warp per bag --------------------------------------------------------
            for (uint32_t g0 = g_lo; g0 < g_hi; g0 += P) {
                const uint32_t g = g0 + sub;
                const bool active = g < g_hi;
                int lo = 0, hi = 0;
                const char* tab = nullptr;
                uint32_t t = 0;
                if (active) {
                    lo = __ldg(a.offsets + g);
                    hi = __ldg(a.offsets + g + 1);
                    t = g % a.T;
                    tab = static_cast<const char*>(a.tables[t]) + sl * 16;
                }
                float acc[kAcc];
#pragma unroll
                for (int i = 0; i < kAcc; ++i) acc[i] = 0.f;
                for (int j = lo; j < hi; j += U) {
                    uint4 v[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        v[u] = make_uint4(0, 0, 0, 0);
                        if (j + u < hi && vec_ok) {
                            const int r = __ldg(a.indices + j + u);
                            v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, no_alloc);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) Tr::add(acc, v[u]);
                }
                if (active && vec_ok) {
                    if (((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                    st_out16(const_cast<char*>(out_lane) + static_cast<size_t>(g) * row_bytes, Tr::pack(acc));
                }
            }
        } else {
            // ---------------- whole warp per bag ------------------------------------------------------
            for (uint32_t g = g_lo; g < g_hi; ++g) {
                const int lo = __ldg(a.offsets + g), hi = __ldg(a.offsets + g + 1);
                const uint32_t t = g % a.T;
                const char* tab = static_cast<const char*>(a.tables[t]) + sl * 16;
                float acc[kAcc];
#pragma unroll
                for (int i = 0; i < kAcc; ++i) acc[i] = 0.f;
                for (int j = lo; j < hi; j += P * U) {
                    uint4 v[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int e = j + u * P + sub;
                        v[u] = make_uint4(0, 0, 0, 0);
                        if (e < hi && vec_ok) {
                            const int r = __ldg(a.indices + e);
                            v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, no_alloc);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) Tr::add(acc, v[u]);
                }
#pragma unroll
                for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                    for (int i = 0; i < kAcc; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], d);
                }
                if (sub == 0 && vec_ok) {
                    if (((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                    st_out16(const_cast<char*>(out_lane) + static_cast<size_t>(g) * row_bytes, Tr::pack(acc));
                }
            }
        }
    }
}

// ---- host-side dispatch (one translation unit per dtype keeps nvcc parallel) ------------------------------
template <class Tr, int W, int U>
cudaError_t launch_one(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(static_cast<unsigned>(l.grid));
    cfg.blockDim = dim3(static_cast<unsigned>(l.block_threads));
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = l.pdl ? 1 : 0;
    count_launch();
    return cudaLaunchKernelEx(&cfg, lookup_kernel<Tr, W, U>, a);
}

template <class Tr, int W, int U>
int occupancy_one(int block_threads) {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, lookup_kernel<Tr, W, U>, block_threads, 0) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

#define DPI_FOR_EACH_U(M, W) M(W, 2) M(W, 4) M(W, 8) M(W, 16)
#define DPI_FOR_EACH_WU(M) \
    DPI_FOR_EACH_U(M, 1) DPI_FOR_EACH_U(M, 2) DPI_FOR_EACH_U(M, 4) DPI_FOR_EACH_U(M, 8) DPI_FOR_EACH_U(M, 16) \
    DPI_FOR_EACH_U(M, 32)

// Each lookup_<dtype>.cu defines DPI_TRAITS / DPI_SUFFIX and includes lookup_dispatch.inc.

}  // namespace dpi
