// nongemm_device.cuh -- device-side pieces of the fused non-GEMM operators that more than one translation unit uses
// (nongemm_kernels.cu: fm_kernel; forward_fused.cu: the FM epilogue of dpi_forward_fm). SURVEY.md 8(f) NEXT-4.
#pragma once

#include "dpi_internal.cuh"

namespace dpi {

// ---- 16-byte vector <-> fp32 lanes -----------------------------------------------------------------------------
template <int DT> struct Elt;
template <> struct Elt<DPI_F32> {
    static constexpr int kPerVec = 4;
    __device__ static __forceinline__ void unpack(const uint4& v, float (&f)[4]) {
        f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
    }
    __device__ static __forceinline__ uint4 pack(const float (&f)[4]) {
        return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
    }
};
template <> struct Elt<DPI_F16> {
    static constexpr int kPerVec = 8;
    __device__ static __forceinline__ void unpack(const uint4& v, float (&f)[8]) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 p = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
            f[2 * i] = p.x; f[2 * i + 1] = p.y;
        }
    }
    __device__ static __forceinline__ uint4 pack(const float (&f)[8]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __half2 h = __floats2half2_rn(f[2 * i], f[2 * i + 1]);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};
template <> struct Elt<DPI_BF16> {
    static constexpr int kPerVec = 8;
    __device__ static __forceinline__ void unpack(const uint4& v, float (&f)[8]) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            f[2 * i] = __uint_as_float(w[i] << 16);
            f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
        }
    }
    __device__ static __forceinline__ uint4 pack(const float (&f)[8]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

// read once: do not keep it in L1. Coherent (no .nc) because the element-wise operators may run in place.
__device__ __forceinline__ uint4 ld_stream16(const void* p, bool pred) {
    uint4 r = make_uint4(0u, 0u, 0u, 0u);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
        "@p ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];\n\t}"
        : "+r"(r.x), "+r"(r.y), "+r"(r.z), "+r"(r.w) : "l"(p), "r"(static_cast<int>(pred)) : "memory");
    return r;
}
__device__ __forceinline__ void st_stream16(void* p, const uint4& v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// ---- FM second-order term ---------------------------------------------------------------------------------------
// Same lane mapping as the lookup: a field's D elements are NV 16-byte vectors, W = pow2ceil(NV) lanes hold one field
// (lane sl < NV loads vector sl), the P = 32/W sub-warps of a warp walk fields sub, sub+P, ... of ONE sample, so a
// warp-wide load covers P consecutive fields = a contiguous piece of the sample's row (output-first: the threads of a
// warp share a sample). Each lane keeps sum and sum-of-squares of its columns over its fields; the
// sub-warps are combined with log2(P) xor-shuffle steps; sub-warp 0 forms 1/2 (s^2 - q) per column, stores v and
// reduces over the columns for y.
struct FmArgs {
    const char* x;
    float* y;
    float* v;
    uint64_t x_pitch;  // bytes between rows
    uint32_t B, T, D, nvec;
};

// One sample's FM term, computed by one warp (all 32 lanes call it): shared by fm_kernel and by the fused forward kernel
// (forward_fused.cu), which runs it on the rows its own CTA has just pooled -- same arithmetic, same order, same result.
template <int DT, int W, int U>
__device__ __forceinline__ void fm_one_sample(const FmArgs& a, uint32_t b, int lane) {
    constexpr int P = 32 / W;
    constexpr int E = Elt<DT>::kPerVec;
    const int sub = lane / W, sl = lane % W;
    const bool vec_ok = static_cast<uint32_t>(sl) < a.nvec;
    const uint32_t field_bytes = a.nvec * 16;
    const char* row = a.x + static_cast<size_t>(b) * a.x_pitch + sl * 16;
    float s[E], q[E];
#pragma unroll
    for (int i = 0; i < E; ++i) { s[i] = 0.f; q[i] = 0.f; }
    for (uint32_t t0 = 0; t0 < a.T; t0 += P * U) {
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t t = t0 + u * P + sub;
            v[u] = ld_stream16(row + static_cast<size_t>(t) * field_bytes, vec_ok && t < a.T);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {  // a predicated-off load left zeros: they add nothing to s or q
            float f[E];
            Elt<DT>::unpack(v[u], f);
#pragma unroll
            for (int i = 0; i < E; ++i) { s[i] += f[i]; q[i] = fmaf(f[i], f[i], q[i]); }
        }
    }
#pragma unroll
    for (int d = W; d < 32; d <<= 1) {
#pragma unroll
        for (int i = 0; i < E; ++i) {
            s[i] += __shfl_xor_sync(0xffffffffu, s[i], d);
            q[i] += __shfl_xor_sync(0xffffffffu, q[i], d);
        }
    }
    float part = 0.f;
    float vc[E];
#pragma unroll
    for (int i = 0; i < E; ++i) {
        vc[i] = 0.5f * fmaf(s[i], s[i], -q[i]);
        part += vc[i];
    }
    if (!vec_ok) part = 0.f;
    if (a.v && sub == 0 && vec_ok) {
        float4* pv = reinterpret_cast<float4*>(a.v + static_cast<size_t>(b) * a.D + sl * E);
#pragma unroll
        for (int i = 0; i < E / 4; ++i) pv[i] = make_float4(vc[4 * i], vc[4 * i + 1], vc[4 * i + 2], vc[4 * i + 3]);
    }
    if (a.y) {
#pragma unroll
        for (int d = 1; d < W; d <<= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
        if (lane == 0) a.y[b] = part;
    }
}

}  // namespace dpi
