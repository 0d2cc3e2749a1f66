// nongemm_kernels.cu -- SURVEY.md 8(f) NEXT-4: the fused non-GEMM operators that consume X_embed
// ("we combine all neighbouring non-GEMM operators into a single operator ... traverse the output
// matrix element by element ... data reads and writes are contiguous in memory").  Boundary: include/dpi_nongemm.h.
//
//   fm_kernel            DeepFM FM second-order term: square, reduce-sum over fields, subtract, halve, reduce-sum over
//                        the embedding dim -- five framework operators, one pass over X_embed, one warp per sample.
//   cross_combine_kernel DCNv2 cross layer minus its GEMM: out = x0 * (u + bias) + xl.
//   bias_act_kernel      MLP layer minus its GEMM: out = act(u + bias).
// All three are streaming, HBM/L2-bound: 128-bit coalesced loads, fp32 arithmetic, one RNE cast at the store. No
// tensor cores (no contraction here; the GEMMs between these operators are the caller's cuBLAS calls).
#include <algorithm>

#include "dpi_internal.cuh"
#include "nongemm_device.cuh"
#include "../../include/dpi_nongemm.h"

namespace dpi {
namespace {

template <int DT, int W, int U>
__global__ void __launch_bounds__(256) fm_kernel(const FmArgs a) {
    const int lane = threadIdx.x & 31;
    const uint32_t warps_per_cta = blockDim.x >> 5;
    const uint32_t n_warps = gridDim.x * warps_per_cta;
    for (uint32_t b = blockIdx.x * warps_per_cta + (threadIdx.x >> 5); b < a.B; b += n_warps) fm_one_sample<DT, W, U>(a, b, lane);
}

// ---- element-wise operators ---------------------------------------------------------------------------------------
// Thread (tx, ty) of a CTA owns column vector blockIdx.x*CX + tx and rows blockIdx.y*RY + ty, +gridDim.y*RY, ...:
// the bias of its columns is loaded once, rows are walked U at a time so U x (inputs) 16-byte loads are in flight.
struct EwArgs {
    const char* x0;   // cross only
    const char* xl;   // cross only
    const char* u;
    const float* bias;
    char* out;
    uint32_t B, vpr;  // rows, 16-byte vectors per row
    int act;
};

template <int E>
__device__ __forceinline__ void load_bias(const float* bias, uint32_t col_vec, bool ok, float (&bv)[E]) {
#pragma unroll
    for (int i = 0; i < E; ++i) bv[i] = 0.f;
    if (bias && ok) {
        const float4* p = reinterpret_cast<const float4*>(bias + static_cast<size_t>(col_vec) * E);
#pragma unroll
        for (int i = 0; i < E / 4; ++i) {
            const float4 b4 = __ldg(p + i);
            bv[4 * i] = b4.x; bv[4 * i + 1] = b4.y; bv[4 * i + 2] = b4.z; bv[4 * i + 3] = b4.w;
        }
    }
}

template <int DT, int U>
__global__ void __launch_bounds__(256) cross_combine_kernel(const EwArgs a, const uint32_t cx_log2) {
    constexpr int E = Elt<DT>::kPerVec;
    const uint32_t cx = 1u << cx_log2, ry = blockDim.x >> cx_log2;
    const uint32_t tx = threadIdx.x & (cx - 1), ty = threadIdx.x >> cx_log2;
    const uint32_t c = blockIdx.x * cx + tx;
    const bool col_ok = c < a.vpr;
    float bv[E];
    load_bias<E>(a.bias, c, col_ok, bv);
    const uint32_t r_step = gridDim.y * ry;
    for (uint32_t r0 = blockIdx.y * ry + ty; r0 < a.B; r0 += r_step * U) {
        uint4 vx0[U], vxl[U], vu[U];
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const uint32_t r = r0 + k * r_step;
            const bool ok = col_ok && r < a.B;
            const size_t off = (static_cast<size_t>(r) * a.vpr + c) * 16;
            vx0[k] = ld_stream16(a.x0 + off, ok);
            vu[k] = ld_stream16(a.u + off, ok);
            vxl[k] = ld_stream16(a.xl + off, ok);
        }
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const uint32_t r = r0 + k * r_step;
            if (col_ok && r < a.B) {
                float f0[E], fl[E], fu[E], o[E];
                Elt<DT>::unpack(vx0[k], f0);
                Elt<DT>::unpack(vxl[k], fl);
                Elt<DT>::unpack(vu[k], fu);
#pragma unroll
                for (int i = 0; i < E; ++i) o[i] = fmaf(f0[i], fu[i] + bv[i], fl[i]);
                st_stream16(a.out + (static_cast<size_t>(r) * a.vpr + c) * 16, Elt<DT>::pack(o));
            }
        }
    }
}

template <int DT, int U>
__global__ void __launch_bounds__(256) bias_act_kernel(const EwArgs a, const uint32_t cx_log2) {
    constexpr int E = Elt<DT>::kPerVec;
    const uint32_t cx = 1u << cx_log2, ry = blockDim.x >> cx_log2;
    const uint32_t tx = threadIdx.x & (cx - 1), ty = threadIdx.x >> cx_log2;
    const uint32_t c = blockIdx.x * cx + tx;
    const bool col_ok = c < a.vpr;
    float bv[E];
    load_bias<E>(a.bias, c, col_ok, bv);
    const uint32_t r_step = gridDim.y * ry;
    for (uint32_t r0 = blockIdx.y * ry + ty; r0 < a.B; r0 += r_step * U) {
        uint4 vu[U];
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const uint32_t r = r0 + k * r_step;
            vu[k] = ld_stream16(a.u + (static_cast<size_t>(r) * a.vpr + c) * 16, col_ok && r < a.B);
        }
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const uint32_t r = r0 + k * r_step;
            if (col_ok && r < a.B) {
                float fu[E], o[E];
                Elt<DT>::unpack(vu[k], fu);
#pragma unroll
                for (int i = 0; i < E; ++i) {
                    float s = fu[i] + bv[i];
                    if (a.act == DPI_ACT_RELU) s = fmaxf(s, 0.f);
                    else if (a.act == DPI_ACT_SIGMOID) s = __fdividef(1.f, 1.f + __expf(-s));  // ex2.approx + rcp.approx: a few fp32 ulps
                    o[i] = s;
                }
                st_stream16(a.out + (static_cast<size_t>(r) * a.vpr + c) * 16, Elt<DT>::pack(o));
            }
        }
    }
}

// ---- DeepFM first-order (logistic regression) term -------------------------------------------------------------------
// One warp per sample; lane l owns bags t = l, l + 32, ... of the sample (their offsets are consecutive words, their
// index entries consecutive runs), gathers the scalar weights of its bags and the warp tree-reduces. T lookups, the
// T-way reduce-sum and the bias add of the framework graph in one launch.
struct LrArgs {
    const float* const* w;
    const int32_t* indices;
    const int32_t* offsets;  // NULL: one-hot
    float* y;
    float bias;
    uint32_t B, T;
    int accumulate;
};

__global__ void __launch_bounds__(256) lr_kernel(const LrArgs a) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t warps_per_cta = blockDim.x >> 5;
    const uint32_t n_warps = gridDim.x * warps_per_cta;
    for (uint32_t b = blockIdx.x * warps_per_cta + (threadIdx.x >> 5); b < a.B; b += n_warps) {
        const size_t g0 = static_cast<size_t>(b) * a.T;
        float acc = 0.f;
        for (uint32_t t = lane; t < a.T; t += 32) {
            const float* wt = reinterpret_cast<const float*>(__ldg(reinterpret_cast<const unsigned long long*>(a.w) + t));
            if (a.offsets) {
                const int lo = __ldg(a.offsets + g0 + t), hi = __ldg(a.offsets + g0 + t + 1);
                for (int j = lo; j < hi; ++j) acc += __ldg(wt + static_cast<uint32_t>(__ldg(a.indices + j)));
            } else {
                acc += __ldg(wt + static_cast<uint32_t>(__ldg(a.indices + g0 + t)));
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        if (lane == 0) a.y[b] = (a.accumulate ? a.y[b] : 0.f) + (a.bias + acc);
    }
}

int pow2ceil_i(int x) { int p = 1; while (p < x) p <<= 1; return p; }
int log2_i(int x) { int l = 0; while ((1 << l) < x) ++l; return l; }

int sm_count() {
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            (void)cudaGetLastError();
            n = 148;
        }
    }
    return n;
}

template <int DT>
cudaError_t launch_fm_dt(const FmArgs& a, int W, cudaStream_t st) {
    const int warps_per_cta = 8;
    const long long want = (static_cast<long long>(a.B) + warps_per_cta - 1) / warps_per_cta;
    const long long cap = static_cast<long long>(sm_count()) * 8 * 4;  // a few waves; warps stride over samples
    const unsigned grid = static_cast<unsigned>(want < cap ? (want < 1 ? 1 : want) : cap);
    count_launch();
    switch (W) {
#define DPI_FM_CASE(w) case w: fm_kernel<DT, w, 4><<<grid, 256, 0, st>>>(a); break;
        DPI_FM_CASE(1) DPI_FM_CASE(2) DPI_FM_CASE(4) DPI_FM_CASE(8) DPI_FM_CASE(16) DPI_FM_CASE(32)
#undef DPI_FM_CASE
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

struct EwGrid { dim3 grid; uint32_t cx_log2; };
EwGrid ew_grid(uint32_t B, uint32_t vpr, int U) {
    const int cx = std::min(256, pow2ceil_i(static_cast<int>(vpr)));
    const int ry = 256 / cx;
    EwGrid g;
    g.cx_log2 = static_cast<uint32_t>(log2_i(cx));
    const unsigned gx = (vpr + cx - 1) / cx;
    const long long rows_blocks = (static_cast<long long>(B) + static_cast<long long>(ry) * U - 1) / (static_cast<long long>(ry) * U);
    long long gy = static_cast<long long>(sm_count()) * 8 / gx;   // ~8 CTAs per SM in total
    if (gy < 1) gy = 1;
    if (gy > rows_blocks) gy = rows_blocks < 1 ? 1 : rows_blocks;
    if (gy > 65535) gy = 65535;
    g.grid = dim3(gx, static_cast<unsigned>(gy));
    return g;
}

}  // namespace

cudaError_t launch_fm(const void* x, int dtype, uint32_t B, uint32_t T, uint32_t D, uint64_t x_pitch_bytes, float* y,
                      float* v, cudaStream_t st) {
    const uint32_t elt = dtype == DPI_F32 ? 4u : 2u;
    FmArgs a{static_cast<const char*>(x), y, v, x_pitch_bytes, B, T, D, D * elt / 16u};
    const int W = pow2ceil_i(static_cast<int>(a.nvec));
    switch (dtype) {
        case DPI_F32: return launch_fm_dt<DPI_F32>(a, W, st);
        case DPI_F16: return launch_fm_dt<DPI_F16>(a, W, st);
        case DPI_BF16: return launch_fm_dt<DPI_BF16>(a, W, st);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_lr(const void* const* w, const int32_t* indices, const int32_t* offsets, uint32_t B, uint32_t T, float bias,
                      float* y, int accumulate, cudaStream_t st) {
    LrArgs a{reinterpret_cast<const float* const*>(w), indices, offsets, y, bias, B, T, accumulate};
    const long long want = (static_cast<long long>(B) + 7) / 8;
    const long long cap = static_cast<long long>(sm_count()) * 8 * 4;
    const unsigned grid = static_cast<unsigned>(want < cap ? (want < 1 ? 1 : want) : cap);
    count_launch();
    lr_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_cross_combine(const void* x0, const void* xl, const void* u, const float* bias, void* out, int dtype,
                                 uint32_t B, uint32_t F, cudaStream_t st) {
    const uint32_t elt = dtype == DPI_F32 ? 4u : 2u;
    EwArgs a{static_cast<const char*>(x0), static_cast<const char*>(xl), static_cast<const char*>(u), bias,
             static_cast<char*>(out), B, F * elt / 16u, 0};
    constexpr int U = 4;
    const EwGrid g = ew_grid(B, a.vpr, U);
    count_launch();
    switch (dtype) {
        case DPI_F32: cross_combine_kernel<DPI_F32, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        case DPI_F16: cross_combine_kernel<DPI_F16, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        case DPI_BF16: cross_combine_kernel<DPI_BF16, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_bias_act(const void* u, const float* bias, void* out, int dtype, uint32_t B, uint32_t F, int act,
                            cudaStream_t st) {
    const uint32_t elt = dtype == DPI_F32 ? 4u : 2u;
    EwArgs a{nullptr, nullptr, static_cast<const char*>(u), bias, static_cast<char*>(out), B, F * elt / 16u, act};
    constexpr int U = 8;
    const EwGrid g = ew_grid(B, a.vpr, U);
    count_launch();
    switch (dtype) {
        case DPI_F32: bias_act_kernel<DPI_F32, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        case DPI_F16: bias_act_kernel<DPI_F16, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        case DPI_BF16: bias_act_kernel<DPI_BF16, U><<<g.grid, 256, 0, st>>>(a, g.cx_log2); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace dpi
