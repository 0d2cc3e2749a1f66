// synth_fill.cu -- libdpi_synth.so: device-side fill of synthetic embedding tables (bench/tests only).
//
// NOT part of the method: this is the input generator of workloads.py restated for the device, so that an
// 82 GB table set can be created in place (the host cannot mirror it). Same counter-based recipe:
//   h = fmix64(key + i*GAMMA),  i = r*D + c,   x = float(h >> 40) * 2^-24,   v = (x - 0.5f) * 0.1f
// then one RNE cast to the table dtype. tests/test_gpu_parity.py::test_synth_fill_matches_host_generator checks host/device equality bit for bit.
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ unsigned long long fmix64(unsigned long long z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ float value_at(unsigned long long key, unsigned long long i) {
    const unsigned long long h = fmix64(key + i * 0x9E3779B97F4A7C15ull);
    const float x = __uint2float_rn(static_cast<unsigned int>(h >> 40)) * 5.9604644775390625e-08f;  // 2^-24, exact
    return __fmul_rn(__fsub_rn(x, 0.5f), 0.1f);
}

// one thread = 16 bytes of output
template <int DT>
__global__ void __launch_bounds__(256) fill_kernel(void* __restrict__ dst, unsigned long long n_elems,
                                                   unsigned long long key) {
    constexpr int kPer = DT == 0 ? 4 : 8;
    const unsigned long long n_vec = n_elems / kPer;
    for (unsigned long long v = blockIdx.x * static_cast<unsigned long long>(blockDim.x) + threadIdx.x; v < n_vec;
         v += static_cast<unsigned long long>(gridDim.x) * blockDim.x) {
        float f[kPer];
#pragma unroll
        for (int k = 0; k < kPer; ++k) f[k] = value_at(key, v * kPer + k);
        uint4 o;
        if (DT == 0) {
            o = make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
        } else {
            uint32_t w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (DT == 1) {
                    const __half2 h = __floats2half2_rn(f[2 * k], f[2 * k + 1]);
                    w[k] = *reinterpret_cast<const uint32_t*>(&h);
                } else {
                    const __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * k], f[2 * k + 1]);
                    w[k] = *reinterpret_cast<const uint32_t*>(&h);
                }
            }
            o = make_uint4(w[0], w[1], w[2], w[3]);
        }
        reinterpret_cast<uint4*>(dst)[v] = o;
    }
}

}  // namespace

// dst: device pointer, 16-byte aligned, n_elems = rows*D elements with (n_elems * sizeof(elt)) % 16 == 0.
// dtype: 0 f32, 1 f16, 2 bf16.  Returns the cudaError_t value (0 = success). Asynchronous on `stream`.
extern "C" int dpi_synth_fill_table(void* dst, uint64_t n_elems, int dtype, uint64_t key, void* stream) {
    if (!dst || dtype < 0 || dtype > 2 || (reinterpret_cast<uintptr_t>(dst) & 15u)) return (int)cudaErrorInvalidValue;
    const int per = dtype == 0 ? 4 : 8;
    if (n_elems % per) return (int)cudaErrorInvalidValue;
    if (n_elems == 0) return 0;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const unsigned long long n_vec = n_elems / per;
    const unsigned int blocks = static_cast<unsigned int>(n_vec / 256 + 1 < 148ull * 16 ? n_vec / 256 + 1 : 148ull * 16);
    switch (dtype) {
        case 0: fill_kernel<0><<<blocks, 256, 0, s>>>(dst, n_elems, key); break;
        case 1: fill_kernel<1><<<blocks, 256, 0, s>>>(dst, n_elems, key); break;
        default: fill_kernel<2><<<blocks, 256, 0, s>>>(dst, n_elems, key); break;
    }
    return (int)cudaGetLastError();
}

// ---- gather ceiling probe (bench context, not part of the method) -----------------------------------------------------
// What can this box sustain for independent reads of whole `row_bytes`-byte rows at random (or consecutive) positions of
// a `span_rows`-row buffer, with no indices to fetch, no pooling and no output? That is the ceiling the fused lookup's
// row stream can be compared with (SURVEY.md 8(d) "random-access ceiling"): W = row_bytes/16 lanes read one row with one
// 128-bit load each, U rows in flight per lane, row ids from a counter hash (random) or the counter itself (sequential).
namespace {
template <int U>
__global__ void __launch_bounds__(256) row_read_probe_kernel(const char* __restrict__ base, unsigned long long span_rows,
                                                             unsigned int row_bytes, unsigned long long n_rows,
                                                             unsigned long long key, int random, unsigned int* sink) {
    const unsigned int W = row_bytes / 16;                     // lanes per row (power of two <= 32)
    const unsigned int lane = threadIdx.x & 31, sl = lane % W, sub = lane / W, P = 32 / W;
    const unsigned long long warp = (blockIdx.x * static_cast<unsigned long long>(blockDim.x) + threadIdx.x) >> 5;
    const unsigned long long n_warps = (gridDim.x * static_cast<unsigned long long>(blockDim.x)) >> 5;
    unsigned int acc = 0;
    for (unsigned long long i0 = warp * (P * U); i0 < n_rows; i0 += n_warps * (P * U)) {
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const unsigned long long i = i0 + u * P + sub;
            // hash -> [0, span_rows) by multiply-high (a 64-bit modulo costs more than the load it feeds)
            const unsigned long long r = random ? __umul64hi(fmix64(key + i * 0x9E3779B97F4A7C15ull), span_rows)
                                                : (i < span_rows ? i : i - span_rows * (i / span_rows));
            v[u] = __ldg(reinterpret_cast<const uint4*>(base + r * row_bytes + sl * 16));
        }
#pragma unroll
        for (int u = 0; u < U; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
    }
    if (acc == 0x9E3779B9u) *sink = acc;                       // keeps the loads alive; practically never taken
}
}  // namespace

// Reads n_rows rows of row_bytes (16..512, power of two) from base[span_rows * row_bytes]. unroll in {2, 4, 8}.
extern "C" int dpi_synth_row_read_probe(const void* base, uint64_t span_rows, uint32_t row_bytes, uint64_t n_rows,
                                        uint64_t key, int random, int unroll, int ctas_per_sm, void* sink_dev, void* stream) {
    if (!base || !sink_dev || span_rows == 0 || row_bytes < 16 || row_bytes > 512 || (row_bytes & (row_bytes - 1)))
        return (int)cudaErrorInvalidValue;
    int dev = 0, sms = 148;
    (void)cudaGetDevice(&dev);
    (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const unsigned int blocks = static_cast<unsigned int>(sms * (ctas_per_sm > 0 ? ctas_per_sm : 8));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const char* b = static_cast<const char*>(base);
    unsigned int* sk = static_cast<unsigned int*>(sink_dev);
    switch (unroll) {
        case 2: row_read_probe_kernel<2><<<blocks, 256, 0, s>>>(b, span_rows, row_bytes, n_rows, key, random, sk); break;
        case 8: row_read_probe_kernel<8><<<blocks, 256, 0, s>>>(b, span_rows, row_bytes, n_rows, key, random, sk); break;
        default: row_read_probe_kernel<4><<<blocks, 256, 0, s>>>(b, span_rows, row_bytes, n_rows, key, random, sk); break;
    }
    return (int)cudaGetLastError();
}

// Test helper: copy n_words 32-bit words between two raw device addresses (how the tests read the borrowed pointers of
// dpi_plan_device_views into a tensor); synchronous.
extern "C" int dpi_synth_copy_words(void* dst_dev, const void* src_dev, uint64_t n_words) {
    if (!dst_dev || !src_dev) return (int)cudaErrorInvalidValue;
    return (int)cudaMemcpy(dst_dev, src_dev, n_words * 4, cudaMemcpyDeviceToDevice);
}
