// plan64_kernels.cu -- steps a1 + a2 with 64-bit offsets (SURVEY.md 8(f) NEXT-2 "int64 indices/offsets"; ids reach the model
// as 64-bit integers; DESIGN.md section 3 / 11.2 V6): the same plan definition as plan_kernels.cu, only
// offsets[], seg_off[], C and N are 64-bit, so a batch may hold N >= 2^31 index entries (G < 2^31 still).
// An interface variant, not the path of BASELINE.json's configs: kept simple -- TWO stream-ordered launches instead of the
// single-launch chained scan (no status records, no epoch): (1) every chunk's {sum len, sum cost, min, max}; (2) every CTA
// adds up the aggregates of the chunks before it (<= kMaxChunks values) and scans its chunk tile by tile, writing
// offsets64[g], the segment records {seg_bag[s], low 32 bits of seg_off[s]} + seg_off64[s], and meta. Integer work only;
// bit-exact against oracle/dpi_oracle.c::oracle_plan64.
#include "dpi_internal.cuh"

namespace dpi {
namespace {

struct Agg64 {
    unsigned long long len, cost;
    uint32_t lo, hi, pad0, pad1;
};
static_assert(sizeof(Agg64) == 32, "aggregate record layout");

__device__ __forceinline__ uint32_t load_len(const Plan64Args& a, uint32_t g) { return g < a.G ? static_cast<uint32_t>(__ldg(a.len + g)) : 0u; }

__global__ void __launch_bounds__(kScanThreads) plan64_aggregate_kernel(const Plan64Args a) {
    __shared__ unsigned long long s_len[kScanThreads / 32], s_cost[kScanThreads / 32];
    __shared__ uint32_t s_lo[kScanThreads / 32], s_hi[kScanThreads / 32];
    const uint32_t chunk = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned long long g_lo = static_cast<unsigned long long>(chunk) * a.tiles_per_chunk * kScanTile;
    const unsigned long long g_hi = min(static_cast<unsigned long long>(a.G), g_lo + static_cast<unsigned long long>(a.tiles_per_chunk) * kScanTile);
    unsigned long long t_len = 0, t_cost = 0;
    uint32_t lo = 0xffffffffu, hi = 0u;
    for (unsigned long long g = g_lo + threadIdx.x; g < g_hi; g += kScanThreads) {
        const uint32_t l = static_cast<uint32_t>(__ldg(a.len + g));
        t_len += l;
        t_cost += max(l, 1u);
        lo = min(lo, l);
        hi = max(hi, l);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        t_len += __shfl_xor_sync(0xffffffffu, t_len, d);
        t_cost += __shfl_xor_sync(0xffffffffu, t_cost, d);
    }
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    if (lane == 0) { s_len[warp] = t_len; s_cost[warp] = t_cost; s_lo[warp] = lo; s_hi[warp] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        Agg64 r{0, 0, 0xffffffffu, 0u, 0u, 0u};
        for (int w = 0; w < kScanThreads / 32; ++w) {
            r.len += s_len[w]; r.cost += s_cost[w];
            r.lo = min(r.lo, s_lo[w]); r.hi = max(r.hi, s_hi[w]);
        }
        reinterpret_cast<Agg64*>(a.agg)[chunk] = r;
    }
}

__global__ void __launch_bounds__(kScanThreads) plan64_scan_kernel(const Plan64Args a) {
    __shared__ unsigned long long s_wlen[kScanThreads / 32], s_wcost[kScanThreads / 32];
    __shared__ unsigned long long s_pre[2];
    const uint32_t chunk = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const Agg64* agg = reinterpret_cast<const Agg64*>(a.agg);
    if (warp == 0) {   // prefix of this chunk = sum of the aggregates before it; the last chunk also reduces min / max
        unsigned long long pl = 0, pc = 0;
        uint32_t lo = 0xffffffffu, hi = 0u;
        const bool last = chunk + 1 == a.num_chunks;
        for (uint32_t c = lane; c < (last ? a.num_chunks : chunk); c += 32) {
            const Agg64 r = agg[c];
            if (c < chunk) { pl += r.len; pc += r.cost; }
            lo = min(lo, r.lo); hi = max(hi, r.hi);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            pl += __shfl_xor_sync(0xffffffffu, pl, d);
            pc += __shfl_xor_sync(0xffffffffu, pc, d);
        }
        lo = __reduce_min_sync(0xffffffffu, lo);
        hi = __reduce_max_sync(0xffffffffu, hi);
        if (lane == 0) {
            s_pre[0] = pl; s_pre[1] = pc;
            if (last) {
                a.meta[META_MINLEN] = lo <= hi ? lo : 0u;
                a.meta[META_MAXLEN] = hi;
            }
        }
    }
    __syncthreads();
    unsigned long long run_len = s_pre[0], run_cost = s_pre[1];
    const uint32_t tile_lo = chunk * a.tiles_per_chunk;
    const uint32_t tile_hi = min(a.num_tiles, tile_lo + a.tiles_per_chunk);
    for (uint32_t tile = tile_lo; tile < tile_hi; ++tile) {
        const uint32_t base = tile * kScanTile + threadIdx.x * kScanItems;
        uint32_t v[kScanItems];
        unsigned long long t_len = 0, t_cost = 0;
        uint32_t n_valid = base < a.G ? min(a.G - base, static_cast<uint32_t>(kScanItems)) : 0u;
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) {
            v[i] = static_cast<uint32_t>(i) < n_valid ? load_len(a, base + i) : 0u;
            t_len += v[i];
            t_cost += static_cast<uint32_t>(i) < n_valid ? max(v[i], 1u) : 0u;
        }
        unsigned long long i_len = t_len, i_cost = t_cost;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long ul = __shfl_up_sync(0xffffffffu, i_len, d);
            const unsigned long long uc = __shfl_up_sync(0xffffffffu, i_cost, d);
            if (lane >= static_cast<uint32_t>(d)) { i_len += ul; i_cost += uc; }
        }
        __syncthreads();   // the previous tile's totals have been consumed
        if (lane == 31) { s_wlen[warp] = i_len; s_wcost[warp] = i_cost; }
        __syncthreads();
        unsigned long long w_len = 0, w_cost = 0, agg_len = 0, agg_cost = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) {
            const unsigned long long l = s_wlen[w], c = s_wcost[w];
            if (static_cast<uint32_t>(w) < warp) { w_len += l; w_cost += c; }
            agg_len += l; agg_cost += c;
        }
        unsigned long long off = run_len + w_len + i_len - t_len;   // offsets[base]
        unsigned long long c = run_cost + w_cost + i_cost - t_cost; // C[base]
        run_len += agg_len;
        run_cost += agg_cost;
        if (n_valid != 0) {
            if (base == 0) { a.seg[0] = make_int2(0, 0); a.seg_off[0] = 0; }
            unsigned long long q = c / a.K;
            unsigned long long next_boundary = (q + 1) * a.K;
#pragma unroll
            for (int i = 0; i < kScanItems; ++i) {
                if (static_cast<uint32_t>(i) < n_valid) {
                    a.offsets[base + i] = static_cast<long long>(off);
                    c += max(v[i], 1u);
                    off += v[i];                              // offsets[base + i + 1]
                    while (c >= next_boundary) {              // boundary s*K in (C[g], C[g+1]] belongs to bag g
                        ++q;
                        if (q < a.seg_cap) {
                            a.seg[q] = make_int2(static_cast<int>(base + i + 1), static_cast<int>(static_cast<uint32_t>(off)));
                            a.seg_off[q] = static_cast<long long>(off);
                        }
                        next_boundary += a.K;
                    }
                }
            }
            if (base + n_valid == a.G) {   // the thread that owns the last bag closes the plan
                a.offsets[a.G] = static_cast<long long>(off);
                const unsigned long long S = c / a.K + ((c % a.K) ? 1u : 0u);
                if ((c % a.K) != 0 && S < a.seg_cap) {
                    a.seg[S] = make_int2(static_cast<int>(a.G), static_cast<int>(static_cast<uint32_t>(off)));
                    a.seg_off[S] = static_cast<long long>(off);
                }
                const bool overflow = off > a.max_indices || S >= a.seg_cap;
                a.meta[META_S] = overflow ? 0 : static_cast<int32_t>(S);
                a.meta[META_N] = static_cast<int32_t>(static_cast<uint32_t>(off));
                a.meta[META_C] = static_cast<int32_t>(static_cast<uint32_t>(c));
                a.meta[META_OVERFLOW] = overflow ? 1 : 0;
                if (overflow) atomicAdd(a.state + kStateOverflows, 1u);
                a.meta[META_K] = static_cast<int32_t>(a.K);
                a.meta[META_G] = static_cast<int32_t>(a.G);
                a.meta[META_N_HI] = static_cast<int32_t>(off >> 32);
                a.meta[META_C_HI] = static_cast<int32_t>(c >> 32);
            }
        }
    }
}

}  // namespace

cudaError_t launch_plan64(const Plan64Args& a, cudaStream_t stream) {
    plan64_aggregate_kernel<<<a.num_chunks, kScanThreads, 0, stream>>>(a);
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    plan64_scan_kernel<<<a.num_chunks, kScanThreads, 0, stream>>>(a);
    count_launch();
    return cudaGetLastError();
}

}  // namespace dpi
