// plan_kernels.cu -- steps a1 + a2 of the path: "anticipate the whole workload".
//
// ONE launch over all G = B*T (sample, table) bags -- no per-table launches:
//   * single-pass decoupled look-back exclusive scan of (len, cost = max(len,1)) pairs  -> offsets[G+1]
//   * fused partition: bag g knows C[g] and C[g+1]; it owns every quantum boundary s*K in (C[g], C[g+1]],
//     i.e. seg_bag[s] = g+1 for s = floor(C[g]/K)+1 .. floor(C[g+1]/K).  That is exactly
//     seg_bag[s] = min{g : C[g] >= s*K} without any binary search or second kernel.
//     Next to it goes seg_off[s] = offsets[seg_bag[s]] (first entry of the task), interleaved as int2
//     {seg_bag, seg_off}, so the lookup reaches a task's indices with one dependent load instead of two.
// Integer work only; results are bit-exact against oracle/dpi_oracle.c::oracle_plan.
//
// Bytes: 4 B read + 4 B written per bag, 4 B per segment -- HBM/L2-bound, ~microseconds at G <= 1e6.
#include "dpi_internal.cuh"

namespace dpi {
namespace {

constexpr uint32_t kStateAggregate = 1u;
constexpr uint32_t kStateInclusive = 2u;

__device__ __forceinline__ unsigned long long ld_relaxed_gpu(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long pack_status(uint32_t epoch, uint32_t state, uint32_t value) {
    return (static_cast<unsigned long long>((epoch << 2) | state) << 32) | value;
}

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// Warp-parallel decoupled look-back over two status arrays at once. Lane l inspects tile pos-l; the window
// slides back 32 tiles until some lane sees an INCLUSIVE word. Tiles before 0 count as inclusive-zero.
__device__ __forceinline__ void lookback(const unsigned long long* st_len, const unsigned long long* st_cost,
                                         uint32_t tile, uint32_t epoch, uint32_t& pre_len, uint32_t& pre_cost) {
    const int lane = threadIdx.x & 31;
    uint32_t run_len = 0, run_cost = 0;
    bool done_len = false, done_cost = false;  // warp-uniform
    int pos = static_cast<int>(tile) - 1;
    while (!(done_len && done_cost)) {
        const int my = pos - lane;
        uint32_t f_len = kStateInclusive, v_len = 0, f_cost = kStateInclusive, v_cost = 0;
        if (my >= 0) {
            if (!done_len) {
                unsigned long long w;
                uint32_t hi;
                do {
                    w = ld_relaxed_gpu(st_len + my);
                    hi = static_cast<uint32_t>(w >> 32);
                } while ((hi >> 2) != epoch || (hi & 3u) == 0u);
                f_len = hi & 3u;
                v_len = static_cast<uint32_t>(w);
            }
            if (!done_cost) {
                unsigned long long w;
                uint32_t hi;
                do {
                    w = ld_relaxed_gpu(st_cost + my);
                    hi = static_cast<uint32_t>(w >> 32);
                } while ((hi >> 2) != epoch || (hi & 3u) == 0u);
                f_cost = hi & 3u;
                v_cost = static_cast<uint32_t>(w);
            }
        }
        if (!done_len) {
            const uint32_t incl = __ballot_sync(0xffffffffu, f_len == kStateInclusive);
            const int first = __ffs(incl) - 1;  // nearest predecessor that already has its inclusive prefix
            run_len += warp_sum((first < 0 || lane <= first) ? v_len : 0u);
            done_len = first >= 0;
        }
        if (!done_cost) {
            const uint32_t incl = __ballot_sync(0xffffffffu, f_cost == kStateInclusive);
            const int first = __ffs(incl) - 1;
            run_cost += warp_sum((first < 0 || lane <= first) ? v_cost : 0u);
            done_cost = first >= 0;
        }
        pos -= 32;
    }
    pre_len = run_len;
    pre_cost = run_cost;
}

__global__ void __launch_bounds__(kScanThreads) plan_scan_partition_kernel(const PlanArgs a) {
    __shared__ uint32_t s_tile, s_epoch;
    __shared__ uint32_t s_wlen[kScanThreads / 32], s_wcost[kScanThreads / 32];
    __shared__ uint32_t s_pre_len, s_pre_cost;

    // The epoch that tags this build's look-back words lives in device memory and is advanced by the last tile
    // to finish, so a build needs no host-side state: the same launch can be replayed from a CUDA graph.
    if (threadIdx.x == 0) {
        s_tile = atomicInc(a.state + kStateTicket, a.num_tiles - 1);  // wraps to 0 after the last tile
        s_epoch = *reinterpret_cast<volatile unsigned int*>(a.state + kStateEpoch);
    }
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t epoch = s_epoch;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t base = tile * kScanTile + threadIdx.x * kScanItems;

    // ---- load kScanItems consecutive lengths (two 128-bit loads when the whole run is in range) ----
    uint32_t v[kScanItems];
    uint32_t n_valid;
    if (base + kScanItems <= a.G && (reinterpret_cast<uintptr_t>(a.len) & 15u) == 0) {
        const int4 p0 = __ldg(reinterpret_cast<const int4*>(a.len + base));
        const int4 p1 = __ldg(reinterpret_cast<const int4*>(a.len + base) + 1);
        v[0] = p0.x; v[1] = p0.y; v[2] = p0.z; v[3] = p0.w;
        v[4] = p1.x; v[5] = p1.y; v[6] = p1.z; v[7] = p1.w;
        n_valid = kScanItems;
    } else {
        n_valid = base < a.G ? min(a.G - base, static_cast<uint32_t>(kScanItems)) : 0u;
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) v[i] = (static_cast<uint32_t>(i) < n_valid) ? __ldg(a.len + base + i) : 0u;
    }
    uint32_t t_len = 0, t_cost = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        t_len += v[i];
        t_cost += (static_cast<uint32_t>(i) < n_valid) ? max(v[i], 1u) : 0u;
    }

    // ---- CTA-wide exclusive scan of the per-thread sums ----
    uint32_t i_len = t_len, i_cost = t_cost;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t ul = __shfl_up_sync(0xffffffffu, i_len, d);
        const uint32_t uc = __shfl_up_sync(0xffffffffu, i_cost, d);
        if (lane >= static_cast<uint32_t>(d)) { i_len += ul; i_cost += uc; }
    }
    if (lane == 31) { s_wlen[warp] = i_len; s_wcost[warp] = i_cost; }
    __syncthreads();
    uint32_t w_len = 0, w_cost = 0, agg_len = 0, agg_cost = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        const uint32_t l = s_wlen[w], c = s_wcost[w];
        if (static_cast<uint32_t>(w) < warp) { w_len += l; w_cost += c; }
        agg_len += l; agg_cost += c;
    }
    const uint32_t ex_len = w_len + i_len - t_len;     // exclusive prefix of this thread inside the tile
    const uint32_t ex_cost = w_cost + i_cost - t_cost;

    // ---- decoupled look-back: publish aggregate, fetch predecessor prefix, publish inclusive ----
    if (warp == 0) {
        if (tile == 0) {
            if (lane == 0) {
                st_relaxed_gpu(a.tile_len + 0, pack_status(epoch, kStateInclusive, agg_len));
                st_relaxed_gpu(a.tile_cost + 0, pack_status(epoch, kStateInclusive, agg_cost));
                s_pre_len = 0; s_pre_cost = 0;
            }
        } else {
            if (lane == 0) {
                st_relaxed_gpu(a.tile_len + tile, pack_status(epoch, kStateAggregate, agg_len));
                st_relaxed_gpu(a.tile_cost + tile, pack_status(epoch, kStateAggregate, agg_cost));
            }
            uint32_t pl, pc;
            lookback(a.tile_len, a.tile_cost, tile, epoch, pl, pc);
            if (lane == 0) {
                st_relaxed_gpu(a.tile_len + tile, pack_status(epoch, kStateInclusive, pl + agg_len));
                st_relaxed_gpu(a.tile_cost + tile, pack_status(epoch, kStateInclusive, pc + agg_cost));
                s_pre_len = pl; s_pre_cost = pc;
            }
        }
    }
    __syncthreads();
    // Let a dependent (PDL) lookup kernel start its prologue; it still waits for this grid to finish
    // and flush before it reads the plan.
    asm volatile("griddepcontrol.launch_dependents;");

    if (n_valid == 0) return;
    uint32_t off = s_pre_len + ex_len;    // offsets[base]
    uint32_t c = s_pre_cost + ex_cost;    // C[base]

    // ---- a1: offsets ----
    if (n_valid == kScanItems) {
        int4 o0, o1;
        uint32_t r = off;
        o0.x = r; r += v[0]; o0.y = r; r += v[1]; o0.z = r; r += v[2]; o0.w = r; r += v[3];
        o1.x = r; r += v[4]; o1.y = r; r += v[5]; o1.z = r; r += v[6]; o1.w = r;
        reinterpret_cast<int4*>(a.offsets + base)[0] = o0;   // offsets is 256-B aligned (cudaMalloc), base % 8 == 0
        reinterpret_cast<int4*>(a.offsets + base)[1] = o1;
    } else {
        uint32_t r = off;
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) {
            if (static_cast<uint32_t>(i) < n_valid) a.offsets[base + i] = r;
            r += v[i];
        }
    }

    // ---- a2: every quantum boundary s*K inside (C[g], C[g+1]] belongs to bag g -> seg_bag[s] = g+1 ----
    if (base == 0) a.seg[0] = make_int2(0, 0);      // s = 0: C[0] = 0 >= 0
    uint32_t q_prev = c / a.K;
    uint32_t run = off;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (static_cast<uint32_t>(i) < n_valid) {
            c += max(v[i], 1u);
            run += v[i];                             // offsets[base + i + 1]
            const uint32_t q = c / a.K;
            for (uint32_t s = q_prev + 1; s <= q; ++s)
                if (s < a.seg_cap) a.seg[s] = make_int2(base + i + 1, run);
            q_prev = q;
        }
    }

    // ---- the thread that owns the last bag closes the plan ----
    if (base + n_valid == a.G) {
        uint32_t n_total = off;
#pragma unroll
        for (int i = 0; i < kScanItems; ++i) n_total += v[i];
        a.offsets[a.G] = n_total;
        const uint32_t S = c / a.K + ((c % a.K) ? 1u : 0u);   // ceil(C[G]/K)
        if ((c % a.K) != 0 && S < a.seg_cap) a.seg[S] = make_int2(a.G, n_total);  // C[G] < S*K: clamped to G
        a.meta[META_S] = (S < a.seg_cap) ? S : 0;             // an overflowed plan must not drive a lookup
        a.meta[META_N] = n_total;
        a.meta[META_C] = c;
        a.meta[META_OVERFLOW] = (n_total > a.max_indices || S >= a.seg_cap) ? 1 : 0;
        a.meta[META_K] = a.K;
        a.meta[META_G] = a.G;
    }

    // ---- close the epoch: no thread of this CTA reads a status word past the barrier above; the last tile to
    // get here advances the tag (a later build starts only after this grid has completed) ----
    if (threadIdx.x == 0 && atomicInc(a.state + kStateDone, a.num_tiles - 1) == a.num_tiles - 1) {
        uint32_t next = epoch + 1;
        if (next >= kEpochLimit) {  // 30-bit tag about to wrap: clear the words once and restart at 1
            for (uint32_t i = 0; i < a.num_tiles; ++i) { a.tile_len[i] = 0ull; a.tile_cost[i] = 0ull; }
            next = 1;
        }
        a.state[kStateEpoch] = next;
    }
}

__global__ void __launch_bounds__(256) check_indices_kernel(const CheckArgs a) {
    unsigned long long bad = 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < a.G; g += gridDim.x * blockDim.x) {
        const long long rows = a.table_rows[a.table_major ? g / a.B : g % a.T];
        const int lo = a.offsets[g], hi = a.offsets[g + 1];
        for (int j = lo; j < hi; ++j) {
            const long long r = a.idx64 ? static_cast<const long long*>(a.indices)[j]
                                        : static_cast<long long>(static_cast<const int*>(a.indices)[j]);
            bad += (r < 0 || r >= rows) ? 1ull : 0ull;
        }
    }
    if (bad) atomicAdd(a.n_bad, bad);
}

}  // namespace

cudaError_t launch_plan(const PlanArgs& a, cudaStream_t stream) {
    plan_scan_partition_kernel<<<a.num_tiles, kScanThreads, 0, stream>>>(a);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_check_indices(const CheckArgs& a, cudaStream_t stream) {
    const uint32_t blocks = min((a.G + 255u) / 256u, 148u * 8u);
    check_indices_kernel<<<blocks ? blocks : 1, 256, 0, stream>>>(a);
    count_launch();
    return cudaGetLastError();
}

}  // namespace dpi
