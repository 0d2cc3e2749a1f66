// plan_kernels.cu -- steps a1 + a2 of the path: "anticipate the whole workload".
//
// ONE launch over all G = B*T (sample, table) bags -- no per-table launches:
//   * chunked single-pass exclusive scan of (len, cost = max(len,1)) pairs -> offsets[G+1]. The bags are cut into
//     C <= kMaxChunks contiguous chunks (whole 2048-bag tiles), one CTA per chunk, all CTAs co-resident:
//       pass 1  the CTA sums its chunk and publishes ONE status record {len aggregate, cost aggregate};
//       look-back  warp 0 reads the records of ALL earlier chunks at once (<= 320 records, 16 B each, every load
//                  in flight together) and adds them up -- one L2 round trip after the last predecessor publishes,
//                  no inclusive state, no chain;
//       pass 2  the CTA scans its chunk tile by tile from that prefix (a one-tile chunk keeps its lengths in
//               registers, larger chunks re-read them from L1/L2) and writes offsets and segments.
//     (The first version was a textbook decoupled look-back over one status word per 2048-bag tile: with hundreds
//     of CTAs polling the same few cache lines it cost ~25 ns per TILE -- 13.5 us at G = 524 K, 75 us at
//     G = 6.5 M -- against ~3 us of launch latency.)
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

__device__ __forceinline__ ulonglong2 ld_status(const ulonglong2* p) {
    // The two 64-bit halves are validated independently (each carries epoch + state), so a torn 128-bit read is
    // harmless: a half that is not ready yet is simply read again.
    ulonglong2 v;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(ulonglong2* p, unsigned long long x, unsigned long long y) {
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(x), "l"(y) : "memory");
}
__device__ __forceinline__ unsigned long long pack_status(uint32_t epoch, uint32_t state, uint32_t value) {
    return (static_cast<unsigned long long>((epoch << 2) | state) << 32) | value;
}
__device__ __forceinline__ bool status_ready(unsigned long long w, uint32_t epoch) {
    const uint32_t hi = static_cast<uint32_t>(w >> 32);
    return (hi >> 2) == epoch && (hi & 3u) != 0u;
}

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// Sum of the aggregates of chunks 0..chunk-1 (warp-wide; every lane returns the totals). Lane l owns chunks
// l, l+32, ...; all its loads are issued before the first is examined; only records that are not ready are re-read.
__device__ __forceinline__ void lookback_all(const ulonglong2* status, uint32_t chunk, uint32_t epoch,
                                             uint32_t& pre_len, uint32_t& pre_cost) {
    constexpr int kDepth = kMaxChunks / 32;
    const uint32_t lane = threadIdx.x & 31;
    ulonglong2 w[kDepth];
#pragma unroll
    for (int k = 0; k < kDepth; ++k) {
        const uint32_t c = lane + 32u * k;
        w[k] = c < chunk ? ld_status(status + c) : make_ulonglong2(pack_status(epoch, kStateAggregate, 0u), pack_status(epoch, kStateAggregate, 0u));
    }
    // Re-read every record that is not ready yet, all of them in flight together, until none is left (a serial
    // re-poll costs one L2 round trip per record: 8 us for the last chunks when traced with %globaltimer).
    for (;;) {
        bool all_ready = true;
#pragma unroll
        for (int k = 0; k < kDepth; ++k) all_ready &= status_ready(w[k].x, epoch) && status_ready(w[k].y, epoch);
        if (all_ready) break;
#pragma unroll
        for (int k = 0; k < kDepth; ++k) {
            if (!(status_ready(w[k].x, epoch) && status_ready(w[k].y, epoch))) w[k] = ld_status(status + lane + 32u * k);
        }
    }
    uint32_t sl = 0, sc = 0;
#pragma unroll
    for (int k = 0; k < kDepth; ++k) {
        sl += static_cast<uint32_t>(w[k].x);
        sc += static_cast<uint32_t>(w[k].y);
    }
    pre_len = warp_sum(sl);
    pre_cost = warp_sum(sc);
}

// Loads the kScanItems consecutive lengths of this thread in tile `tile` (zeros past G); returns how many are valid.
__device__ __forceinline__ uint32_t load_items(const PlanArgs& a, uint32_t tile, uint32_t (&v)[kScanItems]) {
    const uint32_t base = tile * kScanTile + threadIdx.x * kScanItems;
    if (base + kScanItems <= a.G && (reinterpret_cast<uintptr_t>(a.len) & 15u) == 0) {
        const int4 p0 = __ldg(reinterpret_cast<const int4*>(a.len + base));
        const int4 p1 = __ldg(reinterpret_cast<const int4*>(a.len + base) + 1);
        v[0] = p0.x; v[1] = p0.y; v[2] = p0.z; v[3] = p0.w;
        v[4] = p1.x; v[5] = p1.y; v[6] = p1.z; v[7] = p1.w;
        return kScanItems;
    }
    const uint32_t n_valid = base < a.G ? min(a.G - base, static_cast<uint32_t>(kScanItems)) : 0u;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) v[i] = (static_cast<uint32_t>(i) < n_valid) ? __ldg(a.len + base + i) : 0u;
    return n_valid;
}

__device__ __forceinline__ void thread_sums(const uint32_t (&v)[kScanItems], uint32_t n_valid, uint32_t& t_len, uint32_t& t_cost) {
    t_len = 0; t_cost = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        t_len += v[i];
        t_cost += (static_cast<uint32_t>(i) < n_valid) ? max(v[i], 1u) : 0u;
    }
}
// a1's summary of the lengths: running min / max over the valid items of this thread
__device__ __forceinline__ void thread_minmax(const uint32_t (&v)[kScanItems], uint32_t n_valid, uint32_t& lo, uint32_t& hi) {
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (static_cast<uint32_t>(i) < n_valid) {
            lo = min(lo, v[i]);
            hi = max(hi, v[i]);
        }
    }
}

__global__ void __launch_bounds__(kScanThreads) plan_scan_partition_kernel(const PlanArgs a) {
    __shared__ uint32_t s_chunk, s_epoch;
    __shared__ uint32_t s_wlen[2][kScanThreads / 32], s_wcost[2][kScanThreads / 32];
    __shared__ uint32_t s_wmin[kScanThreads / 32], s_wmax[kScanThreads / 32];
    __shared__ uint32_t s_pre_len, s_pre_cost;

    // Chunk ids are handed out by a ticket, so a chunk only ever waits on chunks that already run. The epoch that
    // tags this build's status records lives in device memory and is advanced by the last CTA to finish, so a
    // build needs no host-side state: the same launch can be replayed from a CUDA graph.
    if (threadIdx.x == 0) {
        s_chunk = atomicInc(a.state + kStateTicket, a.num_chunks - 1);  // wraps to 0 after the last chunk
        s_epoch = *reinterpret_cast<volatile unsigned int*>(a.state + kStateEpoch);
    }
    __syncthreads();
    const uint32_t chunk = s_chunk;
    const uint32_t epoch = s_epoch;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t tile_lo = chunk * a.tiles_per_chunk;
    const uint32_t tile_hi = min(a.num_tiles, tile_lo + a.tiles_per_chunk);

    // ---- pass 1: aggregate of the chunk ----
    uint32_t v[kScanItems];            // lengths of the chunk's FIRST tile stay in registers
    uint32_t n_valid = load_items(a, tile_lo, v);
    uint32_t t_len, t_cost;
    thread_sums(v, n_valid, t_len, t_cost);
    uint32_t len_lo = 0xffffffffu, len_hi = 0u;
    thread_minmax(v, n_valid, len_lo, len_hi);
    uint32_t c_len = t_len, c_cost = t_cost;
    for (uint32_t tile = tile_lo + 1; tile < tile_hi; ++tile) {
        uint32_t u[kScanItems], ul, uc;
        const uint32_t nv = load_items(a, tile, u);
        thread_sums(u, nv, ul, uc);
        thread_minmax(u, nv, len_lo, len_hi);
        c_len += ul; c_cost += uc;
    }
    c_len = warp_sum(c_len);
    c_cost = warp_sum(c_cost);
    len_lo = __reduce_min_sync(0xffffffffu, len_lo);
    len_hi = __reduce_max_sync(0xffffffffu, len_hi);
    if (lane == 0) { s_wlen[0][warp] = c_len; s_wcost[0][warp] = c_cost; s_wmin[warp] = len_lo; s_wmax[warp] = len_hi; }
    __syncthreads();
    if (warp == 0) {
        uint32_t agg_len = 0, agg_cost = 0, agg_lo = 0xffffffffu, agg_hi = 0u;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) {
            agg_len += s_wlen[0][w]; agg_cost += s_wcost[0][w];
            agg_lo = min(agg_lo, s_wmin[w]); agg_hi = max(agg_hi, s_wmax[w]);
        }
        if (lane == 0) {
            st_status(a.status + chunk, pack_status(epoch, kStateAggregate, agg_len), pack_status(epoch, kStateAggregate, agg_cost));
            // min / max leave the CTA as two fire-and-forget reductions into the planner state; the last CTA to finish
            // copies them into meta and re-arms the words for the next build
            if (agg_lo <= agg_hi) {
                atomicMin(a.state + kStateMinLen, agg_lo);
                atomicMax(a.state + kStateMaxLen, agg_hi);
            }
        }
        uint32_t pl, pc;
        lookback_all(a.status, chunk, epoch, pl, pc);
        if (lane == 0) { s_pre_len = pl; s_pre_cost = pc; }
    }
    __syncthreads();
    // Let a dependent (PDL) lookup kernel start its prologue; it still waits for this grid to finish
    // and flush before it reads the plan.
    asm volatile("griddepcontrol.launch_dependents;");

    // ---- pass 2: scan the chunk tile by tile from its prefix ----
    uint32_t run_len = s_pre_len, run_cost = s_pre_cost;   // offsets / C at the first bag of the current tile
    for (uint32_t tile = tile_lo; tile < tile_hi; ++tile) {
        const int sb = (tile - tile_lo) & 1;               // double-buffered scratch: one barrier per tile
        uint32_t u[kScanItems];                            // next tile's lengths, requested before this tile is scanned
        uint32_t nv_next = 0;
        const bool has_next = tile + 1 < tile_hi;
        if (has_next) nv_next = load_items(a, tile + 1, u);
        uint32_t i_len = t_len, i_cost = t_cost;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t ul = __shfl_up_sync(0xffffffffu, i_len, d);
            const uint32_t uc = __shfl_up_sync(0xffffffffu, i_cost, d);
            if (lane >= static_cast<uint32_t>(d)) { i_len += ul; i_cost += uc; }
        }
        if (lane == 31) { s_wlen[sb][warp] = i_len; s_wcost[sb][warp] = i_cost; }
        __syncthreads();
        uint32_t w_len = 0, w_cost = 0, agg_len = 0, agg_cost = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) {
            const uint32_t l = s_wlen[sb][w], c = s_wcost[sb][w];
            if (static_cast<uint32_t>(w) < warp) { w_len += l; w_cost += c; }
            agg_len += l; agg_cost += c;
        }
        const uint32_t base = tile * kScanTile + threadIdx.x * kScanItems;
        const uint32_t off = run_len + w_len + i_len - t_len;     // offsets[base]
        uint32_t c = run_cost + w_cost + i_cost - t_cost;         // C[base]
        run_len += agg_len;
        run_cost += agg_cost;
        if (n_valid != 0) {
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
            // One division per thread; after that the next boundary (q+1)*K is carried along (64-bit: it may pass 2^32).
            if (base == 0) a.seg[0] = make_int2(0, 0);      // s = 0: C[0] = 0 >= 0
            uint32_t q = c / a.K;                           // boundaries <= C[base] belong to earlier bags
            unsigned long long next_boundary = static_cast<unsigned long long>(q + 1) * a.K;
            uint32_t run = off;
#pragma unroll
            for (int i = 0; i < kScanItems; ++i) {
                if (static_cast<uint32_t>(i) < n_valid) {
                    c += max(v[i], 1u);
                    run += v[i];                             // offsets[base + i + 1]
                    while (c >= next_boundary) {
                        ++q;
                        if (q < a.seg_cap) a.seg[q] = make_int2(base + i + 1, run);
                        next_boundary += a.K;
                    }
                }
            }

            // ---- the thread that owns the last bag closes the plan ----
            if (base + n_valid == a.G) {
                const uint32_t n_total = run;
                a.offsets[a.G] = n_total;
                const uint32_t S = c / a.K + ((c % a.K) ? 1u : 0u);   // ceil(C[G]/K)
                if ((c % a.K) != 0 && S < a.seg_cap) a.seg[S] = make_int2(a.G, n_total);  // C[G] < S*K: clamped to G
                const bool overflow = n_total > a.max_indices || S >= a.seg_cap;
                a.meta[META_S] = overflow ? 0 : S;                    // an overflowed plan must not drive a lookup (S = 0 is the mark:
                                                                      // a fitting batch has S >= 1), as in plan64_kernels.cu
                a.meta[META_N] = n_total;
                a.meta[META_C] = c;
                a.meta[META_OVERFLOW] = overflow ? 1 : 0;
                if (overflow) atomicAdd(a.state + kStateOverflows, 1u);   // sticky until dpi_plan_status reads it
                a.meta[META_K] = a.K;
                a.meta[META_G] = a.G;
            }
        }
        if (has_next) {
#pragma unroll
            for (int i = 0; i < kScanItems; ++i) v[i] = u[i];
            n_valid = nv_next;
            thread_sums(v, n_valid, t_len, t_cost);
        }
    }
    // ---- close the epoch: no thread of this CTA reads a status record past the barrier after the look-back; the
    // last CTA to get here advances the tag (a later build starts only after this grid has completed) ----
    if (threadIdx.x == 0) __threadfence();  // this CTA's min / max reductions (issued by this thread) before the count
    if (threadIdx.x == 0 && atomicInc(a.state + kStateDone, a.num_chunks - 1) == a.num_chunks - 1) {
        __threadfence();
        const uint32_t lo = *reinterpret_cast<volatile unsigned int*>(a.state + kStateMinLen);
        const uint32_t hi = *reinterpret_cast<volatile unsigned int*>(a.state + kStateMaxLen);
        a.meta[META_MINLEN] = lo <= hi ? lo : 0u;   // G >= 1 always, so lo <= hi; kept total for safety
        a.meta[META_MAXLEN] = hi;
        a.state[kStateMinLen] = 0xffffffffu;
        a.state[kStateMaxLen] = 0u;
        uint32_t next = epoch + 1;
        if (next >= kEpochLimit) {  // 30-bit tag about to wrap: clear the records once and restart at 1
            // all kStatusRecords of them: the buffer is shared with fused_forward_kernel, which tags up to 640 records
            for (uint32_t i = 0; i < static_cast<uint32_t>(kStatusRecords); ++i) a.status[i] = make_ulonglong2(0ull, 0ull);
            next = 1;
        }
        a.state[kStateEpoch] = next;
    }
}

__global__ void __launch_bounds__(256) check_indices_kernel(const CheckArgs a) {
    unsigned long long bad = 0, too_long = 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < a.G; g += gridDim.x * blockDim.x) {
        const long long rows = a.table_rows[a.table_major ? g / a.B : g % a.T];
        const long long lo = a.off64 ? reinterpret_cast<const long long*>(a.offsets)[g] : a.offsets[g];
        const long long hi = a.off64 ? reinterpret_cast<const long long*>(a.offsets)[g + 1] : a.offsets[g + 1];
        too_long += (a.max_bag > 0 && hi - lo > a.max_bag) ? 1ull : 0ull;
        for (long long j = lo; j < hi; ++j) {
            const long long r = a.idx64 ? static_cast<const long long*>(a.indices)[j]
                                        : static_cast<long long>(static_cast<const int*>(a.indices)[j]);
            bad += (r < 0 || r >= rows) ? 1ull : 0ull;
        }
    }
    if (bad) atomicAdd(a.n_bad, bad);
    if (too_long) atomicAdd(a.n_bad + 1, too_long);
}

}  // namespace

cudaError_t launch_plan(const PlanArgs& a, cudaStream_t stream) {
    plan_scan_partition_kernel<<<a.num_chunks, kScanThreads, 0, stream>>>(a);
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
