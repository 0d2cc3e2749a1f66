// forward_fused.cu -- steps a1 + a2 + a3 in ONE launch (dpi_forward on small / short-bag batches).
//
// Why: the paper's motivation is that a lookup is 4.75 us of work behind 21.92 us of launch overhead and
// its answer is ONE operation for all tables. With CSR bags the path became two launches (plan, lookup);
// for batches of microseconds the second launch and the plan's round trip through global memory are half of the step.
// Here the CTA that scans a run of bags pools those same bags right away:
//
//   chunk c = bags [c*chunk_bags, (c+1)*chunk_bags)     256 threads, W lanes per row, 256/W lane groups, <= 8 bags per thread
//     A  every thread loads the lengths of its <= 8 consecutive bags (registers; the chunk id is taken from a ticket, but
//        the loads are issued for chunk = blockIdx.x before the ticket returns -- they agree unless CTAs start out of order)
//     B  thread sums -> warp scan -> CTA totals: publish ONE status record {sum len, sum cost}; min / max by atomics
//     C  look-back: the threads poll the records of ALL earlier chunks at once (<= 3 each) and add them up: one L2 round
//        trip after the last predecessor publishes -- no chain, no grid-wide barrier
//     D  cp.async ALL index entries of the chunk into shared memory (one coalesced round trip, overlapped with:)
//        offsets[g] -> global (a1) and shared; segment records by boundary ownership, meta (a2): bit-exact, the plan stays
//        exportable and reusable by later dpi_lookup calls
//     E  pool the chunk's bags from shared offsets / indices (a3): only the row loads touch L2 / DRAM here
//
// Four CTA-wide barriers per launch in total (the first version scanned and pooled tile by tile, three barriers and one
// index round trip per 512 bags, 2 CTAs of 512 threads per SM: 12.3 / 31.6 us per step on c2 / c3 against 10.8 / 25.5 us for
// planner + lookup). Output-first holds as in the other kernels: consecutive lane groups own
// consecutive bags = consecutive output addresses.
// Pooling: one-hot chunks (longest bag 1) give each lane group 4 bags side by side; short chunks (longest bag <= kShortChunk)
// 2 bags side by side with up to 4 entries of each in flight; chunks with longer bags give each WARP a bag (sub-warps stride
// its entries, shuffle-reduce). Static chunks are not load-balanced across CTAs, which is why dpi_forward only takes this path
// when the plan's capacity says bags are short on average (max_indices <= 8 * G); everything else runs plan + balanced-segment
// lookup. Same arithmetic as lookup_kernel: fp32 accumulation in entry order, one RNE cast at the store, mean by
// reciprocal, bags of length <= 1 bit-exact, empty bags +0.0.
#include "lookup_kernels.cuh"
#include "nongemm_device.cuh"

namespace dpi {
namespace {

constexpr uint32_t kStateAggregate = 1u;
constexpr int kShortChunk = 16;     // chunks whose longest bag is at most this run the lane-group-per-bag path

__device__ __forceinline__ ulonglong2 ld_status(const ulonglong2* p) {
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

// Lane group q pools bags q, q + NG, ... of the chunk, U side by side; the entries of a bag are walked in order, so at
// every step U independent row loads per lane are in flight and nothing is spent on entries a bag does not have beyond the
// longest of the U (the first version kept 4 entries of each bag in flight and paid their conversions and adds whether
// they existed or not: 480 instructions per 16 bags on c3). s_off is padded with the chunk's end offset, so
// bags past the chunk read as empty without a bounds test. STAGED: every index entry of the chunk sits in shared memory.
template <class Tr, int W, bool OUT32, int U, bool STAGED>
__device__ __forceinline__ void pool_lane_groups(const LookupArgs& la, const char* const* s_tab, const int* s_off, const int* sidx,
                                                 uint32_t g_lo, uint32_t nb, uint32_t q, uint32_t sl, bool any_mean) {
    constexpr int NG = kFusedThreads / W;
    constexpr int kAcc2 = Tr::kAcc / 2;
    constexpr int kOutVec = out_vec_bytes<Tr, OUT32>();
    const bool vec_ok = sl < la.nvec;
    const uint32_t row_bytes = la.nvec * 16;
    const uint32_t ish = la.idx_shift;
    const uint32_t t_step = NG % la.T;
    uint32_t t = (g_lo + q) % la.T;
    const size_t bag_out = static_cast<size_t>(la.nvec) * kOutVec;
    char* po = static_cast<char*>(la.out) + (static_cast<size_t>(g_lo + q) * la.nvec + sl) * kOutVec;
    for (uint32_t i0 = q; i0 < nb; i0 += NG * U, po += bag_out * (NG * U)) {
        int lo[U], len[U];
        const char* tab[U];
        uint32_t tt[U];
        int n = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t i = i0 + u * NG;           // < kFusedMaxChunkBags + NG * U: inside the padded s_off
            lo[u] = s_off[i];
            len[u] = vec_ok ? s_off[i + 1] - lo[u] : 0;
            n = max(n, len[u]);
            tt[u] = t;
            tab[u] = s_tab[t] + sl * 16;
            t += t_step;
            if (t >= la.T) t -= la.T;
        }
        float2 acc[U][kAcc2];
#pragma unroll
        for (int u = 0; u < U; ++u) zero_acc(acc[u]);
        for (int j = 0; j < n; ++j) {
            uint4 v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool ok = j < len[u];
                const int e = lo[u] + j;
                uint32_t r = 0u;
                if constexpr (STAGED) r = static_cast<uint32_t>(sidx[e]);   // past a bag's end: a pad word, never used (the load is predicated off)
                else if (ok) r = static_cast<uint32_t>(__ldg(la.indices + (static_cast<size_t>(e) << ish)));
                v[u] = ld_row16(tab[u] + static_cast<uint64_t>(r) * row_bytes, ok);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) Tr::add(acc[u], v[u]);   // entry order; an absent entry adds +0.0
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (vec_ok && i0 + u * NG < nb) {
                if (any_mean && len[u] > 1 && ((la.pool.w[tt[u] >> 5] >> (tt[u] & 31)) & 1u)) scale_mean(acc[u], len[u]);
                store_pooled<Tr, OUT32>(po + bag_out * (u * NG), acc[u]);
            }
        }
    }
}

// ITEMS = bags per thread the scan phases are compiled for (1, 2, 4 or 8 >= the run-time count): with one launch covering
// 64 ... 2048 bags per CTA, code unrolled for 8 bags per thread cost a c2-sized batch (1 bag per thread) 700 instructions per
// warp before the first row was loaded.
template <class Tr, int W, bool OUT32, int ITEMS>
__global__ void __launch_bounds__(kFusedThreads, Tr::kEltBytes == 2 ? 3 : 4) fused_forward_kernel(const FusedArgs a) {
    constexpr int P = 32 / W;
    constexpr int NW = kFusedThreads / 32;         // warps per CTA
    constexpr int kAcc2 = Tr::kAcc / 2;
    constexpr int kOutVec = out_vec_bytes<Tr, OUT32>();
    extern __shared__ const char* s_tab[];         // [T]
    constexpr int kPad = 4 * (kFusedThreads / W);  // bags a lane group may look past the chunk (U <= 4 side by side)
    __shared__ int s_off[kFusedMaxChunkBags + kPad + 1];  // offsets of the chunk's bags (absolute entry positions), end-padded
    __shared__ int s_idx[kFusedIdxStage + kShortChunk];   // the chunk's index entries (low words for int64 ids) + read-ahead pad
    __shared__ uint32_t s_w[4][NW];                // per-warp {len, cost, max, min}
    __shared__ uint32_t s_p[2][NW];                // per-warp look-back partial sums
    __shared__ uint32_t s_bcast[2];                // ticket, epoch

    const PlanArgs& pa = a.plan;
    const LookupArgs& la = a.look;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t I = ITEMS == 1 ? 1u : a.items;  // bags per thread, <= ITEMS

    griddep_wait();  // PDL: nothing is read before the preceding grid (e.g. the previous step) has completed
    if (tid == 0) {
        s_bcast[0] = atomicInc(pa.state + kStateTicket, pa.num_chunks - 1);
        s_bcast[1] = *reinterpret_cast<volatile unsigned int*>(pa.state + kStateEpoch);
    }
    // ---- A: the lengths of this thread's I consecutive bags, issued before the ticket is back ----
    uint32_t v[ITEMS];
    uint32_t chunk = blockIdx.x;
    auto load_lengths = [&](uint32_t c) {
        const uint32_t c_lo = c * a.chunk_bags;
        const uint32_t c_n = min(pa.G - c_lo, a.chunk_bags);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const uint32_t local = tid * I + i;
            v[i] = (static_cast<uint32_t>(i) < I && local < c_n) ? static_cast<uint32_t>(__ldg(pa.len + c_lo + local)) : 0u;
        }
    };
    load_lengths(chunk);
    for (uint32_t t = tid; t < la.T; t += kFusedThreads) s_tab[t] = static_cast<const char*>(la.tables[t]);
    __syncthreads();
    const uint32_t epoch = s_bcast[1];
    if (s_bcast[0] != chunk) {   // CTAs did not start in blockIdx order: take the ticket's chunk (a chunk only waits on chunks
        chunk = s_bcast[0];      // whose CTAs already run)
        load_lengths(chunk);
    }
    const uint32_t g_lo = chunk * a.chunk_bags;
    const uint32_t nb = min(pa.G - g_lo, a.chunk_bags);   // bags of this chunk

    // ---- B: thread sums, warp scan, CTA totals; publish ----
    uint32_t t_len = 0, t_cost = 0, t_lo = 0xffffffffu, t_hi = 0u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const bool ok = static_cast<uint32_t>(i) < I && tid * I + i < nb;
        t_len += v[i];
        t_cost += ok ? max(v[i], 1u) : 0u;
        if (ok) { t_lo = min(t_lo, v[i]); t_hi = max(t_hi, v[i]); }
    }
    uint32_t i_len = t_len, i_cost = t_cost;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t ul = __shfl_up_sync(0xffffffffu, i_len, d);
        const uint32_t uc = __shfl_up_sync(0xffffffffu, i_cost, d);
        if (lane >= static_cast<uint32_t>(d)) { i_len += ul; i_cost += uc; }
    }
    const uint32_t w_hi = __reduce_max_sync(0xffffffffu, t_hi);
    const uint32_t w_lo = __reduce_min_sync(0xffffffffu, t_lo);
    if (lane == 31) { s_w[0][warp] = i_len; s_w[1][warp] = i_cost; s_w[2][warp] = w_hi; s_w[3][warp] = w_lo; }
    __syncthreads();
    uint32_t w_len = 0, w_cost = 0, agg_len = 0, agg_cost = 0, c_hi = 0u, c_lo = 0xffffffffu;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const uint32_t xl = s_w[0][w], xc = s_w[1][w];
        if (static_cast<uint32_t>(w) < warp) { w_len += xl; w_cost += xc; }
        agg_len += xl; agg_cost += xc;
        c_hi = max(c_hi, s_w[2][w]); c_lo = min(c_lo, s_w[3][w]);
    }
    if (tid == 0) {
        st_status(pa.status + chunk, pack_status(epoch, kStateAggregate, agg_len), pack_status(epoch, kStateAggregate, agg_cost));
        if (c_lo <= c_hi) {
            atomicMin(pa.state + kStateMinLen, c_lo);
            atomicMax(pa.state + kStateMaxLen, c_hi);
        }
    }
    // ---- C: look-back over all earlier chunks (every load of the CTA in flight together) ----
    uint32_t p_len = 0, p_cost = 0;
    for (uint32_t c = tid; c < chunk; c += kFusedThreads) {
        ulonglong2 w = ld_status(pa.status + c);
        while (!(status_ready(w.x, epoch) && status_ready(w.y, epoch))) w = ld_status(pa.status + c);
        p_len += static_cast<uint32_t>(w.x);
        p_cost += static_cast<uint32_t>(w.y);
    }
    p_len = __reduce_add_sync(0xffffffffu, p_len);
    p_cost = __reduce_add_sync(0xffffffffu, p_cost);
    if (lane == 0) { s_p[0][warp] = p_len; s_p[1][warp] = p_cost; }
    __syncthreads();
    uint32_t pre_len = 0, pre_cost = 0;   // offsets / C at the first bag of the chunk
#pragma unroll
    for (int w = 0; w < NW; ++w) { pre_len += s_p[0][w]; pre_cost += s_p[1][w]; }
    asm volatile("griddepcontrol.launch_dependents;");

    // ---- D: stage the chunk's index entries; offsets, segment records, meta ----
    const uint32_t ish = la.idx_shift;
    const uint32_t e_lo = pre_len, e_hi = pre_len + agg_len;
    const uint32_t n_stage = min(e_hi - e_lo, static_cast<uint32_t>(kFusedIdxStage));
    {
        const int* src = la.indices + (static_cast<size_t>(e_lo) << ish);
        for (uint32_t i = tid; i < n_stage; i += kFusedThreads) cp_async4(s_idx + i, src + (static_cast<size_t>(i) << ish));
    }
    cp_async_commit();
    {
        uint32_t off = pre_len + w_len + i_len - t_len;       // offsets[first bag of this thread]
        uint32_t c = pre_cost + w_cost + i_cost - t_cost;     // C[first bag of this thread]
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
            const uint32_t local = tid * I + i;
            if (static_cast<uint32_t>(i) < I && local < nb) {
                const uint32_t g = g_lo + local, l = v[i], cost = max(l, 1u);
                // a1: offsets; a2: every quantum boundary s*K inside (C[g], C[g+1]] belongs to bag g -> seg[s] = {g+1, offsets[g+1]}
                pa.offsets[g] = static_cast<int32_t>(off);
                s_off[local] = static_cast<int>(off);
                if (g == 0) pa.seg[0] = make_int2(0, 0);
                const uint32_t c1 = c + cost;
                uint32_t s = a.k_shift < 32u ? c >> a.k_shift : c / pa.K;   // the default quanta are powers of two
                unsigned long long next_boundary = static_cast<unsigned long long>(s + 1) * pa.K;
                while (c1 >= next_boundary) {
                    ++s;
                    if (s < pa.seg_cap) pa.seg[s] = make_int2(static_cast<int>(g + 1), static_cast<int>(off + l));
                    next_boundary += pa.K;
                }
                if (g + 1 == pa.G) {   // the thread that owns the last bag closes the plan
                    const uint32_t n_total = off + l;
                    pa.offsets[pa.G] = static_cast<int32_t>(n_total);
                    const uint32_t S = c1 / pa.K + ((c1 % pa.K) ? 1u : 0u);
                    if ((c1 % pa.K) != 0 && S < pa.seg_cap) pa.seg[S] = make_int2(static_cast<int>(pa.G), static_cast<int>(n_total));
                    const bool overflow = n_total > pa.max_indices || S >= pa.seg_cap;
                    pa.meta[META_S] = overflow ? 0 : S;   // the plan left behind must not drive a later dpi_lookup (this launch's own
                                                          // pooling cannot be held back: chunks pool before N is known, dpi.h)
                    pa.meta[META_N] = n_total;
                    pa.meta[META_C] = c1;
                    pa.meta[META_OVERFLOW] = overflow ? 1 : 0;
                    if (overflow) atomicAdd(pa.state + kStateOverflows, 1u);
                    pa.meta[META_K] = pa.K;
                    pa.meta[META_G] = pa.G;
                }
                off += l;
                c = c1;
            }
        }
        for (uint32_t i = nb + tid; i <= nb + kPad; i += kFusedThreads) s_off[i] = static_cast<int>(e_hi);   // end + padding
    }
    cp_async_wait<0>();
    __syncthreads();   // s_off and s_idx are complete

    // ---- E: pool the chunk's bags (a3) ----
    const uint32_t q = tid / W, sl = tid % W;
    const int* const sidx = s_idx - e_lo;   // indexed by absolute entry position
    const int stage_hi = static_cast<int>(e_lo + n_stage);
    const bool all_staged = n_stage == e_hi - e_lo;
    if (c_hi <= static_cast<uint32_t>(kShortChunk)) {
        if (!all_staged) pool_lane_groups<Tr, W, OUT32, 2, false>(la, s_tab, s_off, sidx, g_lo, nb, q, sl, a.any_mean != 0);
        else if (c_hi <= 1u) pool_lane_groups<Tr, W, OUT32, 4, true>(la, s_tab, s_off, sidx, g_lo, nb, q, sl, a.any_mean != 0);
        else pool_lane_groups<Tr, W, OUT32, 2, true>(la, s_tab, s_off, sidx, g_lo, nb, q, sl, a.any_mean != 0);
    } else {
        // a bag per warp: the P sub-warps stride its entries two rounds at a time, partial sums meet by shuffle
        const uint32_t sub = lane / W;
        const bool vec_ok = sl < la.nvec;
        const uint32_t row_bytes = la.nvec * 16;
        char* const out = static_cast<char*>(la.out);
        auto idx_at = [&](int e) -> uint32_t {
            return static_cast<uint32_t>(e < stage_hi ? sidx[e] : __ldg(la.indices + (static_cast<size_t>(e) << ish)));
        };
        for (uint32_t i = warp; i < nb; i += NW) {
            const int lo = s_off[i], hi = s_off[i + 1];
            const uint32_t t = (g_lo + i) % la.T;
            const char* tab = s_tab[t] + sl * 16;
            float2 acc[kAcc2];
            zero_acc(acc);
            for (int j = lo + static_cast<int>(sub); j < hi; j += 2 * P) {
                const bool ok1 = j + P < hi;
                const uint32_t r0 = idx_at(j);
                const uint32_t r1 = ok1 ? idx_at(j + P) : 0u;
                const uint4 v0 = ld_row16(tab + static_cast<uint64_t>(r0) * row_bytes, vec_ok);
                const uint4 v1 = ld_row16(tab + static_cast<uint64_t>(r1) * row_bytes, vec_ok && ok1);
                Tr::add(acc, v0);
                Tr::add(acc, v1);
            }
#pragma unroll
            for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                for (int x = 0; x < kAcc2; ++x)
                    acc[x] = __fadd2_rn(acc[x], make_float2(__shfl_xor_sync(0xffffffffu, acc[x].x, d),
                                                            __shfl_xor_sync(0xffffffffu, acc[x].y, d)));
            }
            if (sub == 0 && vec_ok) {
                if (((la.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                store_pooled<Tr, OUT32>(out + (static_cast<size_t>(g_lo + i) * la.nvec + sl) * kOutVec, acc);
            }
        }
    }

    // ---- FM epilogue (dpi_forward_fm; "combine all neighbouring non-GEMM operators into a single operator"):
    // chunks hold whole samples, so the FM second-order term of a sample is formed by this CTA from the T pooled vectors it
    // has just stored -- read back through L2 (coherent loads, after a CTA barrier), not from HBM by a second kernel.
    // Same per-sample code as fm_kernel: bit-identical to dpi_fm_interaction run on the block this launch wrote. ----
    if constexpr (!(OUT32 && Tr::kEltBytes == 2)) {
        if (a.fm_y != nullptr || a.fm_v != nullptr) {
            __syncthreads();
            FmArgs fa;
            fa.x = static_cast<const char*>(la.out);
            fa.y = a.fm_y; fa.v = a.fm_v;
            fa.x_pitch = static_cast<uint64_t>(la.T) * la.nvec * 16;
            fa.B = la.B; fa.T = la.T; fa.nvec = la.nvec;
            fa.D = la.nvec * (16 / Tr::kEltBytes);
            const uint32_t b0 = g_lo / la.T, ns = nb / la.T;
            for (uint32_t b = warp; b < ns; b += NW) fm_one_sample<Tr::kDtype, W, 4>(fa, b0 + b, static_cast<int>(lane));
        }
    }

    // ---- close the epoch (as in plan_scan_partition_kernel): the last CTA copies min / max into meta and advances the tag ----
    if (tid == 0) {
        __threadfence();
        if (atomicInc(pa.state + kStateDone, pa.num_chunks - 1) == pa.num_chunks - 1) {
            __threadfence();
            const uint32_t lo = *reinterpret_cast<volatile unsigned int*>(pa.state + kStateMinLen);
            const uint32_t hi = *reinterpret_cast<volatile unsigned int*>(pa.state + kStateMaxLen);
            pa.meta[META_MINLEN] = lo <= hi ? lo : 0u;
            pa.meta[META_MAXLEN] = hi;
            pa.state[kStateMinLen] = 0xffffffffu;
            pa.state[kStateMaxLen] = 0u;
            uint32_t next = epoch + 1;
            if (next >= kEpochLimit) {
                for (uint32_t i = 0; i < static_cast<uint32_t>(kStatusRecords); ++i) pa.status[i] = make_ulonglong2(0ull, 0ull);
                next = 1;
            }
            pa.state[kStateEpoch] = next;
        }
    }
}

template <class Tr, bool OUT32, int ITEMS, class F>
auto for_lanes(int lanes, F&& f) {
    switch (lanes) {
        case 1: return f(fused_forward_kernel<Tr, 1, OUT32, ITEMS>);
        case 2: return f(fused_forward_kernel<Tr, 2, OUT32, ITEMS>);
        case 4: return f(fused_forward_kernel<Tr, 4, OUT32, ITEMS>);
        case 8: return f(fused_forward_kernel<Tr, 8, OUT32, ITEMS>);
        case 16: return f(fused_forward_kernel<Tr, 16, OUT32, ITEMS>);
        case 32: return f(fused_forward_kernel<Tr, 32, OUT32, ITEMS>);
        default: return f(static_cast<void (*)(const FusedArgs)>(nullptr));
    }
}
template <class Tr, bool OUT32, class F>
auto for_items(uint32_t items, int lanes, F&& f) {
    if (items <= 1) return for_lanes<Tr, OUT32, 1>(lanes, f);
    if (items <= 2) return for_lanes<Tr, OUT32, 2>(lanes, f);
    if (items <= 4) return for_lanes<Tr, OUT32, 4>(lanes, f);
    return for_lanes<Tr, OUT32, kFusedItems>(lanes, f);
}
template <class F>
auto for_kernel(int dtype, bool out32, int lanes, uint32_t items, F&& f) {
    switch (dtype) {
        case DPI_F32: return for_items<F32Traits, false>(items, lanes, f);
        case DPI_F16: return out32 ? for_items<F16Traits, true>(items, lanes, f) : for_items<F16Traits, false>(items, lanes, f);
        default: return out32 ? for_items<BF16Traits, true>(items, lanes, f) : for_items<BF16Traits, false>(items, lanes, f);
    }
}

}  // namespace

int fused_occupancy(int dtype, bool out32, int lanes, uint32_t T) {
    return for_kernel(dtype, out32, lanes, kFusedItems, [&](void (*k)(const FusedArgs)) -> int {
        int occ = 0;
        if (!k || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, kFusedThreads, static_cast<size_t>(T) * sizeof(const char*)) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        return occ;
    });
}

cudaError_t launch_fused(const FusedArgs& a, int dtype, bool out32, int lanes, bool pdl, cudaStream_t stream) {
    return for_kernel(dtype, out32, lanes, a.items, [&](void (*k)(const FusedArgs)) -> cudaError_t {
        if (!k) return cudaErrorInvalidValue;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(a.plan.num_chunks);
        cfg.blockDim = dim3(kFusedThreads);
        cfg.dynamicSmemBytes = static_cast<size_t>(a.look.T) * sizeof(const char*);
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
