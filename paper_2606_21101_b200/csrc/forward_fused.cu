// forward_fused.cu -- steps a1 + a2 + a3 in ONE launch (dpi_forward on small / short-bag batches).
//
// Why: the paper's motivation is that a lookup is 4.75 us of work behind 21.92 us of launch overhead and
// its answer is ONE operation for all tables. With CSR bags the path became two launches (plan, lookup);
// for batches of microseconds the second launch and the plan's round trip through global memory are half of the step.
// Here the CTA that scans a run of bags pools those same bags right away:
//
//   chunk c (contiguous bags, handed out by a ticket)            512 threads, W lanes per row, 512/W lane groups
//     pass 1   sum (len, cost), min / max len of the chunk  ->  publish ONE status record  ->  every thread polls ONE
//              predecessor's record (<= 512 chunks), block-reduce = the chunk's prefix: one L2 round trip, no chain
//     pass 2   per tile of 512 bags: block scan -> offsets (global + shared), segment records, meta (a1 + a2, bit-exact:
//              the plan stays exportable and reusable by later dpi_lookup calls)
//              cp.async the tile's index entries into shared memory (one coalesced round trip instead of one per bag)
//              pool the tile's bags from shared offsets / indices (a3)
//
// No grid-wide barrier: a chunk waits only for the aggregates of the chunks before it, which every CTA publishes
// before it does anything else. Output-first holds as in the other kernels: consecutive lane groups own
// consecutive bags = consecutive output addresses.
// Pooling per tile: short tiles (longest bag <= kShortTile) give each lane group U bags side by side with up to J entries
// of each in flight; tiles with longer bags give each WARP a bag (sub-warps stride its entries, shuffle-reduce). Static
// chunks are not load-balanced across CTAs, which is why dpi_forward only takes this path when the plan's capacity says
// bags are short on average (max_indices <= 8 * G); everything else runs plan + balanced-segment lookup.
// Same arithmetic as lookup_kernel: fp32 accumulation in entry order, one RNE cast at the store, mean by reciprocal, bags of
// length <= 1 bit-exact, empty bags +0.0.
#include "lookup_kernels.cuh"

namespace dpi {
namespace {

constexpr uint32_t kStateAggregate = 1u;
constexpr int kKeep = 4;            // tiles whose lengths stay in registers between pass 1 and pass 2
constexpr int kShortTile = 16;      // tiles whose longest bag is at most this run the lane-group-per-bag path
constexpr int kFU = 2, kFJ = 4;     // bags side by side per lane group x entries of each in flight

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

template <class Tr, int W, bool OUT32>
__global__ void __launch_bounds__(kFusedThreads, 2) fused_forward_kernel(const FusedArgs a) {
    constexpr int P = 32 / W;
    constexpr int NG = kFusedThreads / W;          // lane groups per CTA
    constexpr int NW = kFusedThreads / 32;         // warps per CTA
    constexpr int kAcc2 = Tr::kAcc / 2;
    constexpr int kOutVec = (OUT32 && Tr::kAcc == 8) ? 32 : 16;
    extern __shared__ const char* s_tab[];         // [T]
    __shared__ int s_off[kFusedThreads + 1];       // offsets of the tile's bags (absolute entry positions)
    __shared__ int s_idx[kFusedIdxStage];          // the tile's index entries (low words for int64 ids)
    __shared__ uint32_t s_w[3][NW];                // per-warp {len, cost, max} exchange
    __shared__ uint32_t s_bcast[4];                // chunk, epoch, prefix len, prefix cost

    const PlanArgs& pa = a.plan;
    const LookupArgs& la = a.look;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    griddep_wait();  // PDL: nothing is read before the preceding grid (e.g. the previous step) has completed
    for (uint32_t t = tid; t < la.T; t += kFusedThreads) s_tab[t] = static_cast<const char*>(la.tables[t]);
    if (tid == 0) {
        s_bcast[0] = atomicInc(pa.state + kStateTicket, pa.num_chunks - 1);
        s_bcast[1] = *reinterpret_cast<volatile unsigned int*>(pa.state + kStateEpoch);
    }
    __syncthreads();
    const uint32_t chunk = s_bcast[0], epoch = s_bcast[1];
    const uint32_t g_lo = chunk * a.chunk_bags;
    const uint32_t g_hi = min(pa.G, g_lo + a.chunk_bags);
    const uint32_t n_tiles = (g_hi - g_lo + kFusedThreads - 1) / kFusedThreads;

    // ---- pass 1: aggregate of the chunk, published at once ----
    uint32_t keep[kKeep];
    uint32_t c_len = 0, c_cost = 0, c_lo = 0xffffffffu, c_hi = 0u;
#pragma unroll
    for (int k = 0; k < kKeep; ++k) {
        const uint32_t g = g_lo + k * kFusedThreads + tid;
        const bool ok = static_cast<uint32_t>(k) < n_tiles && g < g_hi;
        keep[k] = ok ? static_cast<uint32_t>(__ldg(pa.len + g)) : 0u;
        c_len += keep[k];
        c_cost += ok ? max(keep[k], 1u) : 0u;
        if (ok) { c_lo = min(c_lo, keep[k]); c_hi = max(c_hi, keep[k]); }
    }
    for (uint32_t k = kKeep; k < n_tiles; ++k) {
        const uint32_t g = g_lo + k * kFusedThreads + tid;
        if (g < g_hi) {
            const uint32_t l = static_cast<uint32_t>(__ldg(pa.len + g));
            c_len += l; c_cost += max(l, 1u);
            c_lo = min(c_lo, l); c_hi = max(c_hi, l);
        }
    }
    c_len = __reduce_add_sync(0xffffffffu, c_len);
    c_cost = __reduce_add_sync(0xffffffffu, c_cost);
    c_lo = __reduce_min_sync(0xffffffffu, c_lo);
    c_hi = __reduce_max_sync(0xffffffffu, c_hi);
    if (lane == 0) { s_w[0][warp] = c_len; s_w[1][warp] = c_cost; s_w[2][warp] = c_hi; s_off[warp] = static_cast<int>(c_lo); }
    __syncthreads();
    if (tid == 0) {
        uint32_t agg_len = 0, agg_cost = 0, agg_lo = 0xffffffffu, agg_hi = 0u;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            agg_len += s_w[0][w]; agg_cost += s_w[1][w];
            agg_hi = max(agg_hi, s_w[2][w]); agg_lo = min(agg_lo, static_cast<uint32_t>(s_off[w]));
        }
        st_status(pa.status + chunk, pack_status(epoch, kStateAggregate, agg_len), pack_status(epoch, kStateAggregate, agg_cost));
        if (agg_lo <= agg_hi) {
            atomicMin(pa.state + kStateMinLen, agg_lo);
            atomicMax(pa.state + kStateMaxLen, agg_hi);
        }
    }
    // ---- look-back: thread i polls the record of chunk i (all loads of the CTA in flight together) ----
    uint32_t p_len = 0, p_cost = 0;
    if (tid < chunk) {
        ulonglong2 w = ld_status(pa.status + tid);
        while (!(status_ready(w.x, epoch) && status_ready(w.y, epoch))) w = ld_status(pa.status + tid);
        p_len = static_cast<uint32_t>(w.x);
        p_cost = static_cast<uint32_t>(w.y);
    }
    p_len = __reduce_add_sync(0xffffffffu, p_len);
    p_cost = __reduce_add_sync(0xffffffffu, p_cost);
    __syncthreads();   // pass-1 exchange has been consumed by thread 0
    if (lane == 0) { s_w[0][warp] = p_len; s_w[1][warp] = p_cost; }
    __syncthreads();
    uint32_t run_len = 0, run_cost = 0;   // offsets / C at the first bag of the current tile
#pragma unroll
    for (int w = 0; w < NW; ++w) { run_len += s_w[0][w]; run_cost += s_w[1][w]; }
    asm volatile("griddepcontrol.launch_dependents;");

    const uint32_t q = tid / W, sl = tid % W;
    const uint32_t sub = lane / W;
    const bool vec_ok = sl < la.nvec;
    const uint32_t row_bytes = la.nvec * 16;
    const uint32_t ish = la.idx_shift;
    char* const out = static_cast<char*>(la.out);
    auto is_mean = [&](uint32_t t) -> bool { return (la.pool.w[t >> 5] >> (t & 31)) & 1u; };

    // ---- pass 2: scan, plan records and pooling, tile by tile ----
    for (uint32_t k = 0; k < n_tiles; ++k) {
        const uint32_t tile_g0 = g_lo + k * kFusedThreads;
        const uint32_t g = tile_g0 + tid;
        const bool valid = g < g_hi;
        uint32_t l = 0;
        if (k < kKeep) {
#pragma unroll
            for (int kk = 0; kk < kKeep; ++kk) if (static_cast<uint32_t>(kk) == k) l = keep[kk];
        } else if (valid) {
            l = static_cast<uint32_t>(__ldg(pa.len + g));
        }
        const uint32_t cost = valid ? max(l, 1u) : 0u;
        uint32_t i_len = l, i_cost = cost;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t ul = __shfl_up_sync(0xffffffffu, i_len, d);
            const uint32_t uc = __shfl_up_sync(0xffffffffu, i_cost, d);
            if (lane >= static_cast<uint32_t>(d)) { i_len += ul; i_cost += uc; }
        }
        const uint32_t w_max = __reduce_max_sync(0xffffffffu, l);
        __syncthreads();   // previous tile's pooling is done with s_off / s_idx; the look-back exchange has been read
        if (lane == 31) { s_w[0][warp] = i_len; s_w[1][warp] = i_cost; s_w[2][warp] = w_max; }
        __syncthreads();
        uint32_t w_len = 0, w_cost = 0, agg_len = 0, agg_cost = 0, tile_max = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const uint32_t xl = s_w[0][w], xc = s_w[1][w];
            if (static_cast<uint32_t>(w) < warp) { w_len += xl; w_cost += xc; }
            agg_len += xl; agg_cost += xc;
            tile_max = max(tile_max, s_w[2][w]);
        }
        const uint32_t off = run_len + w_len + i_len - l;       // offsets[g]
        const uint32_t c = run_cost + w_cost + i_cost - cost;   // C[g]
        const uint32_t e_lo = run_len, e_hi = run_len + agg_len;  // the tile's index entries
        run_len += agg_len;
        run_cost += agg_cost;
        s_off[tid] = static_cast<int>(off);                     // threads past g_hi carry off == e_hi (l = 0)
        if (tid == 0) s_off[kFusedThreads] = static_cast<int>(e_hi);

        // the tile's index entries -> shared memory, one coalesced pass (issued before the plan records are written)
        const uint32_t ne = e_hi - e_lo;
        const bool staged = ne <= static_cast<uint32_t>(kFusedIdxStage);
        if (staged) {
            const int* src = la.indices + (static_cast<size_t>(e_lo) << ish);
            for (uint32_t i = tid; i < ne; i += kFusedThreads) cp_async4(s_idx + i, src + (static_cast<size_t>(i) << ish));
        }
        cp_async_commit();

        if (valid) {
            // ---- a1: offsets; a2: every quantum boundary s*K inside (C[g], C[g+1]] belongs to bag g -> seg[s] = {g+1, offsets[g+1]}
            pa.offsets[g] = static_cast<int32_t>(off);
            if (g == 0) pa.seg[0] = make_int2(0, 0);
            const uint32_t c1 = c + cost;
            uint32_t s = c / pa.K;
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
                pa.meta[META_S] = (S < pa.seg_cap) ? S : 0;
                pa.meta[META_N] = n_total;
                pa.meta[META_C] = c1;
                const bool overflow = n_total > pa.max_indices || S >= pa.seg_cap;
                pa.meta[META_OVERFLOW] = overflow ? 1 : 0;
                if (overflow) atomicAdd(pa.state + kStateOverflows, 1u);
                pa.meta[META_K] = pa.K;
                pa.meta[META_G] = pa.G;
            }
        }
        cp_async_wait<0>();
        __syncthreads();   // s_off and s_idx are complete

        // ---- a3: pool the tile's bags ----
        const uint32_t nb = min(static_cast<uint32_t>(kFusedThreads), g_hi - tile_g0);
        const int* const sidx = s_idx - e_lo;   // indexed by absolute entry position
        auto idx_at = [&](int e) -> uint32_t {
            return static_cast<uint32_t>(staged ? sidx[e] : __ldg(la.indices + (static_cast<size_t>(e) << ish)));
        };
        if (tile_max <= static_cast<uint32_t>(kShortTile)) {
            const uint32_t t_step = NG % la.T;
            uint32_t t = (tile_g0 + q) % la.T;
            for (uint32_t i0 = q; i0 < nb; i0 += NG * kFU) {
                int lo[kFU], len[kFU];
                uint32_t tt[kFU];
                int max_len = 0;
#pragma unroll
                for (int u = 0; u < kFU; ++u) {
                    const uint32_t i = i0 + u * NG;
                    const bool ok = i < nb;
                    tt[u] = t;
                    lo[u] = ok ? s_off[i] : 0;
                    len[u] = ok ? s_off[i + 1] - lo[u] : 0;
                    max_len = max(max_len, len[u]);
                    t += t_step;
                    if (t >= la.T) t -= la.T;
                }
                float2 acc[kFU][kAcc2];
#pragma unroll
                for (int u = 0; u < kFU; ++u) zero_acc(acc[u]);
                for (int j0 = 0; j0 < max_len; j0 += kFJ) {
                    uint4 v[kFU][kFJ];
#pragma unroll
                    for (int u = 0; u < kFU; ++u) {
#pragma unroll
                        for (int j = 0; j < kFJ; ++j) {
                            const bool ok = vec_ok && j0 + j < len[u];
                            const uint32_t r = ok ? idx_at(lo[u] + j0 + j) : 0u;
                            v[u][j] = ld_row16(s_tab[tt[u]] + static_cast<uint64_t>(r) * row_bytes + sl * 16, ok);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < kFU; ++u) {
#pragma unroll
                        for (int j = 0; j < kFJ; ++j) Tr::add(acc[u], v[u][j]);   // entry order; absent entries add +0.0
                    }
                }
#pragma unroll
                for (int u = 0; u < kFU; ++u) {
                    const uint32_t i = i0 + u * NG;
                    if (vec_ok && i < nb) {
                        if (is_mean(tt[u]) && len[u] > 1) scale_mean(acc[u], len[u]);
                        store_pooled<Tr, OUT32>(out + (static_cast<size_t>(tile_g0 + i) * la.nvec + sl) * kOutVec, acc[u]);
                    }
                }
            }
        } else {
            // a bag per warp: the P sub-warps stride its entries two rounds at a time, partial sums meet by shuffle
            for (uint32_t i = warp; i < nb; i += NW) {
                const int lo = s_off[i], hi = s_off[i + 1];
                const uint32_t t = (tile_g0 + i) % la.T;
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
                    if (is_mean(t) && hi - lo > 1) scale_mean(acc, hi - lo);
                    store_pooled<Tr, OUT32>(out + (static_cast<size_t>(tile_g0 + i) * la.nvec + sl) * kOutVec, acc);
                }
            }
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

template <class Tr, bool OUT32, class F>
auto for_lanes(int lanes, F&& f) {
    switch (lanes) {
        case 1: return f(fused_forward_kernel<Tr, 1, OUT32>);
        case 2: return f(fused_forward_kernel<Tr, 2, OUT32>);
        case 4: return f(fused_forward_kernel<Tr, 4, OUT32>);
        case 8: return f(fused_forward_kernel<Tr, 8, OUT32>);
        case 16: return f(fused_forward_kernel<Tr, 16, OUT32>);
        case 32: return f(fused_forward_kernel<Tr, 32, OUT32>);
        default: return f(static_cast<void (*)(const FusedArgs)>(nullptr));
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

int fused_occupancy(int dtype, bool out32, int lanes, uint32_t T) {
    return for_kernel(dtype, out32, lanes, [&](void (*k)(const FusedArgs)) -> int {
        int occ = 0;
        if (!k || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, kFusedThreads, static_cast<size_t>(T) * sizeof(const char*)) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        return occ;
    });
}

cudaError_t launch_fused(const FusedArgs& a, int dtype, bool out32, int lanes, bool pdl, cudaStream_t stream) {
    return for_kernel(dtype, out32, lanes, [&](void (*k)(const FusedArgs)) -> cudaError_t {
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
