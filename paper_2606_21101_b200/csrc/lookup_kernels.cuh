// lookup_kernels.cuh -- step a3: the fused multi-table gather-and-pool (Alg. 1, generalised
// to CSR bags per PAPER.md:168).  One persistent launch covers every table and every sample.
//
// Mapping (output-first): warp-task s owns the contiguous bags [seg_bag[s], seg_bag[s+1])
// -> adjacent warps own adjacent output addresses, and out[b, t*D + c] == out[g*D + c] for g = b*T + t, so
// the concatenated [B, T*D] block is written once, in place, with no per-table intermediates.
//
// "Anticipate the whole workload": because the plan is complete before the launch, a warp
// never chases task -> offsets -> indices -> rows serially. It runs a two-deep software pipeline:
//     iteration i:   ld  seg records of task i+2                     (registers)
//                    cp.async offsets + indices of task i+1 -> smem   (needs records loaded at i-1)
//                    gather-and-pool task i from smem-staged indices  (only row loads touch DRAM here)
// Measured on B200 (profiles/): without the pipeline the kernel is bound by ~8 dependent DRAM round
// trips per bag (the 4.4 GB row stream evicts the plan from L2) and reaches 52 % of the HBM roofline.
//
// A row is NV = D*sizeof(elt)/16 128-bit vectors; W = pow2ceil(NV) lanes hold one row (lane sl < NV loads
// vector sl), P = 32/W sub-warps per warp.  Three warp-uniform shapes per task:
//   one-hot   (every bag in the task has length 1): pure row copy, P*U rows in flight per warp (Alg. 1)
//   sub-warp  (mean length < 2P): sub-warp q pools bags g_lo+q, g_lo+q+P, ... with U loads in flight per lane
//   warp      (long bags) : all P sub-warps stride the entries of one bag in batches of P*U rows; batches are
//                           double-buffered across batch AND bag boundaries (U..2U loads in flight per lane);
//                           log2(P) __shfl_xor steps combine the partial sums at the end of a bag
// Row loads are branch-free (predicated ld.global.nc.v4) so the U loads of a batch issue back to back.
// fp32 accumulation in registers; one RNE cast at the store (fp16/bf16 output) or fp32 output (OUT32).
#pragma once

#include "dpi_internal.cuh"

namespace dpi {

constexpr int kStageIdx = 256;  // staged index entries per task buffer (tasks with more read global memory)
constexpr int kStageOff = 72;   // staged offsets per task buffer (bags + 1)
constexpr int kWarpStageInts = 2 * kStageIdx + 2 * kStageOff;
constexpr int kLookupMaxThreads = 256;  // natural register allocation (64-80/thread); a 512 bound made ptxas spill

// ---- memory helpers ----------------------------------------------------------------------------------
// Predicated 128-bit read-only load; lanes with pred == false get zeros and issue no memory request. Rows are
// allowed to allocate in L1 (the unified 256 KB L1/smem): on B200 that measured +17 % (c5) and +20 % (c4) over
// ld.global.nc.L1::no_allocate -- the Zipf head of a table is re-read by neighbouring warps of the same SM,
// and with 256 B rows both 128 B lines of a row are requested by one warp-wide load anyway.
__device__ __forceinline__ uint4 ld_row16(const void* p, bool pred) {
    uint4 r = make_uint4(0u, 0u, 0u, 0u);
    asm("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
        "@p ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];\n\t}"
        : "+r"(r.x), "+r"(r.y), "+r"(r.z), "+r"(r.w) : "l"(p), "r"(static_cast<int>(pred)));
    return r;
}
// streaming stores: the output block is consumed by the next layer, not re-read here
__device__ __forceinline__ void st_out16(void* p, const uint4& v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void st_out32(void* p, const float (&f)[8]) {  // sm_100 256-bit store
    asm volatile("st.global.cs.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(f[0]), "f"(f[1]), "f"(f[2]),
                 "f"(f[3]), "f"(f[4]), "f"(f[5]), "f"(f[6]), "f"(f[7]) : "memory");
}
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(static_cast<uint32_t>(__cvta_generic_to_shared(smem_dst))),
                 "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- per-dtype arithmetic ----------------------------------------------------------------------------
// Accumulators are fp32 pairs so that every add is one sm_100 packed add.rn.f32x2 (FADD2): the kernel is
// issue-bound on L2-resident workloads (c3/c4), and FADD2 halves the adds per 16-byte vector.
__device__ __forceinline__ void add2(float2& a, float x, float y) { a = __fadd2_rn(a, make_float2(x, y)); }

struct F32Traits {
    static constexpr int kAcc = 4;   // fp32 accumulators per lane (one 16-byte vector of the row)
    static constexpr int kEltBytes = 4;
    __device__ static __forceinline__ void add(float2 (&acc)[2], const uint4& v) {
        add2(acc[0], __uint_as_float(v.x), __uint_as_float(v.y));
        add2(acc[1], __uint_as_float(v.z), __uint_as_float(v.w));
    }
    __device__ static __forceinline__ uint4 pack(const float2 (&acc)[2]) {
        return make_uint4(__float_as_uint(acc[0].x), __float_as_uint(acc[0].y), __float_as_uint(acc[1].x),
                          __float_as_uint(acc[1].y));
    }
};
struct F16Traits {
    static constexpr int kAcc = 8;
    static constexpr int kEltBytes = 2;
    __device__ static __forceinline__ void add(float2 (&acc)[4], const uint4& v) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
            acc[i] = __fadd2_rn(acc[i], f);
        }
    }
    __device__ static __forceinline__ uint4 pack(const float2 (&acc)[4]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __half2 h = __floats2half2_rn(acc[i].x, acc[i].y);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};
struct BF16Traits {
    static constexpr int kAcc = 8;
    static constexpr int kEltBytes = 2;
    __device__ static __forceinline__ void add(float2 (&acc)[4], const uint4& v) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)  // bf16 -> fp32 is a 16-bit shift (low element) or a mask (high element)
            add2(acc[i], __uint_as_float(w[i] << 16), __uint_as_float(w[i] & 0xffff0000u));
    }
    __device__ static __forceinline__ uint4 pack(const float2 (&acc)[4]) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(acc[i].x, acc[i].y);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

template <int N2>
__device__ __forceinline__ void zero_acc(float2 (&acc)[N2]) {
#pragma unroll
    for (int i = 0; i < N2; ++i) acc[i] = make_float2(0.f, 0.f);
}

// Mean pooling: one IEEE reciprocal of the bag length, then packed multiplies (R8: divide vs
// multiply-by-reciprocal differ by <= 1 ulp of fp32, far inside the tolerance; bags with L <= 1 skip this and
// stay bit-exact). The eight IEEE divisions this replaces cost ~15 instructions each.
template <int N2>
__device__ __forceinline__ void scale_mean(float2 (&acc)[N2], int len) {
    const float inv = __frcp_rn(static_cast<float>(len));
    const float2 inv2 = make_float2(inv, inv);
#pragma unroll
    for (int i = 0; i < N2; ++i) acc[i] = __fmul2_rn(acc[i], inv2);
}

// Store one pooled vector of bag g: table dtype (16 B per lane) or fp32 (OUT32: 32 B per lane for 16-bit tables).
template <class Tr, bool OUT32>
__device__ __forceinline__ void store_pooled(char* out, size_t g, uint32_t nvec, int sl, const float2 (&acc)[Tr::kAcc / 2]) {
    if constexpr (OUT32 && Tr::kAcc == 8) {
        const float f[8] = {acc[0].x, acc[0].y, acc[1].x, acc[1].y, acc[2].x, acc[2].y, acc[3].x, acc[3].y};
        st_out32(out + g * (static_cast<size_t>(nvec) * 32) + sl * 32, f);
    } else {
        st_out16(out + g * (static_cast<size_t>(nvec) * 16) + sl * 16, Tr::pack(acc));
    }
}

// U = 2 (the default: double buffering makes it 2..4 row loads in flight per lane) is held to 64 registers so
// that 4 CTAs = 32 warps stay resident per SM for every dtype (ptxas: 0-24 bytes of spill, all on cold paths);
// the deeper unrolls keep their natural allocation (<= 80 registers, 3 CTAs).
template <class Tr, int W, int U, bool OUT32>
__global__ void __launch_bounds__(kLookupMaxThreads, U <= 2 ? 4 : 1) lookup_kernel(const LookupArgs a) {
    constexpr int P = 32 / W;
    constexpr int kAcc = Tr::kAcc;
    constexpr int kAcc2 = kAcc / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int lane = threadIdx.x & 31;
    const int sub = lane / W;
    const int sl = lane % W;
    const bool vec_ok = static_cast<uint32_t>(sl) < a.nvec;
    const uint32_t warps_per_cta = blockDim.x >> 5;
    const uint32_t n_warps = gridDim.x * warps_per_cta;
    const uint32_t warp_in_cta = threadIdx.x >> 5;
    const uint32_t warp_id = blockIdx.x * warps_per_cta + warp_in_cta;
    const size_t row_bytes = static_cast<size_t>(a.nvec) * 16;
    char* const out = static_cast<char*>(a.out);

    // smem: [T table base pointers][per warp: idx stage x2, offsets stage x2]
    const char** s_tab = reinterpret_cast<const char**>(smem_raw);
    int* const s_warp = reinterpret_cast<int*>(smem_raw + ((static_cast<size_t>(a.T) * 8 + 15) & ~static_cast<size_t>(15))) +
                        warp_in_cta * kWarpStageInts;
    for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) s_tab[t] = static_cast<const char*>(a.tables[t]);
    __syncthreads();

    griddep_wait();  // PDL: the planner's writes are visible past this point (no-op otherwise)
    const uint32_t S = static_cast<uint32_t>(a.meta[META_S]);
    if (warp_id >= S) return;

    // Stage offsets[g_lo..g_hi] and indices[e_lo..e_hi) of one task into buffer `b` (if they fit).
    auto stage = [&](const int2 r_lo, const int2 r_hi, int b) {
        const int nb1 = r_hi.x - r_lo.x + 1, ne = r_hi.y - r_lo.y;
        if (r_hi.x > r_lo.x && nb1 <= kStageOff && ne <= kStageIdx) {
            int* ib = s_warp + b * kStageIdx;
            int* ob = s_warp + 2 * kStageIdx + b * kStageOff;
            for (int i = lane; i < ne; i += 32) cp_async4(ib + i, a.indices + r_lo.y + i);
            for (int i = lane; i < nb1; i += 32) cp_async4(ob + i, a.offsets + r_lo.x + i);
        }
        cp_async_commit();
    };

    // ---- pipeline prologue ----
    uint32_t s = warp_id;
    int2 cur_lo = __ldg(a.seg + s), cur_hi = __ldg(a.seg + s + 1);
    int2 nxt_lo = cur_lo, nxt_hi = cur_hi;
    bool have_next = s + n_warps < S;
    if (have_next) { nxt_lo = __ldg(a.seg + s + n_warps); nxt_hi = __ldg(a.seg + s + n_warps + 1); }
    stage(cur_lo, cur_hi, 0);
    int buf = 0;

    for (;;) {
        // ---- prefetch: records two tasks ahead, offsets + indices one task ahead ----
        const uint32_t s2 = s + 2 * n_warps;
        const bool have_next2 = s2 < S;
        int2 n2_lo = nxt_lo, n2_hi = nxt_hi;
        if (have_next2) { n2_lo = __ldg(a.seg + s2); n2_hi = __ldg(a.seg + s2 + 1); }
        if (have_next) {
            stage(nxt_lo, nxt_hi, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncwarp();

        const uint32_t g_lo = cur_lo.x, g_hi = cur_hi.x;
        if (g_lo < g_hi) {  // a long bag spanning several quanta leaves empty tasks behind it
            const uint32_t nb = g_hi - g_lo;
            const int e_lo = cur_lo.y, e_hi = cur_hi.y;
            const uint32_t ne = static_cast<uint32_t>(e_hi - e_lo);
            const bool staged = (nb + 1 <= static_cast<uint32_t>(kStageOff)) && (ne <= static_cast<uint32_t>(kStageIdx));
            // generic pointers indexed by ABSOLUTE entry / bag id: staged smem or the global arrays
            const int* ip = staged ? (s_warp + buf * kStageIdx - e_lo) : a.indices;
            const int* op = staged ? (s_warp + 2 * kStageIdx + buf * kStageOff - static_cast<int>(g_lo)) : a.offsets;

            bool onehot = false;
            if (ne == nb && a.mode != 2) {
                // a task with ne == nb could still mix empty and longer bags: verify
                bool all_one = true;
                for (uint32_t i = lane; i < nb; i += 32) all_one &= (op[g_lo + i + 1] - op[g_lo + i]) == 1;
                onehot = __all_sync(0xffffffffu, all_one);
            }
            if (onehot) {
                // ---------------- one-hot task: Alg. 1, a pure row copy (bit-exact) ------------------------
                for (uint32_t i0 = 0; i0 < nb; i0 += P * U) {
                    uint4 v[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        const bool ok = i < nb;
                        const uint32_t g = g_lo + (ok ? i : 0u);
                        const int r = ip[e_lo + (ok ? i : 0u)];
                        v[u] = ld_row16(s_tab[g % a.T] + sl * 16 + static_cast<size_t>(r) * row_bytes, ok && vec_ok);
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        if (i < nb && vec_ok) {
                            if constexpr (OUT32 && kAcc == 8) {
                                float2 f[kAcc2];
                                zero_acc(f);
                                Tr::add(f, v[u]);
                                store_pooled<Tr, OUT32>(out, g_lo + i, a.nvec, sl, f);
                            } else {
                                st_out16(out + static_cast<size_t>(g_lo + i) * row_bytes + sl * 16, v[u]);
                            }
                        }
                    }
                }
            } else if (a.mode == 1 || (a.mode == 0 && ne < 2u * (P == 1 ? U : P) * nb)) {
                // ---------------- sub-warp per bag (short bags) ---------------------------------------------
                for (uint32_t g0 = g_lo; g0 < g_hi; g0 += P) {
                    const uint32_t g = g0 + sub;
                    const bool active = g < g_hi;
                    const uint32_t gc = active ? g : g_lo;
                    const int lo = op[gc];
                    const int hi = active ? op[gc + 1] : lo;
                    const uint32_t t = gc % a.T;
                    const char* tab = s_tab[t] + sl * 16;
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    for (int j = lo; j < hi; j += U) {
                        uint4 v[U];
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            const bool ok = j + u < hi;
                            const int r = ip[ok ? j + u : lo];
                            v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, ok && vec_ok);
                        }
#pragma unroll
                        for (int u = 0; u < U; ++u) Tr::add(acc, v[u]);
                    }
                    if (active && vec_ok) {
                        if (((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                        store_pooled<Tr, OUT32>(out, g, a.nvec, sl, acc);
                    }
                }
            } else if (a.mode == 2) {
                // ---------------- whole warp per bag, one batch at a time (kept for A/B measurements) ------
                for (uint32_t g = g_lo; g < g_hi; ++g) {
                    const int lo = op[g], hi = op[g + 1];
                    const uint32_t t = g % a.T;
                    const char* tab = s_tab[t] + sl * 16;
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    for (int j = lo; j < hi; j += P * U) {
                        uint4 v[U];
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            const int e = j + u * P + sub;
                            const bool ok = e < hi;
                            const int r = ip[ok ? e : lo];
                            v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, ok && vec_ok);
                        }
#pragma unroll
                        for (int u = 0; u < U; ++u) Tr::add(acc, v[u]);
                    }
#pragma unroll
                    for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                        for (int i = 0; i < kAcc2; ++i)
                            acc[i] = __fadd2_rn(acc[i], make_float2(__shfl_xor_sync(0xffffffffu, acc[i].x, d),
                                                                    __shfl_xor_sync(0xffffffffu, acc[i].y, d)));
                    }
                    if (sub == 0 && vec_ok) {
                        if (((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                        store_pooled<Tr, OUT32>(out, g, a.nvec, sl, acc);
                    }
                }
            } else {
                // ---------------- whole warp per bag, double-buffered batches (long bags) -------------------
                // The loads of batch k+1 (possibly the first batch of the NEXT bag: its offsets and indices
                // are already in smem) are issued before batch k is consumed, so a warp keeps U..2U row
                // loads per lane in flight across batch and bag boundaries instead of draining at each one.
                auto store_zero = [&](uint32_t gz) {
                    if (sub == 0 && vec_ok) {
                        float2 z[kAcc2];
                        zero_acc(z);
                        store_pooled<Tr, OUT32>(out, gz, a.nvec, sl, z);
                    }
                };
                auto issue = [&](uint4 (&v)[U], int j, int hi, const char* tab) {
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int e = j + u * P + sub;
                        const bool ok = e < hi;
                        const int r = ip[ok ? e : j];
                        v[u] = ld_row16(tab + static_cast<size_t>(r) * row_bytes, ok && vec_ok);
                    }
                };
                uint32_t g = g_lo;
                int lo = op[g], hi = op[g + 1];
                while (hi == lo) {  // leading empty bags
                    store_zero(g);
                    if (++g == g_hi) break;
                    lo = hi;
                    hi = op[g + 1];
                }
                if (g < g_hi) {
                    int j = lo;
                    const char* tab = s_tab[g % a.T] + sl * 16;
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    uint4 vA[U], vB[U];
                    issue(vA, j, hi, tab);
                    bool more = true;
                    auto step = [&](uint4 (&cv)[U], uint4 (&nv)[U]) {
                        uint32_t g_n = g;
                        int j_n = j + P * U, lo_n = lo, hi_n = hi;
                        const char* tab_n = tab;
                        const bool last_of_bag = j_n >= hi;
                        bool has_next = true;
                        if (last_of_bag) {
                            g_n = g + 1;
                            for (;;) {
                                if (g_n == g_hi) { has_next = false; break; }
                                lo_n = hi_n;
                                hi_n = op[g_n + 1];
                                if (hi_n > lo_n) break;
                                store_zero(g_n);
                                ++g_n;
                            }
                            if (has_next) { j_n = lo_n; tab_n = s_tab[g_n % a.T] + sl * 16; }
                        }
                        if (has_next) issue(nv, j_n, hi_n, tab_n);
#pragma unroll
                        for (int u = 0; u < U; ++u) Tr::add(acc, cv[u]);
                        if (last_of_bag) {
#pragma unroll
                            for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                                for (int i = 0; i < kAcc2; ++i)
                                    acc[i] = __fadd2_rn(acc[i], make_float2(__shfl_xor_sync(0xffffffffu, acc[i].x, d),
                                                                            __shfl_xor_sync(0xffffffffu, acc[i].y, d)));
                            }
                            if (sub == 0 && vec_ok) {
                                const uint32_t t = g % a.T;
                                if (((a.pool.w[t >> 5] >> (t & 31)) & 1u) && hi - lo > 1) scale_mean(acc, hi - lo);
                                store_pooled<Tr, OUT32>(out, g, a.nvec, sl, acc);
                            }
                            zero_acc(acc);
                        }
                        g = g_n; j = j_n; lo = lo_n; hi = hi_n; tab = tab_n;
                        more = has_next;
                    };
                    while (more) {
                        step(vA, vB);
                        if (!more) break;
                        step(vB, vA);
                    }
                }
            }
        }

        if (!have_next) break;
        __syncwarp();  // every lane is done with buffer `buf` before the next iteration refills it
        s += n_warps;
        cur_lo = nxt_lo; cur_hi = nxt_hi;
        nxt_lo = n2_lo; nxt_hi = n2_hi;
        have_next = have_next2;
        buf ^= 1;
    }
}

// ---- host-side dispatch (one translation unit per dtype keeps nvcc parallel) ------------------------------
inline size_t lookup_smem_bytes(uint32_t T, int block_threads) {
    return ((static_cast<size_t>(T) * 8 + 15) & ~static_cast<size_t>(15)) +
           static_cast<size_t>(block_threads / 32) * kWarpStageInts * sizeof(int);
}

template <class Tr, int W, int U, bool OUT32>
cudaError_t launch_one(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream) {
    const size_t smem = lookup_smem_bytes(a.T, l.block_threads);
    static size_t smem_set = 0;  // per instantiation: raise the dynamic smem limit once (or when it grows)
    if (smem > 48 * 1024 && smem > smem_set) {
        cudaError_t e = cudaFuncSetAttribute(lookup_kernel<Tr, W, U, OUT32>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(smem));
        if (e != cudaSuccess) return e;
        smem_set = smem;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(static_cast<unsigned>(l.grid));
    cfg.blockDim = dim3(static_cast<unsigned>(l.block_threads));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = l.pdl ? 1 : 0;
    count_launch();
    return cudaLaunchKernelEx(&cfg, lookup_kernel<Tr, W, U, OUT32>, a);
}

template <class Tr, int W, int U, bool OUT32>
int occupancy_one(uint32_t T, int block_threads) {
    int n = 0;
    const size_t smem = lookup_smem_bytes(T, block_threads);
    if (smem > 48 * 1024)
        (void)cudaFuncSetAttribute(lookup_kernel<Tr, W, U, OUT32>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, lookup_kernel<Tr, W, U, OUT32>, block_threads, smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

#define DPI_FOR_EACH_U(M, W) M(W, 2) M(W, 4) M(W, 8) M(W, 16)
#define DPI_FOR_EACH_WU(M) \
    DPI_FOR_EACH_U(M, 1) DPI_FOR_EACH_U(M, 2) DPI_FOR_EACH_U(M, 4) DPI_FOR_EACH_U(M, 8) DPI_FOR_EACH_U(M, 16) \
    DPI_FOR_EACH_U(M, 32)
// Each lookup_<dtype>.cu defines DPI_TRAITS / DPI_SUFFIX (/ DPI_HAS_OUT32) and includes lookup_dispatch.inc.

}  // namespace dpi
