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
// The sm_100 256-bit form of the same load (LDG.E.256): one lane holds 32 bytes of the row, so a row needs half the lanes,
// a warp holds twice the rows per load instruction and the index reads / address arithmetic per gathered byte halve
// (DESIGN.md 7.2.2). Needs 32-byte aligned rows: row size a multiple of 32 B and 32-byte aligned table bases.
struct Row32 {
    uint4 lo, hi;
};
__device__ __forceinline__ Row32 ld_row32(const void* p, bool pred) {
    Row32 r;
    r.lo = make_uint4(0u, 0u, 0u, 0u);
    r.hi = make_uint4(0u, 0u, 0u, 0u);
    asm("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %9, 0;\n\t"
        "@p ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"
        : "+r"(r.lo.x), "+r"(r.lo.y), "+r"(r.lo.z), "+r"(r.lo.w), "+r"(r.hi.x), "+r"(r.hi.y), "+r"(r.hi.z), "+r"(r.hi.w)
        : "l"(p), "r"(static_cast<int>(pred)));
    return r;
}
// The same loads without a predicate (and so without zero-initialised destination registers): for batches whose every entry
// exists and rows that fill every lane of their lane group.
__device__ __forceinline__ uint4 ld_row16_all(const void* p) {
    uint4 r;
    asm("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ Row32 ld_row32_all(const void* p) {
    Row32 r;
    asm("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=r"(r.lo.x), "=r"(r.lo.y), "=r"(r.lo.z), "=r"(r.lo.w), "=r"(r.hi.x), "=r"(r.hi.y), "=r"(r.hi.z), "=r"(r.hi.w) : "l"(p));
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
__device__ __forceinline__ void st_row(void* p, const uint4& v) { st_out16(p, v); }
__device__ __forceinline__ void st_row(void* p, const Row32& v) {
    asm volatile("st.global.cs.v8.u32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v.lo.x), "r"(v.lo.y), "r"(v.lo.z), "r"(v.lo.w),
                 "r"(v.hi.x), "r"(v.hi.y), "r"(v.hi.z), "r"(v.hi.w) : "memory");
}
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Plan data (segments, offsets, meta) is written by the planner grid this kernel may have been launched under (PDL), so
// it is never read through the non-coherent path (ld.global.nc assumes read-only for the kernel's lifetime): L2 loads.
__device__ __forceinline__ int2 ld_plan(const int2* p) { return __ldcg(p); }
__device__ __forceinline__ int ld_plan(const int32_t* p) { return __ldcg(p); }
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
    static constexpr int kDtype = DPI_F32;
    static constexpr int kVecBytes = 16;  // bytes of a row held by one lane
    using Row = uint4;
    __device__ static __forceinline__ Row load(const void* p, bool pred) { return ld_row16(p, pred); }
    __device__ static __forceinline__ Row load_all(const void* p) { return ld_row16_all(p); }
    static constexpr int kAcc = 4;   // fp32 accumulators per lane (one 16-byte vector of the row)
    static constexpr int kEltBytes = 4;
    __device__ static __forceinline__ void add(float2 (&acc)[2], const uint4& v) {
        add2(acc[0], __uint_as_float(v.x), __uint_as_float(v.y));
        add2(acc[1], __uint_as_float(v.z), __uint_as_float(v.w));
    }
    __device__ static __forceinline__ void fma(float2 (&acc)[2], const uint4& v, const float2 w) {
        acc[0] = __ffma2_rn(make_float2(__uint_as_float(v.x), __uint_as_float(v.y)), w, acc[0]);
        acc[1] = __ffma2_rn(make_float2(__uint_as_float(v.z), __uint_as_float(v.w)), w, acc[1]);
    }
    __device__ static __forceinline__ uint4 pack(const float2 (&acc)[2]) {
        return make_uint4(__float_as_uint(acc[0].x), __float_as_uint(acc[0].y), __float_as_uint(acc[1].x),
                          __float_as_uint(acc[1].y));
    }
};
struct F16Traits {
    static constexpr int kDtype = DPI_F16;
    static constexpr int kVecBytes = 16;  // bytes of a row held by one lane
    using Row = uint4;
    __device__ static __forceinline__ Row load(const void* p, bool pred) { return ld_row16(p, pred); }
    __device__ static __forceinline__ Row load_all(const void* p) { return ld_row16_all(p); }
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
    __device__ static __forceinline__ void fma(float2 (&acc)[4], const uint4& v, const float2 wt) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
            acc[i] = __ffma2_rn(__half22float2(*reinterpret_cast<const __half2*>(&w[i])), wt, acc[i]);
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
    static constexpr int kDtype = DPI_BF16;
    static constexpr int kVecBytes = 16;  // bytes of a row held by one lane
    using Row = uint4;
    __device__ static __forceinline__ Row load(const void* p, bool pred) { return ld_row16(p, pred); }
    __device__ static __forceinline__ Row load_all(const void* p) { return ld_row16_all(p); }
    static constexpr int kAcc = 8;
    static constexpr int kEltBytes = 2;
    __device__ static __forceinline__ void add(float2 (&acc)[4], const uint4& v) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)  // bf16 -> fp32 is a 16-bit shift (low element) or a mask (high element)
            add2(acc[i], __uint_as_float(w[i] << 16), __uint_as_float(w[i] & 0xffff0000u));
    }
    __device__ static __forceinline__ void fma(float2 (&acc)[4], const uint4& v, const float2 wt) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
            acc[i] = __ffma2_rn(make_float2(__uint_as_float(w[i] << 16), __uint_as_float(w[i] & 0xffff0000u)), wt, acc[i]);
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

// 32 bytes of the row per lane (256-bit loads): two halves of the base type side by side, element order preserved.
template <class Base>
struct Wide {
    static constexpr int kDtype = Base::kDtype;
    static constexpr int kAcc = 2 * Base::kAcc;
    static constexpr int kEltBytes = Base::kEltBytes;
    static constexpr int kVecBytes = 32;
    static constexpr int kH = Base::kAcc / 2;   // float2 accumulators per half
    using Row = Row32;
    using Half = float2 (&)[kH];
    using CHalf = const float2 (&)[kH];
    __device__ static __forceinline__ Row load(const void* p, bool pred) { return ld_row32(p, pred); }
    __device__ static __forceinline__ Row load_all(const void* p) { return ld_row32_all(p); }
    __device__ static __forceinline__ void add(float2 (&acc)[2 * kH], const Row32& v) {
        Base::add(reinterpret_cast<Half>(acc[0]), v.lo);
        Base::add(reinterpret_cast<Half>(acc[kH]), v.hi);
    }
    __device__ static __forceinline__ void fma(float2 (&acc)[2 * kH], const Row32& v, const float2 w) {
        Base::fma(reinterpret_cast<Half>(acc[0]), v.lo, w);
        Base::fma(reinterpret_cast<Half>(acc[kH]), v.hi, w);
    }
    __device__ static __forceinline__ Row32 pack(const float2 (&acc)[2 * kH]) {
        Row32 r;
        r.lo = Base::pack(reinterpret_cast<CHalf>(acc[0]));
        r.hi = Base::pack(reinterpret_cast<CHalf>(acc[kH]));
        return r;
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

// Store one pooled vector (kVecBytes of table-dtype elements, or twice that in fp32 for OUT32 with 16-bit tables) at p.
template <class Tr, bool OUT32>
__device__ __forceinline__ void store_pooled(char* p, const float2 (&acc)[Tr::kAcc / 2]) {
    if constexpr (OUT32 && Tr::kEltBytes == 2) {
#pragma unroll
        for (int i = 0; i < Tr::kAcc / 8; ++i) {
            const float f[8] = {acc[4 * i].x, acc[4 * i].y, acc[4 * i + 1].x, acc[4 * i + 1].y,
                                acc[4 * i + 2].x, acc[4 * i + 2].y, acc[4 * i + 3].x, acc[4 * i + 3].y};
            st_out32(p + 32 * i, f);
        }
    } else {
        st_row(p, Tr::pack(acc));
    }
}
template <class Tr, bool OUT32>
__host__ __device__ constexpr int out_vec_bytes() { return (OUT32 && Tr::kEltBytes == 2) ? 2 * Tr::kVecBytes : Tr::kVecBytes; }

// ---- short-bag body (a3 variant) -------------------------------------------------------------
// Algorithm 1's division of labour (every thread fills its own piece of the output matrix, no shared
// control flow) carried over to CSR bags: lane group q (W lanes = one row) of n_groups owns bags q, q + n_groups, ...; for
// each it reads offsets[g], offsets[g+1] straight from the plan (a1), gathers and pools the bag's rows in registers and
// stores the pooled vector; U bags per lane group are processed side by side (independent chains). No segments, no
// staging, no per-task pipeline. Shared by direct_kernel (chosen on the host from DPI_OPT_MAX_BAG_HINT / DPI_OPT_MODE = 6)
// and by lookup_kernel, which branches here when a1's max_len says every bag is short (no promise needed).
// Same arithmetic as the balanced-segment path: fp32 accumulation in entry order, one RNE cast at the store, mean by
// reciprocal, bags of length <= 1 bit-exact, empty bags +0.0. Dense layout only; int64 ids through their low words.
template <class Tr, int W, int U, bool OUT32>
__device__ __forceinline__ void short_bag_body(const LookupArgs& a, const char* const* s_tab, uint32_t q, uint32_t sl,
                                               uint32_t n_groups) {
    constexpr int kAcc2 = Tr::kAcc / 2;
    constexpr int kVB = Tr::kVecBytes;
    constexpr int kOutVec = out_vec_bytes<Tr, OUT32>();
    const bool vec_ok = sl < a.nvec;
    const uint32_t row_bytes = a.nvec * kVB;
    const uint32_t t_step = n_groups % a.T;
    char* const out = static_cast<char*>(a.out);
    uint32_t t = q % a.T;
    for (uint32_t g0 = q; g0 < a.G; g0 += n_groups * U) {
        int lo[U], len[U];
        uint32_t tt[U];
        int max_len = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            const bool ok = g < a.G;
            tt[u] = t;
            lo[u] = ok ? __ldcg(a.offsets + g) : 0;          // plan data: coherent (L2) loads, see ld_plan()
            len[u] = ok ? __ldcg(a.offsets + g + 1) - lo[u] : 0;
            max_len = max(max_len, len[u]);
            t += t_step;
            if (t >= a.T) t -= a.T;
        }
        float2 acc[U][kAcc2];
#pragma unroll
        for (int u = 0; u < U; ++u) zero_acc(acc[u]);
        for (int j = 0; j < max_len; ++j) {
            typename Tr::Row v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool ok = vec_ok && j < len[u];
                // int64 ids are read through their low words (little-endian, rows < 2^31): idx_shift = 1
                const uint32_t r = ok ? static_cast<uint32_t>(__ldg(a.indices + (static_cast<size_t>(lo[u] + j) << a.idx_shift))) : 0u;
                v[u] = Tr::load(s_tab[tt[u]] + static_cast<uint64_t>(r) * row_bytes + sl * kVB, ok);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) Tr::add(acc[u], v[u]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t g = g0 + u * n_groups;
            if (vec_ok && g < a.G) {
                if (((a.pool.w[tt[u] >> 5] >> (tt[u] & 31)) & 1u) && len[u] > 1) scale_mean(acc[u], len[u]);
                store_pooled<Tr, OUT32>(out + (static_cast<size_t>(g) * a.nvec + sl) * kOutVec, acc[u]);
            }
        }
    }
}

// The offsets of a task as the kernel reads them. Plain layout: an int array indexed by bag id, values = absolute entry
// positions. General variant with int64 offsets (NEXT-2, DESIGN.md 11.2 V6): only the LOW words are read (stride 2) and every
// value is rebased to the task's first entry -- inside a task all positions are < 2^32 apart, so the difference of the low
// words is exact -- and the 64-bit part enters once per task, in the base pointer of its index run (seg_off64).
template <bool GEN>
struct OffView {
    const int* p;
    int sh;            // GEN: 1 when p walks the low words of int64 offsets
    uint32_t rebase;   // GEN: low word of the task's first entry when positions are task-relative, else 0
    __device__ __forceinline__ int operator[](ptrdiff_t g) const {
        if constexpr (GEN) return static_cast<int>(static_cast<uint32_t>(p[g << sh]) - rebase);
        else return p[g];
    }
};

// Per-table record of the general (GEN) variant, staged in shared memory.
struct TableInfo {
    const char* base;
    uint32_t nvec;     // 16-byte vectors per row of this table
    uint32_t col_vec;  // first output vector of this table's column block = sum of nvec over earlier tables
};

// One bag as the kernel sees it: where its rows come from and where its pooled vector goes.
struct BagRef {
    const char* tab;   // table base + this lane's 16-byte slot
    char* outp;        // GEN only: this lane's output slot (the dense layout recomputes it from g at the store)
    uint32_t t;
    uint32_t row_bytes;
    bool ok;           // this lane holds a vector of the row
};

// U = 2 (the default: double buffering makes it 2..4 row loads in flight per lane) is held to 64 registers so
// that 4 CTAs = 32 warps stay resident per SM for every dtype (ptxas: 0-24 bytes of spill, all on cold paths);
// the deeper unrolls keep their natural allocation (<= 80 registers, 3 CTAs).
//
// GEN = false is the path of BASELINE.json's configs: one D, int32 ids, sample-major bags, dense [B, T*D] block.
// GEN = true adds the interface variants of SURVEY.md §8(f) NEXT-2 / NEXT-3 (dpi_lookup_ex): per-table dims,
// int64 ids (the low word is read: rows < 2^31), per-entry fp32 weights (acc = fma(w, row, acc)), table-major
// bags (g = t*B + b) and an output row pitch, so a column block can be written into a wider row.
// Resident CTAs per SM the register allocation is held to: 32 bytes of row per load batch and lane (U = 2 x 128-bit, or
// U = 1 x 256-bit) fit 64 registers = 4 CTAs; U = 2 x 256-bit gets 80 registers = 3 CTAs; deeper unrolls stay natural.
template <class Tr, int U, bool GEN>
__host__ __device__ constexpr int lookup_min_ctas() {
    if (GEN) return U <= 2 ? 3 : 1;
    if (Tr::kVecBytes == 32) return U == 1 ? 4 : (U == 2 ? 3 : 1);
    return U <= 2 ? 4 : 1;
}

template <class Tr, int W, int U, bool OUT32, bool GEN>
__global__ void __launch_bounds__(kLookupMaxThreads, lookup_min_ctas<Tr, U, GEN>()) lookup_kernel(const LookupArgs a) {
    constexpr int P = 32 / W;
    constexpr int kAcc = Tr::kAcc;
    constexpr int kAcc2 = kAcc / 2;
    constexpr int kVB = Tr::kVecBytes;                       // row bytes per lane
    constexpr int kOutVec = out_vec_bytes<Tr, OUT32>();      // output bytes per lane
    static_assert(!GEN || kVB == 16, "the general variant keeps per-table widths in 16-byte vectors");
    using Row = typename Tr::Row;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int lane = threadIdx.x & 31;
    const int sub = lane / W;
    const int sl = lane % W;
    const bool vec_ok = static_cast<uint32_t>(sl) < a.nvec;
    const uint32_t warps_per_cta = blockDim.x >> 5;
    const uint32_t n_warps = gridDim.x * warps_per_cta;
    const uint32_t warp_in_cta = threadIdx.x >> 5;
    const uint32_t warp_id = blockIdx.x * warps_per_cta + warp_in_cta;
    const uint32_t row_bytes_u = a.nvec * kVB;  // non-GEN: every table
    char* const out = static_cast<char*>(a.out);

    // smem: [per-table records][per warp: idx stage x2, offsets stage x2, (GEN) weight stage x2]
    const int ish = GEN ? static_cast<int>(a.idx_shift) : 0;
    const int stage_idx = kStageIdx << ish;  // 32-bit words per index buffer
    const char** s_tab = reinterpret_cast<const char**>(smem_raw);
    const TableInfo* s_info = reinterpret_cast<const TableInfo*>(smem_raw);
    const size_t tab_bytes = GEN ? static_cast<size_t>(a.T) * sizeof(TableInfo)
                                 : ((static_cast<size_t>(a.T) * 8 + 15) & ~static_cast<size_t>(15));
    const int warp_words = 2 * stage_idx + 2 * kStageOff + ((GEN && a.weights) ? 2 * kStageIdx : 0);
    int* const s_warp = reinterpret_cast<int*>(smem_raw + tab_bytes) + warp_in_cta * warp_words;
    int* const s_off = s_warp + 2 * stage_idx;
    float* const s_wgt = reinterpret_cast<float*>(s_off + 2 * kStageOff);
    // PDL: everything this kernel reads (table pointers included -- a preceding kernel may have produced them) is read
    // after the preceding grid has completed and flushed; only the launch itself and the index arithmetic above overlap
    // its tail. No-op for a plain launch.
    griddep_wait();
    if constexpr (GEN) {
        TableInfo* w_info = reinterpret_cast<TableInfo*>(smem_raw);
        for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) {
            TableInfo ti;
            ti.base = static_cast<const char*>(a.tables[t]);
            ti.nvec = a.tab_nvec[t];
            ti.col_vec = a.tab_col[t];
            w_info[t] = ti;
        }
    } else {
        const char** w_tab = reinterpret_cast<const char**>(smem_raw);
        for (uint32_t t = threadIdx.x; t < a.T; t += blockDim.x) w_tab[t] = static_cast<const char*>(a.tables[t]);
    }
    __syncthreads();

    const uint32_t S = static_cast<uint32_t>(ld_plan(a.meta + META_S));
    if constexpr (!GEN) {
        // The device picks the a3 variant from a1's max_len ("known in advance"): a batch
        // whose longest bag is short runs the lane-group-per-bag body over the same persistent grid -- no promise from
        // the caller, no extra launch. S == 0 marks an overflowed plan: nothing may be read through its offsets.
        if (a.mode == 0 && S != 0 && short_bag_rule(static_cast<uint32_t>(ld_plan(a.meta + META_MAXLEN)), a.G)) {
            const uint32_t lane_id = blockIdx.x * blockDim.x + threadIdx.x;
            short_bag_body<Tr, W, 2, OUT32>(a, s_tab, lane_id / W, lane_id % W, (gridDim.x * blockDim.x) / W);
            return;
        }
    }
    if (warp_id >= S) return;

    // bag id -> table, rows, output slot
    auto bag_ref = [&](uint32_t g) -> BagRef {
        BagRef r;
        if constexpr (GEN) {
            uint32_t b;
            if (a.table_major) { r.t = g / a.B; b = g - r.t * a.B; }
            else { b = g / a.T; r.t = g - b * a.T; }
            const TableInfo ti = s_info[r.t];
            r.tab = ti.base + sl * kVB;
            r.row_bytes = ti.nvec * kVB;
            r.ok = static_cast<uint32_t>(sl) < ti.nvec;
            char* row0 = out;
            if (a.peer_out) {  // fused all-to-all: sample b lives on peer b / rows_per_peer (NEXT-3)
                const uint32_t pr = b / a.rows_per_peer;
                b -= pr * a.rows_per_peer;
                row0 = reinterpret_cast<char*>(__ldg(reinterpret_cast<const unsigned long long*>(a.peer_out) + pr));
            }
            r.outp = row0 + static_cast<size_t>(b) * a.out_pitch + static_cast<size_t>(ti.col_vec) * kOutVec + sl * kOutVec;
        } else {
            r.t = g % a.T;
            r.tab = s_tab[r.t] + sl * kVB;
            r.row_bytes = row_bytes_u;
            r.ok = vec_ok;
            r.outp = nullptr;
        }
        return r;
    };
    // bag g_new > g_prev given the reference of g_prev: the dense layout steps the table id instead of dividing again
    // (a 32-bit modulo by a run-time T is ~20 instructions, once per bag on the long-bag path)
    auto bag_ref_next = [&](const BagRef& prev, uint32_t g_prev, uint32_t g_new) -> BagRef {
        if constexpr (GEN) {
            return bag_ref(g_new);
        } else {
            BagRef r = prev;
            uint32_t t = prev.t + (g_new - g_prev);
            if (t >= a.T) {
                t -= a.T;
                if (t >= a.T) t %= a.T;  // only after a run of >= T empty bags
            }
            r.t = t;
            r.tab = s_tab[t] + sl * kVB;
            return r;
        }
    };
    auto out_of = [&](uint32_t g, const BagRef& r) -> char* {
        if constexpr (GEN) return r.outp;
        else return out + static_cast<size_t>(g) * (static_cast<size_t>(a.nvec) * kOutVec) + sl * kOutVec;
    };
    // row ids are non-negative (precondition, dpi.h): read as uint32 so that id * row_bytes is one IMAD.WIDE.U32
    auto idx_at = [&](const int* ip, int e) -> uint32_t {
        return static_cast<uint32_t>(GEN ? ip[static_cast<ptrdiff_t>(e) << ish] : ip[e]);  // 64-bit: e may reach 2^30 with int64 ids
    };
    auto wgt_at = [&](const float* wp, int e) -> float { return (GEN && wp) ? wp[e] : 1.f; };
    auto accum = [&](float2 (&acc)[kAcc2], const Row& v, float w) {
        if constexpr (GEN) Tr::fma(acc, v, make_float2(w, w));  // fma(x, 1, acc) == x + acc exactly
        else Tr::add(acc, v);
    };
    auto is_mean = [&](uint32_t t) -> bool { return (a.pool.w[t >> 5] >> (t & 31)) & 1u; };

    // Stage offsets[g_lo..g_hi] and indices[e_lo..e_hi) (and weights) of one task into buffer `b` (if they fit).
    const int osh = GEN ? static_cast<int>(a.off_shift) : 0;   // 1: int64 offsets, the low words are read
    // first entry of task s as a 64-bit position: seg[s].y, or seg_off64[s] when the offsets are 64-bit
    auto task_base = [&](uint32_t s_, const int2 r_lo) -> long long {
        if constexpr (GEN) { if (osh) return a.seg_off64[s_]; }
        return static_cast<long long>(r_lo.y);
    };
    auto stage = [&](const int2 r_lo, const int2 r_hi, long long e_base, int b) {
        const int nb1 = r_hi.x - r_lo.x + 1;
        const uint32_t ne = static_cast<uint32_t>(r_hi.y) - static_cast<uint32_t>(r_lo.y);   // low words: exact inside a task
        if (r_hi.x > r_lo.x && nb1 <= kStageOff && ne <= static_cast<uint32_t>(kStageIdx)) {
            int* ib = s_warp + b * stage_idx;
            int* ob = s_off + b * kStageOff;
            const int nw = static_cast<int>(ne) << ish;
            const int* src = a.indices + (static_cast<size_t>(e_base) << ish);
            for (int i = lane; i < nw; i += 32) cp_async4(ib + i, src + i);
            for (int i = lane; i < nb1; i += 32) cp_async4(ob + i, a.offsets + (static_cast<size_t>(r_lo.x + i) << osh));
            if constexpr (GEN) {
                if (a.weights) {
                    float* wb = s_wgt + b * kStageIdx;
                    for (int i = lane; i < static_cast<int>(ne); i += 32) cp_async4(wb + i, a.weights + e_base + i);
                }
            }
        }
        cp_async_commit();
    };

    // ---- pipeline prologue ----
    uint32_t s = warp_id;
    int2 cur_lo = ld_plan(a.seg + s), cur_hi = ld_plan(a.seg + s + 1);
    int2 nxt_lo = cur_lo, nxt_hi = cur_hi;
    bool have_next = s + n_warps < S;
    if (have_next) { nxt_lo = ld_plan(a.seg + s + n_warps); nxt_hi = ld_plan(a.seg + s + n_warps + 1); }
    long long cur_base = task_base(s, cur_lo);
    stage(cur_lo, cur_hi, cur_base, 0);
    int buf = 0;

    for (;;) {
        // ---- prefetch: records two tasks ahead, offsets + indices one task ahead ----
        const uint32_t s2 = s + 2 * n_warps;
        const bool have_next2 = s2 < S;
        int2 n2_lo = nxt_lo, n2_hi = nxt_hi;
        if (have_next2) { n2_lo = ld_plan(a.seg + s2); n2_hi = ld_plan(a.seg + s2 + 1); }
        long long nxt_base = 0;
        if (have_next) {
            nxt_base = task_base(s + n_warps, nxt_lo);
            stage(nxt_lo, nxt_hi, nxt_base, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncwarp();

        const uint32_t g_lo = cur_lo.x, g_hi = cur_hi.x;
        if (g_lo < g_hi) {  // a long bag spanning several quanta leaves empty tasks behind it
            const uint32_t nb = g_hi - g_lo;
            const uint32_t ne = static_cast<uint32_t>(cur_hi.y) - static_cast<uint32_t>(cur_lo.y);
            const bool staged = (nb + 1 <= static_cast<uint32_t>(kStageOff)) && (ne <= static_cast<uint32_t>(kStageIdx));
            // entry positions are absolute (int32 offsets) or relative to the task's first entry (int64 offsets: osh = 1)
            const int e_lo = osh ? 0 : cur_lo.y;
            // generic pointers indexed by entry position / ABSOLUTE bag id: staged smem or the global arrays
            const int* ip = staged ? (s_warp + buf * stage_idx - (static_cast<ptrdiff_t>(e_lo) << ish))
                                   : (osh ? a.indices + (static_cast<size_t>(cur_base) << ish) : a.indices);
            OffView<GEN> op;
            op.p = staged ? (s_off + buf * kStageOff - static_cast<int>(g_lo)) : a.offsets;
            op.sh = staged ? 0 : osh;
            op.rebase = osh ? static_cast<uint32_t>(cur_lo.y) : 0u;
            const float* wp = nullptr;
            if constexpr (GEN) {
                if (a.weights) wp = staged ? (s_wgt + buf * kStageIdx - e_lo) : (osh ? a.weights + cur_base : a.weights);
            }

            bool onehot = false;
            if (ne == nb && a.mode != 2 && !(GEN && wp)) {
                // a task with ne == nb could still mix empty and longer bags: verify
                bool all_one = true;
                for (uint32_t i = lane; i < nb; i += 32) all_one &= (op[g_lo + i + 1] - op[g_lo + i]) == 1;
                onehot = __all_sync(0xffffffffu, all_one);
            }
            if (onehot) {
                // ---------------- one-hot task: Alg. 1, a pure row copy (bit-exact) ------------------------
                for (uint32_t i0 = 0; i0 < nb; i0 += P * U) {
                    Row v[U];
                    BagRef br[GEN ? U : 1];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        const bool ok = i < nb;
                        BagRef& b = br[GEN ? u : 0];
                        b = bag_ref(g_lo + (ok ? i : 0u));
                        const uint32_t r = idx_at(ip, e_lo + (ok ? i : 0u));
                        v[u] = Tr::load(b.tab + static_cast<uint64_t>(r) * b.row_bytes, ok && b.ok);
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const uint32_t i = i0 + u * P + sub;
                        const BagRef& b = br[GEN ? u : 0];
                        if (i < nb && b.ok) {  // dense layout: b.ok == vec_ok for every bag
                            char* po = out_of(g_lo + i, b);
                            if constexpr (OUT32 && Tr::kEltBytes == 2) {
                                float2 f[kAcc2];
                                zero_acc(f);
                                Tr::add(f, v[u]);
                                store_pooled<Tr, OUT32>(po, f);
                            } else {
                                st_row(po, v[u]);
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
                    const BagRef br = bag_ref(gc);
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    for (int j = lo; j < hi; j += U) {
                        Row v[U];
                        float w[U];
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            const bool ok = j + u < hi;
                            const int e = ok ? j + u : lo;
                            const uint32_t r = idx_at(ip, e);
                            w[u] = wgt_at(wp, e);
                            v[u] = Tr::load(br.tab + static_cast<uint64_t>(r) * br.row_bytes, ok && br.ok);
                        }
#pragma unroll
                        for (int u = 0; u < U; ++u) accum(acc, v[u], w[u]);
                    }
                    if (active && br.ok) {
                        if (is_mean(br.t) && hi - lo > 1) scale_mean(acc, hi - lo);
                        store_pooled<Tr, OUT32>(out_of(g, br), acc);
                    }
                }
            } else if (a.mode == 2) {
                // ---------------- whole warp per bag, one batch at a time (kept for A/B measurements) ------
                for (uint32_t g = g_lo; g < g_hi; ++g) {
                    const int lo = op[g], hi = op[g + 1];
                    const BagRef br = bag_ref(g);
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    for (int j = lo; j < hi; j += P * U) {
                        Row v[U];
                        float w[U];
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            const int e = j + u * P + sub;
                            const bool ok = e < hi;
                            const int ec = ok ? e : lo;
                            const uint32_t r = idx_at(ip, ec);
                            w[u] = wgt_at(wp, ec);
                            v[u] = Tr::load(br.tab + static_cast<uint64_t>(r) * br.row_bytes, ok && br.ok);
                        }
#pragma unroll
                        for (int u = 0; u < U; ++u) accum(acc, v[u], w[u]);
                    }
#pragma unroll
                    for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                        for (int i = 0; i < kAcc2; ++i)
                            acc[i] = __fadd2_rn(acc[i], make_float2(__shfl_xor_sync(0xffffffffu, acc[i].x, d),
                                                                    __shfl_xor_sync(0xffffffffu, acc[i].y, d)));
                    }
                    if (sub == 0 && br.ok) {
                        if (is_mean(br.t) && hi - lo > 1) scale_mean(acc, hi - lo);
                        store_pooled<Tr, OUT32>(out_of(g, br), acc);
                    }
                }
            } else {
                // ---------------- whole warp per bag, double-buffered batches (long bags) -------------------
                // The loads of batch k+1 (possibly the first batch of the NEXT bag: its offsets and indices
                // are already in smem) are issued before batch k is consumed, so a warp keeps U..2U row
                // loads per lane in flight across batch and bag boundaries instead of draining at each one.
                struct Buf {
                    Row v[U];
                    float w[GEN ? U : 1];
                };
                auto store_zero = [&](uint32_t gz) {
                    const BagRef bz = bag_ref(gz);
                    if (sub == 0 && bz.ok) {
                        float2 z[kAcc2];
                        zero_acc(z);
                        store_pooled<Tr, OUT32>(out_of(gz, bz), z);
                    }
                };
                // rows fill every lane of their lane group (row size = W vectors): no lane needs masking (dense layout only)
                const bool lanes_full = !GEN && a.nvec == static_cast<uint32_t>(W);
                auto issue = [&](Buf& bf, int j, int hi, const BagRef& br) {
                    if constexpr (!GEN && Tr::kEltBytes == 4) {
                        // whole batch inside the bag (warp-uniform): no bounds compare, no clamped index, no predicate and
                        // no zeroed destination registers per load; only a bag's ragged last batch takes the predicated
                        // form below. An instruction diet, not a speed-up: on c5 it removes 15 % of the
                        // issued instructions and, in a same-box A/B, no time (the kernel is HBM-bound). fp32 tables only:
                        // on bf16 c4, which IS issue-bound, the extra compare + branch and the second copy of the load code
                        // cost more than they save (0.396 ms, against 0.381-0.384 ms on every other call)
                        if (lanes_full && j + P * U <= hi) {
#pragma unroll
                            for (int u = 0; u < U; ++u) {
                                const uint32_t r = idx_at(ip, j + u * P + sub);
                                bf.v[u] = Tr::load_all(br.tab + static_cast<uint64_t>(r) * br.row_bytes);
                            }
                            return;
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int e = j + u * P + sub;
                        const bool ok = e < hi;
                        const int ec = ok ? e : j;
                        const uint32_t r = idx_at(ip, ec);
                        if constexpr (GEN) bf.w[u] = wgt_at(wp, ec);
                        bf.v[u] = Tr::load(br.tab + static_cast<uint64_t>(r) * br.row_bytes, ok && br.ok);
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
                    BagRef br = bag_ref(g);
                    float2 acc[kAcc2];
                    zero_acc(acc);
                    Buf bA, bB;
                    issue(bA, j, hi, br);
                    bool more = true;
                    auto step = [&](Buf& cv, Buf& nv) {
                        uint32_t g_n = g;
                        int j_n = j + P * U, lo_n = lo, hi_n = hi;
                        BagRef br_n = br;
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
                            if (has_next) { j_n = lo_n; br_n = bag_ref_next(br, g, g_n); }
                        }
                        if (has_next) issue(nv, j_n, hi_n, br_n);
#pragma unroll
                        for (int u = 0; u < U; ++u) accum(acc, cv.v[u], GEN ? cv.w[u] : 1.f);
                        if (last_of_bag) {
#pragma unroll
                            for (int d = W; d < 32; d <<= 1) {
#pragma unroll
                                for (int i = 0; i < kAcc2; ++i)
                                    acc[i] = __fadd2_rn(acc[i], make_float2(__shfl_xor_sync(0xffffffffu, acc[i].x, d),
                                                                            __shfl_xor_sync(0xffffffffu, acc[i].y, d)));
                            }
                            if (sub == 0 && br.ok) {
                                if (is_mean(br.t) && hi - lo > 1) scale_mean(acc, hi - lo);
                                store_pooled<Tr, OUT32>(out_of(g, br), acc);
                            }
                            zero_acc(acc);
                        }
                        g = g_n; j = j_n; lo = lo_n; hi = hi_n; br = br_n;
                        more = has_next;
                    };
                    while (more) {
                        step(bA, bB);
                        if (!more) break;
                        step(bB, bA);
                    }
                }
            }
        }

        if (!have_next) break;
        __syncwarp();  // every lane is done with buffer `buf` before the next iteration refills it
        s += n_warps;
        cur_lo = nxt_lo; cur_hi = nxt_hi;
        cur_base = nxt_base;
        nxt_lo = n2_lo; nxt_hi = n2_hi;
        have_next = have_next2;
        buf ^= 1;
    }
}

// ---- host-side dispatch (one translation unit per dtype keeps nvcc parallel) ------------------------------
inline size_t lookup_smem_bytes(const LookupArgs& a, bool gen, int block_threads) {
    const size_t tab = gen ? static_cast<size_t>(a.T) * sizeof(TableInfo)
                           : ((static_cast<size_t>(a.T) * 8 + 15) & ~static_cast<size_t>(15));
    const int ish = gen ? static_cast<int>(a.idx_shift) : 0;
    const size_t warp_words = 2 * (static_cast<size_t>(kStageIdx) << ish) + 2 * kStageOff + ((gen && a.weights) ? 2 * kStageIdx : 0);
    return tab + static_cast<size_t>(block_threads / 32) * warp_words * sizeof(int);
}

// Launch: no CUDA runtime query and no attribute call here -- prepare_one() did both when the plan was created or
// re-configured (dpi_api.cu::prepare_launches), for the device the plan lives on.
template <class Tr, int W, int U, bool OUT32, bool GEN>
cudaError_t launch_one(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(static_cast<unsigned>(l.grid));
    cfg.blockDim = dim3(static_cast<unsigned>(l.block_threads));
    cfg.dynamicSmemBytes = lookup_smem_bytes(a, GEN, l.block_threads);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = l.pdl ? 1 : 0;
    count_launch();
    return cudaLaunchKernelEx(&cfg, lookup_kernel<Tr, W, U, OUT32, GEN>, a);
}

// Raises the dynamic shared-memory limit of the instantiation on the CURRENT device when it needs more than 48 KB and
// returns its resident CTAs per SM (0 on error). Called per plan, never per lookup.
template <class Tr, int W, int U, bool OUT32, bool GEN>
int prepare_one(const LookupArgs& a, int block_threads) {
    int n = 0;
    const size_t smem = lookup_smem_bytes(a, GEN, block_threads);
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(lookup_kernel<Tr, W, U, OUT32, GEN>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, lookup_kernel<Tr, W, U, OUT32, GEN>, block_threads, smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

#define DPI_FOR_EACH_U(M, W) M(W, 2) M(W, 4) M(W, 8) M(W, 16)
#define DPI_FOR_EACH_WU(M) \
    DPI_FOR_EACH_U(M, 1) DPI_FOR_EACH_U(M, 2) DPI_FOR_EACH_U(M, 4) DPI_FOR_EACH_U(M, 8) DPI_FOR_EACH_U(M, 16) \
    DPI_FOR_EACH_U(M, 32)
// 256-bit row vectors (Wide<Traits>): rows of up to 512 B need at most 16 lanes.
#define DPI_FOR_EACH_U_WIDE(M, W) M(W, 1) M(W, 2) M(W, 4)
#define DPI_FOR_EACH_WU_WIDE(M) \
    DPI_FOR_EACH_U_WIDE(M, 1) DPI_FOR_EACH_U_WIDE(M, 2) DPI_FOR_EACH_U_WIDE(M, 4) DPI_FOR_EACH_U_WIDE(M, 8) M(8, 8) \
    DPI_FOR_EACH_U_WIDE(M, 16) M(16, 8)
// The general variant (GEN) exists for the default unroll only.
#define DPI_FOR_EACH_W_GEN(M) M(1, 2) M(2, 2) M(4, 2) M(8, 2) M(16, 2) M(32, 2)
// Each lookup_<dtype>.cu defines DPI_TRAITS / DPI_SUFFIX (/ DPI_HAS_OUT32) and includes lookup_dispatch.inc.

}  // namespace dpi
