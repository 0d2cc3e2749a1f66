// dpi_internal.cuh -- shared declarations of libdpi (sm_100a only). Not part of the public boundary.
#pragma once

#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include "../../include/dpi.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libdpi is written for sm_100a (B200) only"
#endif

namespace dpi {

constexpr int kMetaWords = 12;  // meta_dev layout: {S, N (low 32), C[G] (low 32), overflow, K, G, min_len, max_len, N (high 32),
                                // C[G] (high 32), -, -}; the high words are written by the 64-bit planner only (else 0)
enum MetaSlot { META_S = 0, META_N = 1, META_C = 2, META_OVERFLOW = 3, META_K = 4, META_G = 5, META_MINLEN = 6, META_MAXLEN = 7,
                META_N_HI = 8, META_C_HI = 9 };
// The device picks the a3 variant from a1's max_len: bags of 2..kShortBagMax entries run the short-bag
// body (one lane group per bag); exactly one entry per bag runs it up to kShortOnehotMaxBags bags, beyond that the
// balanced-segment kernel's row-copy path with its index prefetch pipeline is faster (measured).
constexpr uint32_t kShortBagMax = 8;
constexpr uint32_t kShortOnehotMaxBags = 500000;
__host__ __device__ inline bool short_bag_rule(uint32_t max_len, uint32_t G) {
    return max_len >= 2 ? max_len <= kShortBagMax : G <= kShortOnehotMaxBags;
}

constexpr int kPoolWords = DPI_MAX_TABLES / 32;
struct PoolMask {
    uint32_t w[kPoolWords];  // bit t set -> table t is mean-pooled
};

// ---- planner (plan_kernels.cu) ---------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;                               // consecutive bags per thread (two int4 loads)
constexpr int kScanTile = kScanThreads * kScanItems;        // 2048 bags per tile
constexpr int kMaxChunks = 320;                             // CTAs of the planner (all co-resident); multiple of 32

enum PlanState { kStateTicket = 0, kStateDone = 1, kStateEpoch = 2, kStateOverflows = 3, kStateMinLen = 4, kStateMaxLen = 5,
                 kStateWords = 8 };
constexpr uint32_t kEpochLimit = 1u << 30;  // status words carry a 30-bit epoch

struct PlanArgs {
    const int32_t* __restrict__ len;   // [G]
    int32_t* __restrict__ offsets;     // [G+1]
    int2* __restrict__ seg;            // [seg_cap] {seg_bag[s], seg_off[s] = offsets[seg_bag[s]]}
    int32_t* __restrict__ meta;        // [kMetaWords]
    ulonglong2* status;                // [num_chunks] look-back records {len aggregate, cost aggregate}, each half
                                       // tagged {epoch:30 | state:2 | value:32}
    unsigned int* state;               // [kStateTicket] dynamic tile id, [kStateDone] finished tiles (both
                                       // self-resetting atomicInc), [kStateEpoch] tag of this build's status words,
                                       // [kStateOverflows] builds that exceeded the capacity (sticky, dpi_plan_status),
                                       // [kStateMinLen/MaxLen] running min / max length of the build in flight
    uint32_t G;
    uint32_t K;
    uint32_t seg_cap;
    uint32_t num_tiles;                // ceil(G / kScanTile)
    uint32_t num_chunks;               // CTAs: min(num_tiles, 2 * SMs, kMaxChunks)
    uint32_t tiles_per_chunk;          // ceil(num_tiles / num_chunks) (num_chunks is then re-derived so no chunk is empty)
    uint32_t max_indices;
};

cudaError_t launch_plan(const PlanArgs& a, cudaStream_t stream);

// 64-bit offsets (plan64_kernels.cu; NEXT-2): two stream-ordered launches, no status records
struct Plan64Args {
    const int32_t* __restrict__ len;   // [G]
    long long* __restrict__ offsets;   // [G+1] int64
    int2* __restrict__ seg;            // [seg_cap] {seg_bag[s], low 32 bits of seg_off[s]}
    long long* __restrict__ seg_off;   // [seg_cap] int64
    int32_t* __restrict__ meta;        // [kMetaWords]
    void* agg;                         // [num_chunks] 32-byte chunk aggregates
    unsigned int* state;               // planner state of the plan (sticky overflow counter)
    uint32_t G;
    unsigned long long K;
    unsigned long long seg_cap;
    uint32_t num_tiles, num_chunks, tiles_per_chunk;
    unsigned long long max_indices;
};
cudaError_t launch_plan64(const Plan64Args& a, cudaStream_t stream);

// ---- a1 + a2 + a3 in one launch (forward_fused.cu) ----
constexpr int kFusedThreads = 256;
constexpr int kFusedItems = 8;                              // bags per thread, held in registers across the look-back
constexpr int kFusedMaxChunkBags = kFusedThreads * kFusedItems;
constexpr int kFusedMaxChunks = 640;                        // CTAs (one resident wave: 148 SMs x 4)
constexpr int kFusedIdxStage = 3072;                        // index entries of a chunk staged in shared memory
constexpr int kStatusRecords = kFusedMaxChunks > kMaxChunks ? kFusedMaxChunks : kMaxChunks;

struct CheckArgs {
    const void* __restrict__ indices;        // int32 or int64 (idx64)
    const int32_t* __restrict__ offsets;     // int32[G+1], or int64[G+1] when off64
    const int64_t* __restrict__ table_rows;  // device [T]
    unsigned long long* n_bad;               // [0] indices out of range, [1] bags longer than max_bag (when max_bag > 0)
    int32_t max_bag;                         // DPI_OPT_MAX_BAG_HINT, 0 = no promise to check
    uint32_t G;
    uint32_t T;
    uint32_t B;
    bool idx64;
    bool table_major;
    bool off64;
};
cudaError_t launch_check_indices(const CheckArgs& a, cudaStream_t stream);

// ---- lookup (lookup_*.cu) --------------------------------------------------------------------------
struct LookupArgs {
    const void* const* __restrict__ tables;  // device [T] table base pointers
    const int32_t* __restrict__ indices;     // [N]
    const int32_t* __restrict__ offsets;     // [G+1]
    const int2* __restrict__ seg;            // [S+1] {seg_bag, seg_off}
    const int32_t* __restrict__ meta;        // meta[META_S] = S
    void* __restrict__ out;                  // [G * D] in the output dtype (out[b, t*D + c] == out[g*D + c])
    uint32_t G;
    uint32_t T;
    uint32_t nvec;                           // lane vectors per row = D*sizeof(elt)/16 (the widest table when dims differ); the
                                             // 256-bit instantiations of lookup_kernel take D*sizeof(elt)/32
    int32_t mode;                            // 0 auto, 1 sub-warp per bag, 2 warp per bag
    // ---- general variant only (dpi_lookup_ex; lookup_kernel<..., GEN = true>) ----
    const float* __restrict__ weights;       // NULL or fp32[N]: one weight per index entry
    const uint32_t* __restrict__ tab_nvec;   // device [T] vectors per row of each table
    const uint32_t* __restrict__ tab_col;    // device [T] first output vector of each table's column block
    const void* const* __restrict__ peer_out; // NULL, or device [n_peers] output base pointers (peer-mapped memory)
    uint32_t rows_per_peer;                  // samples per peer when peer_out is set
    uint64_t out_pitch;                      // bytes between consecutive output rows
    uint32_t B;
    uint32_t idx_shift;                      // 0: int32 ids, 1: int64 ids (indices then points at the low words)
    uint32_t table_major;                    // 0: g = b*T + t, 1: g = t*B + b
    uint32_t off_shift;                      // 0: int32 offsets; 1: int64 offsets (offsets then points at the low words; GEN only)
    const long long* __restrict__ seg_off64; // off_shift = 1: 64-bit first entry of every task (seg[s].y holds its low word)
    PoolMask pool;
};

// plan.num_chunks = CTAs, chunk c owns bags [c*chunk_bags, min(G, (c+1)*chunk_bags)); plan.num_tiles / tiles_per_chunk unused
struct FusedArgs {
    PlanArgs plan;
    LookupArgs look;
    uint32_t chunk_bags;                 // <= kFusedMaxChunkBags
    uint32_t items;                      // bags per thread = ceil(chunk_bags / kFusedThreads)
    uint32_t any_mean;                   // some table is mean-pooled (else the pooling mask is never consulted)
    uint32_t k_shift;                    // log2(K) when the quantum is a power of two, else 32 (divide)
    float* fm_y;                         // dpi_forward_fm: fp32[B] FM second-order term (chunk_bags is then a multiple of T), or NULL
    float* fm_v;                         // dpi_forward_fm: fp32[B, D] or NULL
};
cudaError_t launch_fused(const FusedArgs& a, int dtype, bool out32, int lanes, bool pdl, cudaStream_t stream);
int fused_occupancy(int dtype, bool out32, int lanes, uint32_t T);   // resident CTAs per SM (0: no instantiation)

struct LookupLaunch {
    int lanes;          // lanes per row (power of two >= nvec)
    int unroll;         // 2, 4, 8, 16
    int block_threads;  // 128, 256, 512
    int grid;           // persistent grid size
    bool pdl;           // programmatic dependent launch
    bool out32;         // 16-bit tables only: emit the output block in fp32
    bool general;       // the GEN instantiation (interface variants)
    bool vec32;         // 256-bit row vectors (Wide<Traits>): lanes = pow2ceil(row bytes / 32); dense layout only
};

// Each returns cudaErrorInvalidValue when (lanes, unroll, block_threads) has no instantiation.
cudaError_t launch_lookup_f32(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream);
cudaError_t launch_lookup_f16(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream);
cudaError_t launch_lookup_bf16(const LookupArgs& a, const LookupLaunch& l, cudaStream_t stream);
// Per plan, not per lookup: raises the instantiation's dynamic shared-memory limit on the current device if needed and
// returns its resident CTAs per SM (0 if there is no such instantiation). Only a.T, a.idx_shift and a.weights matter.
int lookup_prepare_f32(const LookupArgs& a, const LookupLaunch& l);
int lookup_prepare_f16(const LookupArgs& a, const LookupLaunch& l);
int lookup_prepare_bf16(const LookupArgs& a, const LookupLaunch& l);

// Ablation (ablation_input_first.cu): one thread per sample.
cudaError_t launch_input_first(const LookupArgs& a, uint32_t B, int dtype, bool out32, cudaStream_t stream);

// Short-bag variant of a3 (lookup_direct.cu): one lane group per bag straight from the plan's offsets, no segments.
// grid_cap = SMs x resident CTAs per SM of the instantiation (direct_occupancy, queried once per plan).
cudaError_t launch_direct(const LookupArgs& a, int dtype, bool out32, int lanes, int grid_cap, bool pdl, cudaStream_t stream);
int direct_occupancy(int dtype, bool out32, int lanes, uint32_t T);

// Algorithm 1, plan-free one-hot lookup (lookup_onehot.cu).
cudaError_t launch_onehot(const void* const* tables, const void* ids, uint32_t idx_shift, void* out, uint32_t G, uint32_t T,
                          uint32_t nvec, int lanes, int num_sms, cudaStream_t stream);

void count_launch();

// ---- NEXT-4: non-GEMM consumers of X_embed (nongemm_kernels.cu; boundary in include/dpi_nongemm.h) ---------
cudaError_t launch_fm(const void* x, int dtype, uint32_t B, uint32_t T, uint32_t D, uint64_t x_pitch_bytes, float* y,
                      float* v, cudaStream_t st);
cudaError_t launch_lr(const void* const* w, const int32_t* indices, const int32_t* offsets, uint32_t B, uint32_t T, float bias,
                      float* y, int accumulate, cudaStream_t st);
cudaError_t launch_cross_combine(const void* x0, const void* xl, const void* u, const float* bias, void* out, int dtype,
                                 uint32_t B, uint32_t F, cudaStream_t st);
cudaError_t launch_bias_act(const void* u, const float* bias, void* out, int dtype, uint32_t B, uint32_t F, int act,
                            cudaStream_t st);
// error text of the calling thread (dpi_last_error); defined in dpi_api.cu
dpi_status_t report_error(dpi_status_t st, const char* fmt, ...);

}  // namespace dpi
