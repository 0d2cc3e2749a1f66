// dpi_api.cu -- the C ABI of include/dpi.h. Host-side validation, plan ownership and launches only:
// every step of the path runs in plan_kernels.cu / lookup_*.cu. No CPU fallback anywhere.
#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "dpi_internal.cuh"
#include "../../include/dpi_nongemm.h"

namespace dpi {
namespace {

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

dpi_status_t fail(dpi_status_t st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}
dpi_status_t cuda_fail(cudaError_t e, const char* what) {
    (void)cudaGetLastError();
    return fail(e == cudaErrorMemoryAllocation ? DPI_ERR_ALLOC : DPI_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define DPI_CUDA(call)                                       \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);  \
    } while (0)

int pow2ceil(int x) {
    int p = 1;
    while (p < x) p <<= 1;
    return p;
}

}  // namespace

void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

dpi_status_t report_error(dpi_status_t st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}

}  // namespace dpi

using namespace dpi;

struct dpi_plan_s {
    // shape
    int32_t T = 0, B = 0, D = 0;   // D = the widest table's dim
    int64_t out_width = 0;         // sum of dims = elements per output row
    bool mixed_dims = false;
    bool custom_columns = false;   // dpi_plan_set_columns: tables placed at caller-given columns
    std::vector<int32_t> dims;
    dpi_bag_order_t bag_order = DPI_BAGS_SAMPLE_MAJOR;
    dpi_index_type_t index_type = DPI_IDX_I32;
    dpi_dtype_t dtype = DPI_F32;
    dpi_dtype_t out_dtype = DPI_F32;
    uint32_t G = 0;
    int64_t max_indices = 0;
    uint32_t nvec = 0;   // 16-byte vectors per row
    int lanes = 0;       // lanes per row at 16 bytes per lane
    bool wide = false;   // 256-bit row vectors in the dense balanced-segment kernel (every row a multiple of 32 B)
    uint32_t nvec_w = 0; // 32-byte vectors per row
    int lanes_w = 0;     // lanes per row at 32 bytes per lane
    std::vector<int64_t> table_rows;
    // plan parameters
    int32_t K = 0;           // effective quantum
    int32_t K_user = 0;      // 0 = default
    uint32_t seg_cap = 0;    // capacity of seg_bag (elements), sized for K_min
    uint32_t num_tiles = 0, num_chunks = 0, tiles_per_chunk = 0;
    int32_t opt[DPI_OPT_COUNT_] = {0, 0, 0, 0, -1, 1, 0, 0, 0, 0, 0, 0};  // PDL on: 4-10 % per step on small batches, neutral on large ones
    // device
    int device = 0, num_sms = 0;
    int32_t* offsets = nullptr;
    int2* seg = nullptr;          // {seg_bag[s], seg_off[s]} interleaved
    int32_t* meta = nullptr;
    ulonglong2* status = nullptr;    // planner look-back records, one per chunk
    unsigned int* state = nullptr;   // planner device state {ticket, done, epoch, -}
    int64_t* table_rows_dev = nullptr;
    uint32_t* tab_nvec_dev = nullptr;   // [T] 16-byte vectors per row of each table
    uint32_t* tab_col_dev = nullptr;    // [T] first output vector of each table's column block
    unsigned long long* n_bad_dev = nullptr;
    // 64-bit offsets (dpi_plan_set_offset_type; NEXT-2): the plan then lives in these instead of `offsets`
    bool off64 = false;
    long long* offsets64 = nullptr;   // [G+1]
    long long* seg_off64 = nullptr;   // [seg_cap]
    void* agg64 = nullptr;            // [num_chunks] chunk aggregates of the two-launch 64-bit planner
    // staging for dpi_forward_host
    int32_t* stage_len = nullptr;
    void* stage_idx = nullptr;
    size_t stage_idx_bytes = 0;
    void* stage_out = nullptr;
    struct HostPipeline* pipe = nullptr;   // dpi_forward_host: sample-chunked sub-plans + copy/compute streams
    bool built = false;
    // Launch configurations, computed when the plan is created or re-configured (prepare_launches): occupancy queries
    // and shared-memory attributes happen there, for the plan's device -- a lookup only fills in pointers and launches.
    LookupLaunch launch_dense{}, launch_gen{}, launch_gen_w{};   // balanced-segment kernel: dense / general / general + weights
    LookupLaunch launch_dense16{};                               // dense with 128-bit row vectors (output not 32-byte aligned)
    int direct_grid_cap = 0;       // short-bag variant as its own launch: SMs x resident CTAs
    uint32_t fused_chunks = 0;     // fused single-launch path: CTAs (0 = no instantiation) and bags per CTA
    uint32_t fused_chunk_bags = 0;
    uint32_t fused_fm_chunks = 0;  // the same with chunks of whole samples (dpi_forward_fm); 0 = not possible
    uint32_t fused_fm_chunk_bags = 0;
    std::vector<int64_t> columns;  // dpi_plan_set_columns, kept for the sub-plans of dpi_forward_host
};

// dpi_forward_host cuts a large batch into chunks of whole samples; chunk c runs H2D -> plan -> lookup -> D2H on
// stream c % 3, so the copy engines (both PCIe directions) and the SMs work on different chunks at the same time.
struct HostPipeline {
    static constexpr int kStreams = 3;
    int n_requested = 0;                // the chunk count this pipeline was built for
    std::vector<dpi_plan_t*> sub;       // one plan per chunk (B_c samples each)
    std::vector<int32_t> sample_lo;     // first sample of each chunk (+ B at the end)
    cudaStream_t st[kStreams] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_in = nullptr, ev_done[kStreams] = {nullptr, nullptr, nullptr};
};

namespace {

// 256-bit row vectors in the dense balanced-segment kernel (DPI_OPT_VEC_BYTES = v). Possible whenever all dims are equal and
// the row size is a multiple of 32 B; chosen by default only where it measured faster: fp32 rows of
// >= 256 B (c5: 0.734 -> 0.716 ms). On 16-bit tables the wider accumulator set spills at the 64-register bound and halving
// the lanes per row doubles the sub-warps whose partial sums meet by shuffle (c4: 0.382 -> 0.515 ms), so they stay at 128 bit.
bool wide_allowed(const dpi_plan_t* p, int32_t v) {
    const int64_t row_bytes = static_cast<int64_t>(p->D) * (p->dtype == DPI_F32 ? 4 : 2);
    if (v == 16 || p->mixed_dims || row_bytes % 32 != 0) return false;
    return v == 32 || (p->dtype == DPI_F32 && row_bytes >= 256);
}

int32_t default_quantum(const dpi_plan_t* p) {
    // Measured on B200 (DESIGN.md section 3 and 12 "Balanced quantum"): K = 128 is best once there are plenty of tasks per warp (c4/c5:
    // the per-task pipeline refill is amortised); small batches want more, smaller tasks so that every resident
    // warp has work: aim at >= 4 tasks per warp of a full persistent grid (32 warps per SM), within [16, 128].
    const uint64_t cost_bound = static_cast<uint64_t>(p->max_indices) + p->G;   // >= C[G]
    const uint64_t warps = static_cast<uint64_t>(p->num_sms > 0 ? p->num_sms : 148) * 32;
    uint64_t k = cost_bound / (4 * warps);
    int32_t K = 16;
    while (K < 128 && static_cast<uint64_t>(K) * 2 <= k) K *= 2;
    return K;
}

uint32_t seg_capacity_for(const dpi_plan_t* p, int32_t K) {
    // S = ceil(C[G]/K) <= ceil((max_indices + G)/K); +2 for seg_bag[S] and slack
    const uint64_t c_max = static_cast<uint64_t>(p->max_indices) + p->G;
    return static_cast<uint32_t>((c_max + K - 1) / K + 2);
}

dpi_status_t ensure_seg_capacity(dpi_plan_t* p, int32_t K) {
    const uint64_t c_max = static_cast<uint64_t>(p->max_indices) + p->G;
    if ((c_max + K - 1) / K + 2 >= (1ull << 31)) return fail(DPI_ERR_INVALID_ARG, "quantum K=%d gives more than 2^31 segments for max_indices=%lld", K, (long long)p->max_indices);
    const uint32_t need = seg_capacity_for(p, K);
    if (need <= p->seg_cap && p->seg && (!p->off64 || p->seg_off64)) return DPI_OK;
    int2* fresh = nullptr;
    long long* fresh64 = nullptr;
    const uint32_t cap = std::max(need, p->seg_cap);
    DPI_CUDA(cudaMalloc(&fresh, static_cast<size_t>(cap) * sizeof(int2)));   // on failure the old buffers stay in place
    if (p->off64) {
        cudaError_t e = cudaMalloc(&fresh64, static_cast<size_t>(cap) * sizeof(long long));
        if (e != cudaSuccess) { (void)cudaFree(fresh); return cuda_fail(e, "cudaMalloc(seg_off64)"); }
    }
    if (p->seg) (void)cudaFree(p->seg);
    if (p->seg_off64) (void)cudaFree(p->seg_off64);
    p->seg = fresh;
    p->seg_off64 = fresh64;
    p->seg_cap = cap;
    return DPI_OK;
}

void free_pipeline(dpi_plan_t* p);

void free_plan(dpi_plan_t* p) {
    if (!p) return;
    free_pipeline(p);
    cudaFree(p->offsets); cudaFree(p->seg); cudaFree(p->meta); cudaFree(p->status);
    cudaFree(p->state); cudaFree(p->table_rows_dev); cudaFree(p->n_bad_dev);
    cudaFree(p->tab_nvec_dev); cudaFree(p->tab_col_dev);
    cudaFree(p->offsets64); cudaFree(p->seg_off64); cudaFree(p->agg64);
    cudaFree(p->stage_len); cudaFree(p->stage_idx); cudaFree(p->stage_out);
    (void)cudaGetLastError();
    delete p;
}

int prepare(const dpi_plan_t* p, const LookupArgs& a, const LookupLaunch& l) {
    switch (p->dtype) {
        case DPI_F32: return lookup_prepare_f32(a, l);
        case DPI_F16: return lookup_prepare_f16(a, l);
        default: return lookup_prepare_bf16(a, l);
    }
}

LookupLaunch prepare_one_launch(const dpi_plan_t* p, bool general, bool weights, bool wide = false) {
    LookupArgs a{};   // only T, idx_shift and weights != NULL enter the shared-memory size
    a.T = static_cast<uint32_t>(p->T);
    a.idx_shift = p->index_type == DPI_IDX_I64 ? 1u : 0u;
    a.weights = weights ? reinterpret_cast<const float*>(sizeof(float)) : nullptr;
    LookupLaunch l{};
    l.lanes = wide ? p->lanes_w : p->lanes;
    l.general = general;
    l.vec32 = wide;
    l.unroll = (p->opt[DPI_OPT_UNROLL] && !general) ? p->opt[DPI_OPT_UNROLL] : 2;  // x2 by double buffering
    // DPI_OPT_UNROLL counts 128-bit loads in flight per lane: a 256-bit load is two of them (default: ONE 256-bit load)
    // (measured on c5: four 256-bit loads per batch and lane, 2 CTAs of 256 threads per SM, beat every
    // 128-bit configuration and the shallower / deeper 256-bit ones)
    if (wide) l.unroll = p->opt[DPI_OPT_UNROLL] ? std::min(l.lanes >= 8 ? 8 : 4, std::max(1, l.unroll / 2)) : 4;
    l.block_threads = p->opt[DPI_OPT_BLOCK_THREADS] ? p->opt[DPI_OPT_BLOCK_THREADS] : 256;
    l.out32 = p->dtype != DPI_F32 && p->out_dtype == DPI_F32;
    int per_sm = prepare(p, a, l);   // also raises the instantiation's dynamic shared-memory limit when needed
    if (p->opt[DPI_OPT_BLOCKS_PER_SM] > 0) per_sm = p->opt[DPI_OPT_BLOCKS_PER_SM];
    if (per_sm <= 0) per_sm = 1;
    l.grid = p->num_sms * per_sm;  // persistent: a whole number of waves, every CTA resident
    const int64_t warps_per_cta = l.block_threads / 32;
    const int64_t need = (static_cast<int64_t>(p->seg_cap) + warps_per_cta - 1) / warps_per_cta;  // one warp per possible task
    if (need < l.grid) l.grid = static_cast<int>(need > 0 ? need : 1);
    l.pdl = p->opt[DPI_OPT_PDL] != 0;
    return l;
}

// Everything a launch needs that costs a CUDA runtime call. Runs in dpi_plan_create and in every setter that changes an
// input of it (options, quantum, output dtype, layout) -- never in dpi_lookup / dpi_forward.
void prepare_launches(dpi_plan_t* p) {
    p->launch_dense16 = prepare_one_launch(p, false, false);
    p->launch_dense = p->wide ? prepare_one_launch(p, false, false, true) : p->launch_dense16;
    p->launch_gen = prepare_one_launch(p, true, false);
    p->launch_gen_w = prepare_one_launch(p, true, true);
    const bool out32 = p->dtype != DPI_F32 && p->out_dtype == DPI_F32;
    p->direct_grid_cap = p->num_sms * direct_occupancy(p->dtype, out32, p->lanes, static_cast<uint32_t>(p->T));
    // fused single-launch path: at most one resident wave, at most kFusedMaxChunks chunks (one look-back record per
    // thread), and no chunk smaller than one bag per lane group
    const int occ = fused_occupancy(p->dtype, out32, p->lanes, static_cast<uint32_t>(p->T));
    p->fused_chunks = 0;
    p->fused_chunk_bags = 0;
    if (occ > 0) {
        uint64_t chunks = std::min<uint64_t>(kFusedMaxChunks, static_cast<uint64_t>(p->num_sms) * occ);
        const uint32_t min_bags = static_cast<uint32_t>(kFusedThreads / p->lanes);
        chunks = std::min<uint64_t>(chunks, (static_cast<uint64_t>(p->G) + min_bags - 1) / min_bags);
        if (chunks < 1) chunks = 1;
        p->fused_chunk_bags = static_cast<uint32_t>((p->G + chunks - 1) / chunks);
        p->fused_chunks = (p->G + p->fused_chunk_bags - 1) / p->fused_chunk_bags;
        if (p->fused_chunk_bags > static_cast<uint32_t>(kFusedMaxChunkBags)) p->fused_chunks = 0;   // a thread keeps <= 8 bags in registers
        // chunks of whole samples for the FM epilogue: the bag count of a chunk rounded up to a multiple of T
        const uint64_t T = static_cast<uint64_t>(p->T);
        const uint64_t fm_bags = (p->fused_chunk_bags + T - 1) / T * T;
        p->fused_fm_chunks = 0;
        if (p->fused_chunks && fm_bags <= static_cast<uint64_t>(kFusedMaxChunkBags)) {
            p->fused_fm_chunk_bags = static_cast<uint32_t>(fm_bags);
            p->fused_fm_chunks = static_cast<uint32_t>((p->G + fm_bags - 1) / fm_bags);
        }
    }
}

void free_pipeline(dpi_plan_t* p) {
    HostPipeline* h = p->pipe;
    if (!h) return;
    for (dpi_plan_t* q : h->sub) free_plan(q);
    for (int i = 0; i < HostPipeline::kStreams; ++i) {
        if (h->st[i]) cudaStreamDestroy(h->st[i]);
        if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
    }
    if (h->ev_in) cudaEventDestroy(h->ev_in);
    (void)cudaGetLastError();
    delete h;
    p->pipe = nullptr;
}

struct LookupCall {
    const void* const* tables = nullptr;
    const void* indices = nullptr;
    const int32_t* offsets = nullptr;
    const float* weights = nullptr;
    const uint8_t* pooling = nullptr;
    void* out = nullptr;
    int64_t out_ld = 0;     // elements; 0 = dense
    const void* const* peers = nullptr;   // device [n_peers] output base pointers
    int32_t n_peers = 0;
    int32_t rows_per_peer = 0;
    bool force_general = false;
};

size_t out_elt_bytes(const dpi_plan_t* p) { return p->out_dtype == DPI_F32 ? 4 : 2; }

dpi_status_t do_lookup(const dpi_plan_t* p, const LookupCall& c, cudaStream_t stream, bool input_first = false) {
    LookupArgs a{};
    a.tables = c.tables;
    a.indices = static_cast<const int32_t*>(c.indices);
    a.offsets = c.offsets ? c.offsets : (p->off64 ? reinterpret_cast<const int32_t*>(p->offsets64) : p->offsets);
    a.off_shift = p->off64 ? 1u : 0u;
    a.seg_off64 = p->seg_off64;
    a.seg = p->seg;
    a.meta = p->meta;
    a.out = c.out;
    a.G = p->G;
    a.T = static_cast<uint32_t>(p->T);
    a.B = static_cast<uint32_t>(p->B);
    a.nvec = p->nvec;
    a.mode = p->opt[DPI_OPT_MODE];
    a.weights = c.weights;
    a.tab_nvec = p->tab_nvec_dev;
    a.tab_col = p->tab_col_dev;
    a.idx_shift = p->index_type == DPI_IDX_I64 ? 1u : 0u;
    a.table_major = p->bag_order == DPI_BAGS_TABLE_MAJOR ? 1u : 0u;
    const int64_t ld = c.out_ld ? c.out_ld : p->out_width;
    if (ld < p->out_width) return fail(DPI_ERR_INVALID_ARG, "out_ld=%lld is smaller than the row width %lld", (long long)ld, (long long)p->out_width);
    a.out_pitch = static_cast<uint64_t>(ld) * out_elt_bytes(p);
    const uintptr_t out_align = (p->dtype != DPI_F32 && p->out_dtype == DPI_F32) ? 31u : 15u;
    if (a.out_pitch & out_align) return fail(DPI_ERR_INVALID_ARG, "output row pitch %llu B is not a multiple of %d B", (unsigned long long)a.out_pitch, (int)out_align + 1);
    std::memset(&a.pool, 0, sizeof a.pool);
    if (c.pooling) {
        for (int t = 0; t < p->T; ++t) {
            if (c.pooling[t] > 1) return fail(DPI_ERR_INVALID_ARG, "pooling[%d] = %d is not a dpi_pool_t", t, c.pooling[t]);
            if (c.pooling[t] == DPI_POOL_MEAN) {
                if (c.weights) return fail(DPI_ERR_UNSUPPORTED, "per-entry weights need sum pooling (table %d is mean-pooled)", t);
                a.pool.w[t >> 5] |= 1u << (t & 31);
            }
        }
    }
    if (c.peers) {
        if (c.n_peers < 1 || c.rows_per_peer < 1) return fail(DPI_ERR_INVALID_ARG, "n_peers=%d, rows_per_peer=%d", c.n_peers, c.rows_per_peer);
        if (static_cast<int64_t>(c.n_peers) * c.rows_per_peer < p->B) return fail(DPI_ERR_INVALID_ARG, "n_peers*rows_per_peer=%lld does not cover B=%d", (long long)c.n_peers * c.rows_per_peer, p->B);
        a.peer_out = c.peers;
        a.rows_per_peer = static_cast<uint32_t>(c.rows_per_peer);
    }
    const bool general = c.force_general || p->mixed_dims || p->custom_columns || a.idx_shift || a.table_major || c.weights ||
                         c.peers || ld != p->out_width || p->off64;
    if (input_first) {
        if (general) return fail(DPI_ERR_UNSUPPORTED, "the input-first ablation kernel only takes the dense int32 sample-major layout");
        cudaError_t e = launch_input_first(a, static_cast<uint32_t>(p->B), p->dtype, p->dtype != DPI_F32 && p->out_dtype == DPI_F32, stream);
        if (e != cudaSuccess) return cuda_fail(e, "input-first kernel launch");
        return DPI_OK;
    }
    // Without a hint lookup_kernel reads a1's max_len on the device and takes the short-bag body by the same rule
    // (short_bag_rule); the OPTIONAL promise DPI_OPT_MAX_BAG_HINT (or DPI_OPT_MODE = 6) picks the short-bag variant as its own
    // launch on the host. Measured on B200: with multi-hot bags of <= 8 entries it wins at every batch size;
    // with at most ONE entry per bag the balanced-segment kernel's row-copy path overtakes it beyond ~5e5 bags.
    const int32_t hint = p->opt[DPI_OPT_MAX_BAG_HINT];
    const bool short_bags = hint >= 1 && short_bag_rule(static_cast<uint32_t>(hint), p->G);
    // the short-bag variant also takes int64 ids (the one interface variant every framework feeds)
    const bool general_but_ids = c.force_general || p->mixed_dims || p->custom_columns || a.table_major || c.weights || c.peers ||
                                 ld != p->out_width || p->off64;
    if (!general_but_ids && (p->opt[DPI_OPT_MODE] == 6 || (p->opt[DPI_OPT_MODE] == 0 && short_bags))) {
        cudaError_t e = launch_direct(a, p->dtype, p->dtype != DPI_F32 && p->out_dtype == DPI_F32, p->lanes, p->direct_grid_cap,
                                      p->opt[DPI_OPT_PDL] != 0, stream);
        if (e != cudaSuccess) return cuda_fail(e, "direct lookup kernel launch");
        return DPI_OK;
    }
    // 256-bit row vectors store 32 bytes per lane: an output block that is only 16-byte aligned takes the 128-bit kernel
    const bool out32b = ((reinterpret_cast<uintptr_t>(c.out) | a.out_pitch) & 31u) == 0;
    const LookupLaunch& l = !general ? (out32b ? p->launch_dense : p->launch_dense16) : (c.weights ? p->launch_gen_w : p->launch_gen);
    if (l.vec32) a.nvec = p->nvec_w;
    cudaError_t e;
    switch (p->dtype) {
        case DPI_F32: e = launch_lookup_f32(a, l, stream); break;
        case DPI_F16: e = launch_lookup_f16(a, l, stream); break;
        default: e = launch_lookup_bf16(a, l, stream); break;
    }
    if (e != cudaSuccess) return cuda_fail(e, "lookup kernel launch");
    return DPI_OK;
}

dpi_status_t check_lookup_pointers(const dpi_plan_t* p, const void* tables, const void* indices, const void* out) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (!p->built) return fail(DPI_ERR_INVALID_ARG, "plan has not been built (call dpi_plan_build first)");
    if (!tables || !out) return fail(DPI_ERR_INVALID_ARG, "table_ptrs_dev/out_dev is NULL");
    if (!indices && p->max_indices > 0) return fail(DPI_ERR_INVALID_ARG, "indices_dev is NULL");
    const uintptr_t out_align = (p->dtype != DPI_F32 && p->out_dtype == DPI_F32) ? 31u : 15u;
    if (reinterpret_cast<uintptr_t>(out) & out_align) return fail(DPI_ERR_INVALID_ARG, "out_dev is not %d-byte aligned", (int)out_align + 1);
    const uintptr_t idx_align = p->index_type == DPI_IDX_I64 ? 7u : 3u;
    if (reinterpret_cast<uintptr_t>(indices) & idx_align) return fail(DPI_ERR_INVALID_ARG, "indices_dev is not %d-byte aligned", (int)idx_align + 1);
    return DPI_OK;
}

PlanArgs plan_args(const dpi_plan_t* p, const int32_t* lengths_dev) {
    PlanArgs a{};
    a.len = lengths_dev;
    a.offsets = p->offsets;
    a.seg = p->seg;
    a.meta = p->meta;
    a.status = p->status;
    a.state = p->state;
    a.G = p->G;
    a.K = static_cast<uint32_t>(p->K);
    a.seg_cap = p->seg_cap;
    a.num_tiles = p->num_tiles;
    a.num_chunks = p->num_chunks;
    a.tiles_per_chunk = p->tiles_per_chunk;
    a.max_indices = static_cast<uint32_t>(p->max_indices);
    return a;
}

// Default ceiling of the fused single-launch path (bags). Measured on B200 (profiles/r02_forward_crossover.md):
// against planner + lookup WITHOUT a bag-length promise the single launch is within 3 % at worst (one id per bag, < 2e5 bags) and
// 6-22 % faster elsewhere, up to the size where a chunk no longer fits the kernel's 2048 bags (~1.2e6 bags at one wave). Against
// the PROMISED two-launch path it loses 11-24 % on one-hot batches below ~2e5 bags: see fused_eligible().
constexpr uint64_t kFusedDefaultMaxBags = 1u << 20;

// May this call run as ONE launch (forward_fused.cu)? Host-known facts only: the layout is the dense one, and the plan's
// capacity says bags are short on average (max_indices <= 8 * G) -- the fused kernel is correct for any bag length but
// does not balance load across CTAs, so long-bag batches keep the planner + balanced-segment lookup.
bool fused_eligible(const dpi_plan_t* p, const LookupCall& c) {
    if (p->fused_chunks == 0 || p->opt[DPI_OPT_FUSED] == 2 || p->opt[DPI_OPT_MODE] != 0 || p->off64) return false;
    if (c.force_general || p->mixed_dims || p->custom_columns || p->bag_order != DPI_BAGS_SAMPLE_MAJOR || c.weights || c.peers ||
        c.offsets || (c.out_ld && c.out_ld != p->out_width))
        return false;
    if (p->opt[DPI_OPT_FUSED] == 1) return true;
    // A caller who promised at most ONE id per bag gets planner + the lean short-bag launch below 4e5 bags: 7.5 / 8.1 / 9.3 / 11.3 us
    // against 8.3 / 10.0 / 10.6 / 13.2 us fused at 1.3e4 / 5.3e4 / 1.1e5 / 2.1e5 bags (the fused launch has nothing to amortise its
    // look-back over); from 4.3e5 bags on the single launch wins again (16.9 vs 18.6 us).
    if (p->opt[DPI_OPT_MAX_BAG_HINT] == 1 && p->G < 400000u) return false;
    const uint64_t max_bags = p->opt[DPI_OPT_FUSED_MAX_BAGS] > 0 ? static_cast<uint64_t>(p->opt[DPI_OPT_FUSED_MAX_BAGS]) : kFusedDefaultMaxBags;
    return p->G <= max_bags && static_cast<uint64_t>(p->max_indices) <= 8ull * p->G;
}

dpi_status_t launch_fused_forward(dpi_plan_t* p, const int32_t* lengths_dev, const LookupCall& c, cudaStream_t stream,
                                  float* fm_y = nullptr, float* fm_v = nullptr) {
    FusedArgs f{};
    f.plan = plan_args(p, lengths_dev);
    const bool fm = fm_y || fm_v;
    f.plan.num_chunks = fm ? p->fused_fm_chunks : p->fused_chunks;
    f.chunk_bags = fm ? p->fused_fm_chunk_bags : p->fused_chunk_bags;
    f.fm_y = fm_y;
    f.fm_v = fm_v;
    f.items = (f.chunk_bags + kFusedThreads - 1) / kFusedThreads;
    f.k_shift = 32;
    for (uint32_t b = 0; b < 31; ++b) if (static_cast<uint32_t>(p->K) == (1u << b)) f.k_shift = b;
    LookupArgs& a = f.look;
    a.tables = c.tables;
    a.indices = static_cast<const int32_t*>(c.indices);
    a.offsets = p->offsets;
    a.seg = p->seg;
    a.meta = p->meta;
    a.out = c.out;
    a.G = p->G;
    a.T = static_cast<uint32_t>(p->T);
    a.B = static_cast<uint32_t>(p->B);
    a.nvec = p->nvec;
    a.idx_shift = p->index_type == DPI_IDX_I64 ? 1u : 0u;
    std::memset(&a.pool, 0, sizeof a.pool);
    if (c.pooling) {
        for (int t = 0; t < p->T; ++t) {
            if (c.pooling[t] > 1) return fail(DPI_ERR_INVALID_ARG, "pooling[%d] = %d is not a dpi_pool_t", t, c.pooling[t]);
            if (c.pooling[t] == DPI_POOL_MEAN) {
                a.pool.w[t >> 5] |= 1u << (t & 31);
                f.any_mean = 1;
            }
        }
    }
    cudaError_t e = launch_fused(f, p->dtype, p->dtype != DPI_F32 && p->out_dtype == DPI_F32, p->lanes, p->opt[DPI_OPT_PDL] != 0, stream);
    if (e != cudaSuccess) return cuda_fail(e, "fused forward kernel launch");
    p->built = true;
    return DPI_OK;
}

// a1 + a2 + a3 on device-resident inputs: one launch when fused_eligible(), else the planner launch followed by the lookup.
dpi_status_t forward_device(dpi_plan_t* p, const int32_t* lengths_dev, const LookupCall& c, cudaStream_t stream) {
    if (fused_eligible(p, c)) return launch_fused_forward(p, lengths_dev, c, stream);
    dpi_status_t st = dpi_plan_build(p, lengths_dev, stream);
    if (st != DPI_OK) return st;
    return do_lookup(p, c, stream);
}

}  // namespace

extern "C" {

dpi_status_t dpi_plan_create(int32_t T, const int64_t* table_rows, const int32_t* dims, dpi_dtype_t dtype, int32_t B,
                             int64_t max_indices, dpi_plan_t** plan) {
    if (!plan) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    *plan = nullptr;
    if (!table_rows || !dims) return fail(DPI_ERR_INVALID_ARG, "table_rows/dims is NULL");
    if (T < 1 || B < 1) return fail(DPI_ERR_INVALID_ARG, "T=%d and B=%d must be >= 1", T, B);
    if (T > DPI_MAX_TABLES) return fail(DPI_ERR_UNSUPPORTED, "T=%d exceeds DPI_MAX_TABLES=%d", T, DPI_MAX_TABLES);
    if (dtype != DPI_F32 && dtype != DPI_F16 && dtype != DPI_BF16) return fail(DPI_ERR_INVALID_ARG, "unknown dtype %d", (int)dtype);
    if (max_indices < 0 || max_indices >= (1ll << 31)) return fail(DPI_ERR_INVALID_ARG, "max_indices=%lld outside [0, 2^31)", (long long)max_indices);
    const int64_t G64 = static_cast<int64_t>(B) * T;
    if (G64 >= (1ll << 31) || G64 + max_indices >= (1ll << 32) - 16) return fail(DPI_ERR_INVALID_ARG, "B*T=%lld too large", (long long)G64);
    const int elt = dtype == DPI_F32 ? 4 : 2;
    int32_t D = dims[0];
    bool mixed = false;
    int64_t out_width = 0;
    for (int t = 0; t < T; ++t) {
        if (dims[t] < 1) return fail(DPI_ERR_INVALID_ARG, "dims[%d]=%d", t, dims[t]);
        const int64_t rb = static_cast<int64_t>(dims[t]) * elt;
        if (rb % 16 != 0) return fail(DPI_ERR_UNSUPPORTED, "row size %lld B of table %d is not a multiple of 16 B", (long long)rb, t);
        if (rb > 512) return fail(DPI_ERR_UNSUPPORTED, "row size %lld B of table %d exceeds 512 B (one warp-wide 128-bit load)", (long long)rb, t);
        if (dims[t] != dims[0]) mixed = true;
        if (dims[t] > D) D = dims[t];
        out_width += dims[t];
        if (table_rows[t] < 1) return fail(DPI_ERR_INVALID_ARG, "table_rows[%d]=%lld must be >= 1", t, (long long)table_rows[t]);
        if (table_rows[t] > 0x7fffffffll) return fail(DPI_ERR_UNSUPPORTED, "table_rows[%d] exceeds int32 index range", t);
    }
    const int64_t row_bytes = static_cast<int64_t>(D) * elt;   // the widest table

    int dev = 0, n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev == 0) {
        (void)cudaGetLastError();
        return fail(DPI_ERR_CUDA, "no CUDA device (%s); libdpi has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    DPI_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    DPI_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return fail(DPI_ERR_UNSUPPORTED, "device sm_%d%d: libdpi is built for sm_100a only", prop.major, prop.minor);

    dpi_plan_t* p = new (std::nothrow) dpi_plan_s();
    if (!p) return fail(DPI_ERR_ALLOC, "host allocation failed");
    p->T = T; p->B = B; p->D = D; p->dtype = dtype; p->out_dtype = dtype;
    p->G = static_cast<uint32_t>(G64);
    p->max_indices = max_indices;
    p->nvec = static_cast<uint32_t>(row_bytes / 16);
    p->lanes = pow2ceil(static_cast<int>(p->nvec));
    p->nvec_w = static_cast<uint32_t>(row_bytes / 32);
    p->lanes_w = pow2ceil(static_cast<int>(p->nvec_w > 0 ? p->nvec_w : 1));
    p->table_rows.assign(table_rows, table_rows + T);
    p->dims.assign(dims, dims + T);
    p->mixed_dims = mixed;
    p->wide = wide_allowed(p, 0);
    p->out_width = out_width;
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;
    p->num_tiles = (p->G + kScanTile - 1) / kScanTile;
    {
        // planner grid: whole tiles per CTA, at most 2 CTAs per SM (all co-resident: 64 registers x 256 threads)
        uint32_t max_chunks = static_cast<uint32_t>(2 * p->num_sms);
        if (max_chunks > static_cast<uint32_t>(kMaxChunks)) max_chunks = kMaxChunks;
        if (max_chunks < 1) max_chunks = 1;
        p->tiles_per_chunk = (p->num_tiles + max_chunks - 1) / max_chunks;
        if (p->tiles_per_chunk < 1) p->tiles_per_chunk = 1;
        p->num_chunks = (p->num_tiles + p->tiles_per_chunk - 1) / p->tiles_per_chunk;
        if (p->num_chunks < 1) p->num_chunks = 1;
    }
    p->K = default_quantum(p);

#define DPI_TRY(call)                                   \
    do {                                                \
        cudaError_t e2_ = (call);                       \
        if (e2_ != cudaSuccess) {                       \
            dpi_status_t st_ = cuda_fail(e2_, #call);   \
            free_plan(p);                               \
            return st_;                                 \
        }                                               \
    } while (0)
    DPI_TRY(cudaMalloc(&p->offsets, (static_cast<size_t>(p->G) + 1) * sizeof(int32_t)));
    DPI_TRY(cudaMalloc(&p->meta, kMetaWords * sizeof(int32_t)));
    DPI_TRY(cudaMemset(p->meta, 0, kMetaWords * sizeof(int32_t)));
    DPI_TRY(cudaMalloc(&p->status, kStatusRecords * sizeof(ulonglong2)));
    DPI_TRY(cudaMemset(p->status, 0, kStatusRecords * sizeof(ulonglong2)));
    {
        // ticket, done, epoch = 1 (status words start at 0), overflowed builds, running min / max length
        const unsigned int init[kStateWords] = {0u, 0u, 1u, 0u, 0xffffffffu, 0u, 0u, 0u};
        DPI_TRY(cudaMalloc(&p->state, sizeof init));
        DPI_TRY(cudaMemcpy(p->state, init, sizeof init, cudaMemcpyHostToDevice));
    }
    DPI_TRY(cudaMalloc(&p->table_rows_dev, T * sizeof(int64_t)));
    DPI_TRY(cudaMemcpy(p->table_rows_dev, table_rows, T * sizeof(int64_t), cudaMemcpyHostToDevice));
    DPI_TRY(cudaMalloc(&p->n_bad_dev, 2 * sizeof(unsigned long long)));
    {
        std::vector<uint32_t> nv(T), col(T);
        uint32_t c = 0;
        for (int t = 0; t < T; ++t) {
            nv[t] = static_cast<uint32_t>(static_cast<int64_t>(dims[t]) * elt / 16);
            col[t] = c;
            c += nv[t];
        }
        DPI_TRY(cudaMalloc(&p->tab_nvec_dev, T * sizeof(uint32_t)));
        DPI_TRY(cudaMalloc(&p->tab_col_dev, T * sizeof(uint32_t)));
        DPI_TRY(cudaMemcpy(p->tab_nvec_dev, nv.data(), T * sizeof(uint32_t), cudaMemcpyHostToDevice));
        DPI_TRY(cudaMemcpy(p->tab_col_dev, col.data(), T * sizeof(uint32_t), cudaMemcpyHostToDevice));
    }
#undef DPI_TRY
    dpi_status_t st = ensure_seg_capacity(p, p->K);
    if (st != DPI_OK) { free_plan(p); return st; }
    prepare_launches(p);
    *plan = p;
    return DPI_OK;
}

dpi_status_t dpi_plan_set_quantum(dpi_plan_t* p, int32_t K) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (K < 0) return fail(DPI_ERR_INVALID_ARG, "K=%d must be >= 0", K);
    const int32_t K_new = K ? K : default_quantum(p);
    // the segment buffer may be re-allocated and the old records describe another quantum: whatever was built is gone
    p->built = false;
    dpi_status_t st = ensure_seg_capacity(p, K_new);
    if (st != DPI_OK) return st;   // K unchanged: the plan still matches its (old, intact or re-allocated larger) buffer
    p->K_user = K;
    p->K = K_new;
    prepare_launches(p);           // the persistent grid is capped by the segment capacity
    return DPI_OK;
}

dpi_status_t dpi_plan_set_option(dpi_plan_t* p, dpi_option_t opt, int32_t v) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    bool ok = false;
    switch (opt) {
        case DPI_OPT_UNROLL: ok = v == 0 || v == 2 || v == 4 || v == 8 || v == 16; break;
        case DPI_OPT_BLOCK_THREADS: ok = v == 0 || (v >= 32 && v <= 256 && v % 32 == 0); break;
        case DPI_OPT_BLOCKS_PER_SM: ok = v >= 0 && v <= 32; break;
        case DPI_OPT_MODE: ok = (v >= 0 && v <= 3) || v == 6; break;
        case DPI_OPT_ROW_L1_NO_ALLOC: ok = v == -1 || v == 0; break;  // the bypass variant was removed (see dpi.h)
        case DPI_OPT_PDL: ok = v == 0 || v == 1; break;
        case DPI_OPT_HOST_CHUNKS: ok = v >= 0 && v <= 64; break;
        case DPI_OPT_HOST_DIRECT_OUT: ok = v >= 0 && v <= 2; break;
        case DPI_OPT_MAX_BAG_HINT: ok = v >= 0; break;
        case DPI_OPT_FUSED: ok = v >= 0 && v <= 2; break;
        case DPI_OPT_FUSED_MAX_BAGS: ok = v >= 0; break;
        case DPI_OPT_VEC_BYTES: ok = v == 0 || v == 16 || v == 32; break;
        default: return fail(DPI_ERR_INVALID_ARG, "unknown option %d", (int)opt);
    }
    if (!ok) return fail(DPI_ERR_INVALID_ARG, "value %d not supported for option %d", v, (int)opt);
    if (p->opt[opt] == v) return DPI_OK;
    p->opt[opt] = v;
    if (opt == DPI_OPT_VEC_BYTES) {
        p->wide = wide_allowed(p, v);
        if (v == 32 && !p->wide) {
            p->opt[opt] = 0;
            return fail(DPI_ERR_UNSUPPORTED, "DPI_OPT_VEC_BYTES = 32 needs equal dims and a row size that is a multiple of 32 B");
        }
    }
    if (opt == DPI_OPT_UNROLL || opt == DPI_OPT_BLOCK_THREADS || opt == DPI_OPT_BLOCKS_PER_SM || opt == DPI_OPT_PDL || opt == DPI_OPT_VEC_BYTES)
        prepare_launches(p);
    return DPI_OK;
}

dpi_status_t dpi_plan_get_option(const dpi_plan_t* p, dpi_option_t opt, int32_t* v) {
    if (!p || !v || opt < 0 || opt >= DPI_OPT_COUNT_) return fail(DPI_ERR_INVALID_ARG, "bad argument");
    *v = p->opt[opt];
    return DPI_OK;
}

dpi_status_t dpi_plan_build(dpi_plan_t* p, const int32_t* lengths_dev, void* stream) {
    if (!p || !lengths_dev) return fail(DPI_ERR_INVALID_ARG, "plan/lengths_dev is NULL");
    if (reinterpret_cast<uintptr_t>(lengths_dev) & 3u) return fail(DPI_ERR_INVALID_ARG, "lengths_dev is not 4-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (p->off64) {
        Plan64Args b{};
        b.len = lengths_dev; b.offsets = p->offsets64; b.seg = p->seg; b.seg_off = p->seg_off64; b.meta = p->meta;
        b.agg = p->agg64; b.state = p->state; b.G = p->G; b.K = static_cast<unsigned long long>(p->K); b.seg_cap = p->seg_cap;
        b.num_tiles = p->num_tiles; b.num_chunks = p->num_chunks; b.tiles_per_chunk = p->tiles_per_chunk;
        b.max_indices = static_cast<unsigned long long>(p->max_indices);
        cudaError_t e64 = launch_plan64(b, s);
        if (e64 != cudaSuccess) return cuda_fail(e64, "64-bit plan kernel launch");
        p->built = true;
        return DPI_OK;
    }
    const PlanArgs a = plan_args(p, lengths_dev);
    cudaError_t e = launch_plan(a, s);
    if (e != cudaSuccess) return cuda_fail(e, "plan kernel launch");
    p->built = true;
    return DPI_OK;
}

dpi_status_t dpi_plan(const int64_t* table_rows, int32_t T, const int32_t* dims, dpi_dtype_t dtype,
                      const int32_t* lengths_dev, int32_t B, int64_t max_indices, void* stream, dpi_plan_t** plan) {
    dpi_status_t st = dpi_plan_create(T, table_rows, dims, dtype, B, max_indices, plan);
    if (st != DPI_OK) return st;
    st = dpi_plan_build(*plan, lengths_dev, stream);
    if (st != DPI_OK) {
        dpi_plan_destroy(*plan);
        *plan = nullptr;
    }
    return st;
}

dpi_status_t dpi_plan_device_views(const dpi_plan_t* p, const int32_t** offsets_dev, const int32_t** seg_dev,
                                   const int32_t** meta_dev) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (offsets_dev) *offsets_dev = p->off64 ? reinterpret_cast<const int32_t*>(p->offsets64) : p->offsets;
    if (seg_dev) *seg_dev = reinterpret_cast<const int32_t*>(p->seg);
    if (meta_dev) *meta_dev = p->meta;
    return DPI_OK;
}

dpi_status_t dpi_plan_info(const dpi_plan_t* p, int32_t* T, int32_t* B, int32_t* D, int32_t* dtype, int64_t* G,
                           int32_t* K, int64_t* seg_capacity) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (T) *T = p->T;
    if (B) *B = p->B;
    if (D) *D = p->D;
    if (dtype) *dtype = static_cast<int32_t>(p->dtype);
    if (G) *G = p->G;
    if (K) *K = p->K;
    if (seg_capacity) *seg_capacity = p->seg_cap;
    return DPI_OK;
}

dpi_status_t dpi_plan_export(const dpi_plan_t* p, int32_t* offsets_host, int32_t* seg_bag_host, int32_t* seg_off_host,
                             int64_t seg_cap, int32_t* S, int64_t* N, void* stream) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (!p->built) return fail(DPI_ERR_INVALID_ARG, "plan has not been built");
    if (p->off64) return fail(DPI_ERR_INVALID_ARG, "the plan holds 64-bit offsets: use dpi_plan_export64");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int32_t meta[kMetaWords];
    DPI_CUDA(cudaMemcpyAsync(meta, p->meta, sizeof meta, cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    if (meta[META_OVERFLOW]) return fail(DPI_ERR_INVALID_ARG, "batch has N=%u > max_indices=%lld (plan capacity exceeded)", static_cast<uint32_t>(meta[META_N]), (long long)p->max_indices);
    if (S) *S = meta[META_S];
    if (N) *N = static_cast<uint32_t>(meta[META_N]);
    if (offsets_host) DPI_CUDA(cudaMemcpyAsync(offsets_host, p->offsets, (static_cast<size_t>(p->G) + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    if (seg_bag_host || seg_off_host) {
        const size_t n = static_cast<size_t>(meta[META_S]) + 1;
        if (seg_cap < static_cast<int64_t>(n)) return fail(DPI_ERR_INVALID_ARG, "seg_cap=%lld < S+1=%zu", (long long)seg_cap, n);
        std::vector<int2> rec(n);
        DPI_CUDA(cudaMemcpyAsync(rec.data(), p->seg, n * sizeof(int2), cudaMemcpyDeviceToHost, s));
        DPI_CUDA(cudaStreamSynchronize(s));
        for (size_t i = 0; i < n; ++i) {
            if (seg_bag_host) seg_bag_host[i] = rec[i].x;
            if (seg_off_host) seg_off_host[i] = rec[i].y;
        }
    }
    DPI_CUDA(cudaStreamSynchronize(s));
    return DPI_OK;
}

dpi_status_t dpi_plan_set_offset_type(dpi_plan_t* p, dpi_offset_type_t type, int64_t max_indices) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (type != DPI_OFF_I32 && type != DPI_OFF_I64) return fail(DPI_ERR_INVALID_ARG, "unknown offset type %d", (int)type);
    if (max_indices == 0) max_indices = p->max_indices;
    const int64_t limit = type == DPI_OFF_I64 ? (1ll << 40) : (1ll << 31);
    if (max_indices < 0 || max_indices >= limit) return fail(DPI_ERR_INVALID_ARG, "max_indices=%lld outside [0, 2^%d)", (long long)max_indices, type == DPI_OFF_I64 ? 40 : 31);
    if (type == DPI_OFF_I32 && static_cast<int64_t>(p->G) + max_indices >= (1ll << 32) - 16) return fail(DPI_ERR_INVALID_ARG, "B*T + max_indices too large for 32-bit offsets");
    p->built = false;
    const bool was64 = p->off64;
    const int64_t was_max = p->max_indices;
    const int32_t was_K = p->K;
    p->off64 = type == DPI_OFF_I64;
    p->max_indices = max_indices;
    dpi_status_t st = DPI_OK;
    if (p->off64) {
        if (!p->offsets64) {
            cudaError_t e = cudaMalloc(&p->offsets64, (static_cast<size_t>(p->G) + 1) * sizeof(long long));
            if (e != cudaSuccess) st = cuda_fail(e, "cudaMalloc(offsets64)");
        }
        if (st == DPI_OK && !p->agg64) {
            cudaError_t e = cudaMalloc(&p->agg64, static_cast<size_t>(kMaxChunks) * 32);
            if (e != cudaSuccess) st = cuda_fail(e, "cudaMalloc(agg64)");
        }
    }
    if (st == DPI_OK) {
        if (!p->K_user) p->K = default_quantum(p);
        st = ensure_seg_capacity(p, p->K);
    }
    if (st != DPI_OK) {   // the plan keeps its previous offset type, capacity and quantum (the segment buffer is still sized for them)
        p->off64 = was64;
        p->max_indices = was_max;
        p->K = was_K;
        return st;
    }
    if (!p->off64 && was64) {   // dpi.h: the high words of N / C[G] are zero unless the plan holds 64-bit offsets
        cudaError_t e = cudaMemset(p->meta + META_N_HI, 0, 2 * sizeof(int32_t));
        if (e != cudaSuccess) return cuda_fail(e, "cudaMemset(meta high words)");
    }
    if (p->stage_idx) { (void)cudaFree(p->stage_idx); p->stage_idx = nullptr; p->stage_idx_bytes = 0; }
    free_pipeline(p);
    prepare_launches(p);
    return DPI_OK;
}

dpi_status_t dpi_plan_export64(const dpi_plan_t* p, int64_t* offsets_host, int32_t* seg_bag_host, int64_t* seg_off_host,
                               int64_t seg_cap, int64_t* S, int64_t* N, void* stream) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (!p->built) return fail(DPI_ERR_INVALID_ARG, "plan has not been built");
    if (!p->off64) return fail(DPI_ERR_INVALID_ARG, "the plan holds 32-bit offsets: use dpi_plan_export");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int32_t meta[kMetaWords];
    DPI_CUDA(cudaMemcpyAsync(meta, p->meta, sizeof meta, cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    const int64_t n_total = (static_cast<int64_t>(meta[META_N_HI]) << 32) | static_cast<uint32_t>(meta[META_N]);
    if (meta[META_OVERFLOW]) return fail(DPI_ERR_INVALID_ARG, "batch has N=%lld > max_indices=%lld (plan capacity exceeded)", (long long)n_total, (long long)p->max_indices);
    if (S) *S = meta[META_S];
    if (N) *N = n_total;
    if (offsets_host) DPI_CUDA(cudaMemcpyAsync(offsets_host, p->offsets64, (static_cast<size_t>(p->G) + 1) * sizeof(long long), cudaMemcpyDeviceToHost, s));
    const size_t n = static_cast<size_t>(meta[META_S]) + 1;
    if ((seg_bag_host || seg_off_host) && seg_cap < static_cast<int64_t>(n)) return fail(DPI_ERR_INVALID_ARG, "seg_cap=%lld < S+1=%zu", (long long)seg_cap, n);
    if (seg_bag_host) {
        std::vector<int2> rec(n);
        DPI_CUDA(cudaMemcpyAsync(rec.data(), p->seg, n * sizeof(int2), cudaMemcpyDeviceToHost, s));
        DPI_CUDA(cudaStreamSynchronize(s));
        for (size_t i = 0; i < n; ++i) seg_bag_host[i] = rec[i].x;
    }
    if (seg_off_host) DPI_CUDA(cudaMemcpyAsync(seg_off_host, p->seg_off64, n * sizeof(long long), cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    return DPI_OK;
}

dpi_status_t dpi_plan_stats(const dpi_plan_t* p, int32_t* min_len, int32_t* max_len, void* stream) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (!p->built) return fail(DPI_ERR_INVALID_ARG, "plan has not been built");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int32_t meta[kMetaWords];
    DPI_CUDA(cudaMemcpyAsync(meta, p->meta, sizeof meta, cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    if (min_len) *min_len = meta[META_MINLEN];
    if (max_len) *max_len = meta[META_MAXLEN];
    return DPI_OK;
}

dpi_status_t dpi_plan_set_out_dtype(dpi_plan_t* p, dpi_dtype_t out_dtype) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (out_dtype != p->dtype && out_dtype != DPI_F32) return fail(DPI_ERR_UNSUPPORTED, "output dtype %d: must be the table dtype or DPI_F32", (int)out_dtype);
    if (p->out_dtype != out_dtype) {
        p->out_dtype = out_dtype;
        prepare_launches(p);
    }
    return DPI_OK;
}

dpi_status_t dpi_lookup(const void* const* table_ptrs_dev, const int32_t* indices_dev, const int32_t* offsets_dev,
                        const dpi_plan_t* p, const uint8_t* pooling, void* out_dev, void* stream) {
    dpi_status_t st = check_lookup_pointers(p, table_ptrs_dev, indices_dev, out_dev);
    if (st != DPI_OK) return st;
    LookupCall c;
    c.tables = table_ptrs_dev; c.indices = indices_dev; c.offsets = offsets_dev; c.pooling = pooling; c.out = out_dev;
    return do_lookup(p, c, static_cast<cudaStream_t>(stream));
}

dpi_status_t dpi_lookup_ex(const dpi_lookup_args_t* args, const dpi_plan_t* p, void* stream) {
    if (!args) return fail(DPI_ERR_INVALID_ARG, "args is NULL");
    if (args->struct_size != sizeof(dpi_lookup_args_t)) return fail(DPI_ERR_INVALID_ARG, "args->struct_size=%u, expected %zu", args->struct_size, sizeof(dpi_lookup_args_t));
    dpi_status_t st = check_lookup_pointers(p, args->table_ptrs_dev, args->indices_dev,
                                            args->out_peers_dev ? static_cast<const void*>(args->out_peers_dev) : args->out_dev);
    if (st != DPI_OK) return st;
    if (reinterpret_cast<uintptr_t>(args->weights_dev) & 3u) return fail(DPI_ERR_INVALID_ARG, "weights_dev is not 4-byte aligned");
    if (args->out_ld < 0) return fail(DPI_ERR_INVALID_ARG, "out_ld=%lld", (long long)args->out_ld);
    LookupCall c;
    c.tables = args->table_ptrs_dev; c.indices = args->indices_dev; c.offsets = args->offsets_dev;
    c.weights = args->weights_dev; c.pooling = args->pooling; c.out = args->out_dev; c.out_ld = args->out_ld;
    c.peers = args->out_peers_dev; c.n_peers = args->n_peers; c.rows_per_peer = args->rows_per_peer;
    c.force_general = (args->flags & DPI_LOOKUP_FORCE_GENERAL) != 0;
    return do_lookup(p, c, static_cast<cudaStream_t>(stream));
}

dpi_status_t dpi_forward(dpi_plan_t* p, const int32_t* lengths_dev, const void* const* table_ptrs_dev, const void* indices_dev,
                         const uint8_t* pooling, void* out_dev, void* stream) {
    if (!p || !lengths_dev) return fail(DPI_ERR_INVALID_ARG, "plan/lengths_dev is NULL");
    if (reinterpret_cast<uintptr_t>(lengths_dev) & 3u) return fail(DPI_ERR_INVALID_ARG, "lengths_dev is not 4-byte aligned");
    const bool was_built = p->built;
    p->built = true;   // check_lookup_pointers only wants a plan that will be built by the time the lookup runs
    dpi_status_t st = check_lookup_pointers(p, table_ptrs_dev, indices_dev, out_dev);
    p->built = was_built;
    if (st != DPI_OK) return st;
    LookupCall c;
    c.tables = table_ptrs_dev; c.indices = indices_dev; c.pooling = pooling; c.out = out_dev;
    return forward_device(p, lengths_dev, c, static_cast<cudaStream_t>(stream));
}

dpi_status_t dpi_forward_fm(dpi_plan_t* p, const int32_t* lengths_dev, const void* const* table_ptrs_dev, const void* indices_dev,
                            const uint8_t* pooling, void* out_dev, float* y_dev, float* v_dev, void* stream) {
    if (!p || !lengths_dev) return fail(DPI_ERR_INVALID_ARG, "plan/lengths_dev is NULL");
    if (!y_dev && !v_dev) return fail(DPI_ERR_INVALID_ARG, "dpi_forward_fm: neither y_dev nor v_dev given");
    if ((reinterpret_cast<uintptr_t>(lengths_dev) & 3u) || (reinterpret_cast<uintptr_t>(y_dev) & 3u) || (reinterpret_cast<uintptr_t>(v_dev) & 15u))
        return fail(DPI_ERR_INVALID_ARG, "dpi_forward_fm: misaligned pointer");
    if (p->mixed_dims || p->custom_columns || p->bag_order != DPI_BAGS_SAMPLE_MAJOR)
        return fail(DPI_ERR_UNSUPPORTED, "dpi_forward_fm needs one common dim, default columns and sample-major bags");
    const bool was_built = p->built;
    p->built = true;
    dpi_status_t st = check_lookup_pointers(p, table_ptrs_dev, indices_dev, out_dev);
    p->built = was_built;
    if (st != DPI_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    LookupCall c;
    c.tables = table_ptrs_dev; c.indices = indices_dev; c.pooling = pooling; c.out = out_dev;
    // one launch: the fused forward kernel with chunks of whole samples and the FM epilogue
    if (fused_eligible(p, c) && p->fused_fm_chunks != 0 && p->out_dtype == p->dtype)
        return launch_fused_forward(p, lengths_dev, c, s, y_dev, v_dev);
    // otherwise the chain: dpi_forward, then fm_kernel on the block it wrote (same per-sample arithmetic)
    st = forward_device(p, lengths_dev, c, s);
    if (st != DPI_OK) return st;
    cudaError_t e = launch_fm(out_dev, p->out_dtype, static_cast<uint32_t>(p->B), static_cast<uint32_t>(p->T), static_cast<uint32_t>(p->D),
                              static_cast<uint64_t>(p->out_width) * out_elt_bytes(p), y_dev, v_dev, s);
    if (e != cudaSuccess) return cuda_fail(e, "fm_kernel launch");
    return DPI_OK;
}

dpi_status_t dpi_plan_status(const dpi_plan_t* p, int32_t* overflowed_builds, void* stream) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    unsigned int n = 0;
    DPI_CUDA(cudaMemcpyAsync(&n, p->state + kStateOverflows, sizeof n, cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    if (overflowed_builds) *overflowed_builds = static_cast<int32_t>(n > 0x7fffffffu ? 0x7fffffffu : n);
    if (n == 0) return DPI_OK;
    DPI_CUDA(cudaMemsetAsync(p->state + kStateOverflows, 0, sizeof n, s));   // reported once
    return fail(DPI_ERR_INVALID_ARG, "%u build(s) since the last dpi_plan_status exceeded the plan's capacity (N > max_indices=%lld): "
                "their plans were left with S = 0 and the lookups launched on them wrote nothing (only dpi_forward's fused single launch "
                "pools such a batch anyway)", n, (long long)p->max_indices);
}

dpi_status_t dpi_lookup_input_first(const void* const* table_ptrs_dev, const int32_t* indices_dev, const int32_t* offsets_dev,
                                    const dpi_plan_t* p, const uint8_t* pooling, void* out_dev, void* stream) {
    dpi_status_t st = check_lookup_pointers(p, table_ptrs_dev, indices_dev, out_dev);
    if (st != DPI_OK) return st;
    LookupCall c;
    c.tables = table_ptrs_dev; c.indices = indices_dev; c.offsets = offsets_dev; c.pooling = pooling; c.out = out_dev;
    return do_lookup(p, c, static_cast<cudaStream_t>(stream), true);
}

dpi_status_t dpi_lookup_onehot(const void* const* table_ptrs_dev, const void* ids_dev, const dpi_plan_t* p, void* out_dev,
                               void* stream) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (!table_ptrs_dev || !ids_dev || !out_dev) return fail(DPI_ERR_INVALID_ARG, "table_ptrs_dev/ids_dev/out_dev is NULL");
    if (p->mixed_dims || p->custom_columns || p->bag_order != DPI_BAGS_SAMPLE_MAJOR || p->out_dtype != p->dtype)
        return fail(DPI_ERR_UNSUPPORTED, "dpi_lookup_onehot covers equal dims, sample-major ids, default columns and table-dtype output only");
    if (reinterpret_cast<uintptr_t>(out_dev) & 15u) return fail(DPI_ERR_INVALID_ARG, "out_dev is not 16-byte aligned");
    const bool i64 = p->index_type == DPI_IDX_I64;
    if (reinterpret_cast<uintptr_t>(ids_dev) & (i64 ? 7u : 3u)) return fail(DPI_ERR_INVALID_ARG, "ids_dev is misaligned");
    cudaError_t e = launch_onehot(table_ptrs_dev, ids_dev, i64 ? 1u : 0u, out_dev, p->G, static_cast<uint32_t>(p->T), p->nvec,
                                  p->lanes, p->num_sms, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "onehot_kernel launch");
    return DPI_OK;
}

dpi_status_t dpi_plan_set_layout(dpi_plan_t* p, dpi_bag_order_t order, dpi_index_type_t index_type) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    if (order != DPI_BAGS_SAMPLE_MAJOR && order != DPI_BAGS_TABLE_MAJOR) return fail(DPI_ERR_INVALID_ARG, "unknown bag order %d", (int)order);
    if (index_type != DPI_IDX_I32 && index_type != DPI_IDX_I64) return fail(DPI_ERR_INVALID_ARG, "unknown index type %d", (int)index_type);
    const bool changed = p->index_type != index_type;
    p->bag_order = order;
    p->index_type = index_type;
    if (changed) prepare_launches(p);   // int64 ids double the staged index words of the general kernel
    return DPI_OK;
}

dpi_status_t dpi_plan_set_columns(dpi_plan_t* p, const int64_t* columns) {
    if (!p) return fail(DPI_ERR_INVALID_ARG, "plan is NULL");
    const int elt = p->dtype == DPI_F32 ? 4 : 2;
    std::vector<uint32_t> col(p->T);
    int64_t width = 0;
    if (columns) {
        for (int t = 0; t < p->T; ++t) {
            if (columns[t] < 0 || (columns[t] * elt) % 16 != 0) return fail(DPI_ERR_INVALID_ARG, "columns[%d]=%lld must be >= 0 and 16-byte aligned", t, (long long)columns[t]);
            if (columns[t] * elt / 16 > 0x7fffffffll) return fail(DPI_ERR_INVALID_ARG, "columns[%d] too large", t);
            col[t] = static_cast<uint32_t>(columns[t] * elt / 16);
            width = std::max<int64_t>(width, columns[t] + p->dims[t]);
        }
    } else {
        uint32_t c = 0;
        for (int t = 0; t < p->T; ++t) {
            col[t] = c;
            c += static_cast<uint32_t>(static_cast<int64_t>(p->dims[t]) * elt / 16);
            width += p->dims[t];
        }
    }
    DPI_CUDA(cudaMemcpy(p->tab_col_dev, col.data(), p->T * sizeof(uint32_t), cudaMemcpyHostToDevice));
    p->custom_columns = columns != nullptr;
    if (columns) p->columns.assign(columns, columns + p->T); else p->columns.clear();
    p->out_width = width;
    if (p->stage_out) { DPI_CUDA(cudaFree(p->stage_out)); p->stage_out = nullptr; }
    free_pipeline(p);
    return DPI_OK;
}

dpi_status_t dpi_plan_out_width(const dpi_plan_t* p, int64_t* width) {
    if (!p || !width) return fail(DPI_ERR_INVALID_ARG, "NULL argument");
    *width = p->out_width;
    return DPI_OK;
}

namespace {

// Sum of lengths[g0, g1) and whether any of them is negative: branch-free so that the host compiler vectorises it (the
// loop runs once per dpi_forward_host call over all G lengths; with an early return inside it cost 0.15 ms at G = 360 K).
bool sum_lengths(const int32_t* lengths, size_t g0, size_t g1, int64_t* total) {
    int64_t sum = 0;
    int32_t sign = 0;
    for (size_t g = g0; g < g1; ++g) {
        sum += lengths[g];
        sign |= lengths[g];
    }
    *total = sum;
    return sign < 0;
}

int host_chunks(const dpi_plan_t* p, size_t bytes_moved) {
    if (p->bag_order == DPI_BAGS_TABLE_MAJOR) return 1;  // a chunk of samples is not a contiguous run of bags
    int n = p->opt[DPI_OPT_HOST_CHUNKS];
    if (n == 0) {  // auto: ~16 MB of PCIe traffic per chunk, at most 8 chunks; small batches stay in one piece
        n = static_cast<int>(bytes_moved / (16u << 20));
        if (n > 8) n = 8;
        if (n < 2) n = 1;
    }
    if (n > p->B) n = p->B;
    return n < 1 ? 1 : n;
}

// A chunk's sub-plan follows its parent's layout and options: output dtype, id width, column placement (the sub-plan writes
// rows of the parent's width at the parent's columns), quantum and tuning knobs. Launch configurations are re-derived only
// when something changed.
dpi_status_t sync_subplan(const dpi_plan_t* p, dpi_plan_t* q) {
    bool changed = q->out_dtype != p->out_dtype || q->index_type != p->index_type;
    q->out_dtype = p->out_dtype;
    q->index_type = p->index_type;
    q->bag_order = p->bag_order;
    for (int o = 0; o < DPI_OPT_COUNT_; ++o) {
        changed |= q->opt[o] != p->opt[o];
        q->opt[o] = p->opt[o];
    }
    q->wide = wide_allowed(q, q->opt[DPI_OPT_VEC_BYTES]);
    if (p->custom_columns != q->custom_columns || p->columns != q->columns) {
        dpi_status_t st = dpi_plan_set_columns(q, p->custom_columns ? p->columns.data() : nullptr);
        if (st != DPI_OK) return st;
    }
    if (p->K_user && q->K != p->K_user) return dpi_plan_set_quantum(q, p->K_user);   // re-derives the launches as well
    if (changed) prepare_launches(q);
    return DPI_OK;
}

dpi_status_t ensure_pipeline(dpi_plan_t* p, int n_chunks) {
    if (p->pipe && p->pipe->n_requested == n_chunks) return DPI_OK;
    free_pipeline(p);
    HostPipeline* h = new (std::nothrow) HostPipeline();
    if (!h) return fail(DPI_ERR_ALLOC, "host allocation failed");
    p->pipe = h;
    h->n_requested = n_chunks;
    for (int i = 0; i < HostPipeline::kStreams; ++i) {
        DPI_CUDA(cudaStreamCreateWithFlags(&h->st[i], cudaStreamNonBlocking));
        DPI_CUDA(cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming));
    }
    DPI_CUDA(cudaEventCreateWithFlags(&h->ev_in, cudaEventDisableTiming));
    // Chunk sizes: the device -> host stream of the output block is the bottleneck and cannot start before the first chunk
    // has been copied in and pooled, so the first chunk is a quarter of the others (c5, 8 chunks: the output stream starts
    // after ~0.07 ms instead of ~0.26 ms); the rest are equal.
    std::vector<int32_t> sizes;
    if (n_chunks >= 4 && p->B >= 4 * n_chunks) {
        const int32_t first = std::max<int32_t>(1, p->B / (4 * n_chunks));
        const int32_t rest = p->B - first, m = n_chunks - 1;
        sizes.push_back(first);
        for (int i = 0; i < m; ++i) sizes.push_back(rest / m + (i < rest % m ? 1 : 0));
    } else {
        const int32_t per = (p->B + n_chunks - 1) / n_chunks;
        for (int32_t lo = 0; lo < p->B; lo += per) sizes.push_back(std::min(per, p->B - lo));
    }
    int32_t lo = 0;
    for (int32_t Bc : sizes) {
        dpi_plan_t* q = nullptr;
        dpi_status_t st = dpi_plan_create(p->T, p->table_rows.data(), p->dims.data(), p->dtype, Bc, p->max_indices, &q);
        if (st != DPI_OK) return st;
        h->sub.push_back(q);
        h->sample_lo.push_back(lo);
        lo += Bc;
    }
    h->sample_lo.push_back(p->B);
    return DPI_OK;
}

}  // namespace

dpi_status_t dpi_forward_host(dpi_plan_t* p, const void* const* table_ptrs_dev, const int32_t* lengths_host,
                              const void* indices_host, int64_t n_indices, const uint8_t* pooling, void* out_host,
                              void* stream) {
    if (!p || !table_ptrs_dev || !lengths_host || !out_host) return fail(DPI_ERR_INVALID_ARG, "NULL argument");
    if (p->off64) return fail(DPI_ERR_UNSUPPORTED, "dpi_forward_host covers 32-bit offsets only (N < 2^31 per call)");
    if (n_indices < 0 || n_indices > p->max_indices) return fail(DPI_ERR_INVALID_ARG, "n_indices=%lld outside [0, max_indices=%lld]", (long long)n_indices, (long long)p->max_indices);
    if (n_indices > 0 && !indices_host) return fail(DPI_ERR_INVALID_ARG, "indices_host is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t oelt = out_elt_bytes(p);
    const size_t out_bytes = static_cast<size_t>(p->B) * p->out_width * oelt;
    const size_t idx_elt = p->index_type == DPI_IDX_I64 ? 8 : 4;
    const size_t idx_bytes = (static_cast<size_t>(p->max_indices) + 4) * idx_elt;
    if (!p->stage_len) DPI_CUDA(cudaMalloc(&p->stage_len, static_cast<size_t>(p->G) * sizeof(int32_t)));
    if (p->stage_idx_bytes < idx_bytes) {
        if (p->stage_idx) DPI_CUDA(cudaFree(p->stage_idx));
        p->stage_idx = nullptr; p->stage_idx_bytes = 0;
        DPI_CUDA(cudaMalloc(&p->stage_idx, idx_bytes));
        p->stage_idx_bytes = idx_bytes;
    }

    // Direct output: if out_host is page-locked and mapped into this device's address space, the lookup stores into
    // it over PCIe and the separate device->host copy disappears (DPI_OPT_HOST_DIRECT_OUT).
    char* out_direct = nullptr;
    if (p->opt[DPI_OPT_HOST_DIRECT_OUT] != 1) {
        cudaPointerAttributes pa{};
        if (cudaPointerGetAttributes(&pa, out_host) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer &&
            (reinterpret_cast<uintptr_t>(pa.devicePointer) & 31u) == 0) {
            out_direct = static_cast<char*>(pa.devicePointer);
        } else {
            (void)cudaGetLastError();
            if (p->opt[DPI_OPT_HOST_DIRECT_OUT] == 2)
                return fail(DPI_ERR_INVALID_ARG, "DPI_OPT_HOST_DIRECT_OUT = 2 but out_host is not page-locked device-mapped memory (32-byte aligned)");
        }
    }
    if (!out_direct && !p->stage_out) DPI_CUDA(cudaMalloc(&p->stage_out, static_cast<size_t>(p->B) * p->out_width * 4));
    char* const out_base = out_direct ? out_direct : static_cast<char*>(p->stage_out);

    // with direct output only the inputs cross PCIe as copies; the chunking then follows the input bytes alone
    const int n_chunks = host_chunks(p, static_cast<size_t>(p->G) * 4 + static_cast<size_t>(n_indices) * idx_elt + out_bytes);
    if (n_chunks <= 1) {
        int64_t total = 0;  // same host-side check as the pipelined path: the lengths must add up to n_indices
        if (sum_lengths(lengths_host, 0, p->G, &total)) return fail(DPI_ERR_INVALID_ARG, "lengths_host holds a negative length");
        if (total != n_indices) return fail(DPI_ERR_INVALID_ARG, "n_indices=%lld but the lengths sum to %lld", (long long)n_indices, (long long)total);
        DPI_CUDA(cudaMemcpyAsync(p->stage_len, lengths_host, static_cast<size_t>(p->G) * sizeof(int32_t), cudaMemcpyHostToDevice, s));
        if (n_indices) DPI_CUDA(cudaMemcpyAsync(p->stage_idx, indices_host, static_cast<size_t>(n_indices) * idx_elt, cudaMemcpyHostToDevice, s));
        LookupCall c;
        c.tables = table_ptrs_dev; c.indices = p->stage_idx; c.pooling = pooling; c.out = out_base;
        dpi_status_t st = forward_device(p, p->stage_len, c, s);   // one launch when eligible, else plan + lookup
        if (st != DPI_OK) return st;
        if (!out_direct) DPI_CUDA(cudaMemcpyAsync(out_host, p->stage_out, out_bytes, cudaMemcpyDeviceToHost, s));
        DPI_CUDA(cudaStreamSynchronize(s));
        return DPI_OK;
    }

    // ---- pipelined: chunks of whole samples, each an independent sub-batch with its own device plan ----
    dpi_status_t st = ensure_pipeline(p, n_chunks);
    if (st != DPI_OK) return st;
    HostPipeline* h = p->pipe;
    const size_t n_sub = h->sub.size();
    // Copy sizes only: how many index entries belong to each chunk (the plan itself -- offsets, segments -- is still
    // computed on the device, per chunk). The host adds up a chunk's lengths right before it enqueues that chunk, so the
    // sums of the later chunks run under the transfers of the earlier ones.
    DPI_CUDA(cudaEventRecord(h->ev_in, s));
    for (int i = 0; i < HostPipeline::kStreams; ++i) DPI_CUDA(cudaStreamWaitEvent(h->st[i], h->ev_in, 0));
    const size_t row_bytes = static_cast<size_t>(p->out_width) * oelt;
    int64_t e0 = 0;
    dpi_status_t bad = DPI_OK;
    for (size_t c = 0; c < n_sub && bad == DPI_OK; ++c) {
        cudaStream_t cs = h->st[c % HostPipeline::kStreams];
        dpi_plan_t* q = h->sub[c];
        const size_t g0 = static_cast<size_t>(h->sample_lo[c]) * p->T;
        const size_t n_g = static_cast<size_t>(q->G);
        int64_t n_e = 0;
        if (sum_lengths(lengths_host, g0, g0 + n_g, &n_e)) { bad = fail(DPI_ERR_INVALID_ARG, "lengths_host holds a negative length"); break; }
        if (e0 + n_e > n_indices) { bad = fail(DPI_ERR_INVALID_ARG, "n_indices=%lld but the lengths sum to more", (long long)n_indices); break; }
        bad = sync_subplan(p, q);
        if (bad != DPI_OK) break;
        char* idx_dev = static_cast<char*>(p->stage_idx) + static_cast<size_t>(e0) * idx_elt;
        char* out_dev = out_base + static_cast<size_t>(h->sample_lo[c]) * row_bytes;
        cudaError_t ce = cudaMemcpyAsync(p->stage_len + g0, lengths_host + g0, n_g * sizeof(int32_t), cudaMemcpyHostToDevice, cs);
        if (ce == cudaSuccess && n_e)
            ce = cudaMemcpyAsync(idx_dev, static_cast<const char*>(indices_host) + static_cast<size_t>(e0) * idx_elt,
                                 static_cast<size_t>(n_e) * idx_elt, cudaMemcpyHostToDevice, cs);
        if (ce != cudaSuccess) { bad = cuda_fail(ce, "cudaMemcpyAsync (host -> device)"); break; }
        LookupCall lc;
        lc.tables = table_ptrs_dev; lc.indices = idx_dev; lc.pooling = pooling; lc.out = out_dev;
        bad = forward_device(q, p->stage_len + g0, lc, cs);
        if (bad != DPI_OK) break;
        if (!out_direct) {
            ce = cudaMemcpyAsync(static_cast<char*>(out_host) + static_cast<size_t>(h->sample_lo[c]) * row_bytes, out_dev,
                                 static_cast<size_t>(q->B) * row_bytes, cudaMemcpyDeviceToHost, cs);
            if (ce != cudaSuccess) { bad = cuda_fail(ce, "cudaMemcpyAsync (device -> host)"); break; }
        }
        e0 += n_e;
    }
    if (bad == DPI_OK && e0 != n_indices) bad = fail(DPI_ERR_INVALID_ARG, "n_indices=%lld but the lengths sum to %lld", (long long)n_indices, (long long)e0);
    if (bad != DPI_OK) {   // chunks already enqueued run to completion before the error is returned (out_host is then undefined)
        char keep[sizeof g_err];
        std::memcpy(keep, g_err, sizeof keep);
        for (int i = 0; i < HostPipeline::kStreams; ++i) (void)cudaStreamSynchronize(h->st[i]);
        (void)cudaGetLastError();
        std::memcpy(g_err, keep, sizeof keep);
        return bad;
    }
    for (int i = 0; i < HostPipeline::kStreams; ++i) {
        DPI_CUDA(cudaEventRecord(h->ev_done[i], h->st[i]));
        DPI_CUDA(cudaStreamWaitEvent(s, h->ev_done[i], 0));
    }
    DPI_CUDA(cudaStreamSynchronize(s));
    return DPI_OK;
}

dpi_status_t dpi_check_indices(const dpi_plan_t* p, const void* indices_dev, int64_t* n_bad, void* stream) {
    if (!p || !n_bad) return fail(DPI_ERR_INVALID_ARG, "NULL argument");
    if (!p->built) return fail(DPI_ERR_INVALID_ARG, "plan has not been built");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    DPI_CUDA(cudaMemsetAsync(p->n_bad_dev, 0, 2 * sizeof(unsigned long long), s));
    CheckArgs a{};
    a.indices = indices_dev;
    a.offsets = p->off64 ? reinterpret_cast<const int32_t*>(p->offsets64) : p->offsets;
    a.off64 = p->off64;
    a.table_rows = p->table_rows_dev;
    a.n_bad = p->n_bad_dev;
    a.max_bag = p->opt[DPI_OPT_MAX_BAG_HINT];
    a.G = p->G;
    a.T = static_cast<uint32_t>(p->T);
    a.B = static_cast<uint32_t>(p->B);
    a.idx64 = p->index_type == DPI_IDX_I64;
    a.table_major = p->bag_order == DPI_BAGS_TABLE_MAJOR;
    cudaError_t e = launch_check_indices(a, s);
    if (e != cudaSuccess) return cuda_fail(e, "check_indices launch");
    unsigned long long counts[2] = {0, 0};
    DPI_CUDA(cudaMemcpyAsync(counts, p->n_bad_dev, sizeof counts, cudaMemcpyDeviceToHost, s));
    DPI_CUDA(cudaStreamSynchronize(s));
    *n_bad = static_cast<int64_t>(counts[0]);
    if (counts[0]) return fail(DPI_ERR_INDEX_RANGE, "%llu indices outside [0, table_rows[t])", counts[0]);
    if (counts[1]) return fail(DPI_ERR_INVALID_ARG, "%llu bags are longer than the promised DPI_OPT_MAX_BAG_HINT = %d", counts[1], a.max_bag);
    return DPI_OK;
}

dpi_status_t dpi_plan_destroy(dpi_plan_t* p) {
    if (!p) return DPI_OK;
    free_plan(p);
    return DPI_OK;
}

int64_t dpi_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
int32_t dpi_version(void) { return DPI_VERSION; }

const char* dpi_status_string(dpi_status_t st) {
    switch (st) {
        case DPI_OK: return "DPI_OK";
        case DPI_ERR_INVALID_ARG: return "DPI_ERR_INVALID_ARG";
        case DPI_ERR_UNSUPPORTED: return "DPI_ERR_UNSUPPORTED";
        case DPI_ERR_ALLOC: return "DPI_ERR_ALLOC";
        case DPI_ERR_CUDA: return "DPI_ERR_CUDA";
        case DPI_ERR_INDEX_RANGE: return "DPI_ERR_INDEX_RANGE";
        default: return "DPI_ERR_UNKNOWN";
    }
}

const char* dpi_last_error(void) { return g_err; }

}  // extern "C"
