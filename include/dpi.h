/*
 * dpi.h -- C ABI of the B200-native fused multi-table embedding lookup (DPIFrame, arxiv 2606.21101).
 *
 * The path (citations are /root/reference/PAPER.md line numbers; DESIGN.md has the full readings):
 *
 *   a1  plan: offset scan        "the overall embedding workload is deterministic and known in advance"
 *                                (PAPER.md:109), sizes computed before the traversal (Alg. 1 lines 1-2,
 *                                PAPER.md:150-151); multi-hot "by marking offset information"
 *   a2  plan: balanced segments  workload allocation across threads, output-first: adjacent workers own
 *                                adjacent output addresses (§IV-C)
 *   a3  fused gather-and-pool    Algorithm 1 "Multi-table Lookup" generalised to bags:
 *                                one pass writes the concatenated EmbedOut[b x (k*d)]
 *
 * Notation: T tables (the paper's k), B samples (b), D embedding dim (d), G = B*T bags,
 * bag id g = b*T + t (sample-major, Alg. 1 line 7 "IDs[row*k + table_id]"),
 * len[g] bag length, N = sum len, K = cost quantum of a segment.
 *
 * Plan definition (integer, one correct answer; checked bit for bit against oracle/):
 *   offsets[0] = 0, offsets[g+1] = offsets[g] + len[g]
 *   C[0] = 0,       C[g+1] = C[g] + max(len[g], 1)
 *   S = ceil(C[G] / K)
 *   seg_bag[s] = min(G, min{ g in [0,G] : C[g] >= s*K })   for s = 0..S
 *   seg_off[s] = offsets[seg_bag[s]]                       (first index entry of task s)
 *   warp-task s owns bags [seg_bag[s], seg_bag[s+1]) = entries [seg_off[s], seg_off[s+1]).
 *
 * Lookup definition: for every bag g = (b,t), c < D
 *   acc[c] = sum_{j in [offsets[g], offsets[g+1])} float(table_t[indices[j]][c])     (fp32 accumulate)
 *   if pooling[t] == MEAN and len > 0: acc[c] /= len;   empty bag -> +0.0
 *   out[b, t*D + c] = cast_to_table_dtype(acc[c])       (one RNE cast at the store)
 *
 * Conventions for every entry point
 *   - extern "C"; nothing throws across the boundary; every call returns dpi_status_t.
 *   - "host" pointers are ordinary CPU memory; "device" pointers are CUDA device memory of the current
 *     device. The library never takes torch types.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Caller owns tables, table_ptrs, lengths, indices, out. The library owns everything inside dpi_plan_t.
 *   - Asynchronous calls (dpi_plan_build, dpi_lookup, dpi_check_indices without result read) only enqueue
 *     work; device-side faults surface at the caller's next synchronisation.
 *   - There is NO CPU fallback: without a CUDA device every call that needs one returns DPI_ERR_CUDA.
 *   - A plan is not thread-safe; distinct plans are independent: every launch configuration (occupancy, shared-memory
 *     attribute) is derived when the plan is created or re-configured and stored in the plan, so two host threads may
 *     drive two plans on two streams concurrently. A plan belongs to the device that was current in dpi_plan_create;
 *     make that device current for every call that takes the plan. dpi_lookup / dpi_forward make no CUDA runtime call
 *     other than the kernel launch itself.
 */
#ifndef DPI_H_
#define DPI_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DPI_VERSION 100       /* 0.1.0 */
#define DPI_MAX_TABLES 2048   /* pooling modes travel to the kernel as a by-value bit mask */

typedef struct dpi_plan_s dpi_plan_t; /* opaque, library-owned */

typedef enum {
    DPI_OK = 0,
    DPI_ERR_INVALID_ARG = 1,  /* NULL, non-positive sizes, misaligned pointers, capacity exceeded */
    DPI_ERR_UNSUPPORTED = 2,  /* row size not a multiple of 16 B or > 512 B, T > DPI_MAX_TABLES, weights + mean */
    DPI_ERR_ALLOC = 3,        /* host or device allocation failed */
    DPI_ERR_CUDA = 4,         /* CUDA runtime error (text in dpi_last_error) */
    DPI_ERR_INDEX_RANGE = 5   /* dpi_check_indices found indices outside [0, table_rows[t]) */
} dpi_status_t;

typedef enum { DPI_F32 = 0, DPI_F16 = 1, DPI_BF16 = 2 } dpi_dtype_t;
typedef enum { DPI_POOL_SUM = 0, DPI_POOL_MEAN = 1 } dpi_pool_t;
/* Order of the bags in lengths / offsets / indices (interface variant, see dpi_plan_set_layout). */
typedef enum {
    DPI_BAGS_SAMPLE_MAJOR = 0, /* g = b*T + t: Alg. 1 line 7 "IDs[row*k + table_id]" -- the default */
    DPI_BAGS_TABLE_MAJOR = 1   /* g = t*B + b: all bags of field 0, then field 1, ... (how jagged feature tensors
                                  usually arrive from a serving stack) */
} dpi_bag_order_t;
typedef enum { DPI_IDX_I32 = 0, DPI_IDX_I64 = 1 } dpi_index_type_t;

/* Tuning knobs for dpi_plan_set_option (all kernel-internal; none changes a result). */
typedef enum {
    DPI_OPT_UNROLL = 0,         /* independent 128-bit row loads in flight per lane: 2, 4, 8 or 16; 0 = auto (a 256-bit load,
                                   DPI_OPT_VEC_BYTES, counts as two) */
    DPI_OPT_BLOCK_THREADS = 1,  /* lookup CTA size: a multiple of 32 up to 256; 0 = auto */
    DPI_OPT_BLOCKS_PER_SM = 2,  /* persistent grid = SMs * this; 0 = auto (occupancy) */
    DPI_OPT_MODE = 3,           /* 0 auto per task, 1 sub-warp per bag, 2 warp per bag (single-buffered),
                                   3 warp per bag (double-buffered batches), 6 short-bag variant (see
                                   DPI_OPT_MAX_BAG_HINT) whatever the hint says */
    DPI_OPT_ROW_L1_NO_ALLOC = 4,/* reserved: accepts -1 / 0 only. Rows always allocate in L1; the L1::no_allocate
                                   variant measured 17-20 % slower on B200 and was removed */
    DPI_OPT_PDL = 5,            /* 1 (default): the lookup (and the fused dpi_forward kernel) is launched with programmatic
                                   dependent launch, so its launch and scheduling overlap the tail of the planner (or of
                                   whatever precedes it on the stream); it executes griddepcontrol.wait before its first
                                   memory read -- table pointers included -- so inputs produced by the preceding kernel are
                                   safe. 0: plain launch */
    DPI_OPT_HOST_CHUNKS = 6,    /* dpi_forward_host only: number of sample chunks pipelined over the copy engines and the
                                   SMs; 0 = auto (~16 MB of PCIe traffic per chunk, <= 8), 1 = no pipelining, up to 64 */
    DPI_OPT_HOST_DIRECT_OUT = 7,/* dpi_forward_host only: 0 = auto, 1 = always stage (lookup -> device block -> D2H copy),
                                   2 = require direct. Direct: when out_host is page-locked, device-mapped memory
                                   (cudaHostAlloc / cudaHostRegister), the lookup kernel stores the pooled vectors
                                   straight into it over PCIe -- the device->host transfer is fused into the kernel's
                                   store, no staging block and no D2H copy. Auto uses it whenever out_host qualifies;
                                   2 returns DPI_ERR_INVALID_ARG if it does not. */
    DPI_OPT_MAX_BAG_HINT = 8,   /* OPTIONAL. 0 = unknown (default): the planner measures the longest bag of every batch (a1's
                                   max_len, meta word 7) and the lookup kernel picks its variant from it on the device --
                                   2 <= max_len <= 8 (or max_len <= 1 and at most 5e5 bags) runs the short-bag body (one lane
                                   group per bag straight from the plan's offsets, no segments), anything else the balanced
                                   segments. L >= 1: the caller's promise that no bag is longer than L (a schema fact in CTR
                                   serving: "at most 3 tags per item"); the same rule is then applied on the host and the
                                   short-bag variant runs as its own, leaner launch. A longer bag is still pooled correctly,
                                   only without load balancing; dpi_check_indices verifies the promise off the hot path. */
    DPI_OPT_FUSED = 9,          /* dpi_forward / dpi_forward_host: 0 = auto (one fused launch when the layout is the dense one,
                                   G <= DPI_OPT_FUSED_MAX_BAGS and the capacity says bags are short on average,
                                   max_indices <= 8*G; not when DPI_OPT_MAX_BAG_HINT = 1 promises one id per bag and G < 4e5:
                                   planner + the short-bag launch measured 11-24 % faster there), 1 = fused whenever the layout
                                   allows, 2 = always plan + lookup */
    DPI_OPT_FUSED_MAX_BAGS = 10,/* ceiling of the auto rule above in bags; 0 = library default (2^20) */
    DPI_OPT_VEC_BYTES = 11,     /* bytes of a row one lane loads at a time in the dense balanced-segment kernel: 0 = auto: 32 (the
                                   sm_100 256-bit load, half the lanes and load instructions per row) for fp32 tables with equal
                                   dims and rows of >= 256 B that are a multiple of 32 B -- the one case where it measured faster
                                    -- and 16 for everything else (16-bit tables, narrower rows, mixed dims);
                                   16 = always 128-bit loads; 32 = require 256-bit for any dtype (DPI_ERR_UNSUPPORTED unless all
                                   dims are equal and the row size is a multiple of 32 B). Whenever 32-byte vectors are in use
                                   (auto on fp32 rows >= 256 B, or forced) every table BASE must be 32-byte aligned -- tighter than
                                   the 16 bytes dpi_lookup otherwise asks for; any cudaMalloc / framework allocation is, a table
                                   sliced at an odd 16-byte offset is not and faults with a misaligned address. The library
                                   cannot check this (the pointers live on the device, and dpi_check_indices does not take
                                   them): set 16 to keep such tables. An output block that is only 16-byte aligned
                                   silently takes the 128-bit kernel. */
    DPI_OPT_COUNT_
} dpi_option_t;

/*
 * dpi_plan_create -- host side. Validates the shape and allocates the plan's device buffers once; the plan
 * is reusable for any batch of the same (T, B, dims, dtype) whose N <= max_indices.
 *   T            number of tables, 1..DPI_MAX_TABLES
 *   table_rows   host int64[T], heights n_t >= 1; copied
 *   dims         host int32[T], embedding dim of each table; every dims[t]*sizeof(dtype) must be a multiple of
 *                16 B and <= 512 B, else DPI_ERR_UNSUPPORTED. The paper has one d; tables of
 *                different widths are an interface variant (R10, §11): table t then occupies columns
 *                [col[t], col[t] + dims[t]) with col[t] = sum of dims[u], u < t ("concatenated")
 *   dtype        storage type of the tables and, by default, of the output
 *   B            samples per batch >= 1;  G = B*T must be < 2^31
 *   max_indices  upper bound on N for any batch built with this plan, 0 <= max_indices < 2^31
 *   plan         receives the handle; destroy with dpi_plan_destroy
 */
dpi_status_t dpi_plan_create(int32_t T, const int64_t* table_rows, const int32_t* dims, dpi_dtype_t dtype,
                             int32_t B, int64_t max_indices, dpi_plan_t** plan);

/* Output element type of dpi_lookup: the table dtype (default) or DPI_F32. bf16 has 8 significand bits, so a
 * correctly rounded bf16 output carries up to 2^-8 = 3.9e-3 relative error by itself; fp32 output keeps the
 * fp32 accumulator (R6). Anything else -> DPI_ERR_UNSUPPORTED. */
dpi_status_t dpi_plan_set_out_dtype(dpi_plan_t* plan, dpi_dtype_t out_dtype);

/*
 * dpi_plan_set_layout -- interface variants of the sparse input (the paper only says multi-hot
 * is supported "by marking offset information", and that ids reach the model as 64-bit integers,
 * PAPER.md:336). Takes effect for the next dpi_plan_build / dpi_lookup*.
 *   order       DPI_BAGS_SAMPLE_MAJOR (default) or DPI_BAGS_TABLE_MAJOR: the position g of bag (b, t) in `lengths`,
 *               `offsets` and the bag-contiguous `indices`. The plan itself (offsets, segments) is a function of the
 *               length sequence only, so its definition does not change; the output stays [B, sum dims] with table
 *               t in its own column block.
 *   index_type  DPI_IDX_I32 (default) or DPI_IDX_I64: element type of `indices` (values must still lie in
 *               [0, table_rows[t]), table_rows[t] < 2^31). The element type of the offsets is a separate setting:
 *               dpi_plan_set_offset_type below (int32 by default, N < 2^31).
 */
dpi_status_t dpi_plan_set_layout(dpi_plan_t* plan, dpi_bag_order_t order, dpi_index_type_t index_type);

/*
 * dpi_plan_set_offset_type -- 64-bit offsets (SURVEY.md 8(f) NEXT-2 "int64 indices/offsets"; ids and their positions reach a
 * serving stack as 64-bit integers). DPI_OFF_I32 (default): offsets, seg_off and N are int32, N < 2^31.
 * DPI_OFF_I64: the same plan definition with int64 offsets[G+1], seg_off[S+1] and N, so one batch may hold N >= 2^31 index
 * entries (G = B*T < 2^31 still; every single bag shorter than 2^31). max_indices: the new capacity (0 = keep), < 2^31 for
 * DPI_OFF_I32, < 2^40 for DPI_OFF_I64. Invalidates the current build. With 64-bit offsets:
 *   - dpi_plan_build runs the 64-bit planner (two stream-ordered launches instead of one);
 *   - dpi_lookup / dpi_lookup_ex / dpi_forward run the general kernel (one launch); a caller-provided offsets_dev must be a
 *     device int64[G+1] passed through the int32 pointer; dpi_plan_device_views returns offsets_dev as such a pointer and
 *     meta words 8 / 9 hold the high halves of N / C[G];
 *   - dpi_plan_export64 replaces dpi_plan_export; dpi_check_indices works unchanged;
 *   - dpi_forward_host, dpi_lookup_input_first and the short-bag / fused single-launch variants are not available
 *     (DPI_ERR_UNSUPPORTED, or silently not chosen).
 */
typedef enum { DPI_OFF_I32 = 0, DPI_OFF_I64 = 1 } dpi_offset_type_t;
dpi_status_t dpi_plan_set_offset_type(dpi_plan_t* plan, dpi_offset_type_t type, int64_t max_indices);
/* dpi_plan_export for a plan with 64-bit offsets: offsets_host int64[G+1], seg_bag_host int32[seg_cap], seg_off_host
 * int64[seg_cap] (S+1 entries each; any may be NULL), S, N. Synchronises `stream`. */
dpi_status_t dpi_plan_export64(const dpi_plan_t* plan, int64_t* offsets_host, int32_t* seg_bag_host, int64_t* seg_off_host,
                               int64_t seg_cap, int64_t* S, int64_t* N, void* stream);

/*
 * dpi_plan_set_columns -- place table t's block at column columns[t] (in elements) of the output row instead of the
 * running prefix of dims. columns: host int64[T], each columns[t]*sizeof(dtype) a multiple of 16 B; blocks must not
 * overlap (not checked); NULL restores the default. The row width becomes max_t(columns[t] + dims[t]). This is what a
 * rank of a table-sharded model uses to write ITS tables into the global [B, sum of all dims] row.
 * Synchronous (one small host->device copy); call it before dpi_lookup*, not between a build and its lookup on
 * another thread.
 */
dpi_status_t dpi_plan_set_columns(dpi_plan_t* plan, const int64_t* columns);

/* Elements per output row = sum of dims (T*D when every table has the same D), or the span set by
 * dpi_plan_set_columns. */
dpi_status_t dpi_plan_out_width(const dpi_plan_t* plan, int64_t* width);

/* Cost quantum K >= 1 of the balanced segments (0 = library default for this row size). Takes effect at the
 * next dpi_plan_build and invalidates the current one (the plan must be built again before dpi_lookup).
 * DPI_ERR_INVALID_ARG if K < 0; on an allocation failure the plan keeps its previous quantum. */
dpi_status_t dpi_plan_set_quantum(dpi_plan_t* plan, int32_t K);

/* Kernel-internal tuning (see dpi_option_t). Unknown option or unsupported value -> DPI_ERR_INVALID_ARG. */
dpi_status_t dpi_plan_set_option(dpi_plan_t* plan, dpi_option_t opt, int32_t value);
dpi_status_t dpi_plan_get_option(const dpi_plan_t* plan, dpi_option_t opt, int32_t* value);

/*
 * dpi_plan_build -- steps a1 + a2 on the device, asynchronous on `stream`, ONE kernel launch for all
 * (sample, table) bags (no per-table launches, no host synchronisation):
 *   lengths_dev  device int32[G], len[g] >= 0, g = b*T + t, 4-byte aligned
 * Writes the plan's offsets[G+1], {seg_bag, seg_off}[S+1] and S (device memory). If the batch has N > max_indices
 * the device sets an overflow flag that dpi_plan_export / dpi_plan_stats report (DPI_ERR_INVALID_ARG);
 * seg_bag writes beyond the capacity are suppressed, never out of bounds.
 */
dpi_status_t dpi_plan_build(dpi_plan_t* plan, const int32_t* lengths_dev, void* stream);

/* north_star spelling: dpi_plan(table_rows[T], dims, lengths, B) = create (max_indices given) + build. */
dpi_status_t dpi_plan(const int64_t* table_rows, int32_t T, const int32_t* dims, dpi_dtype_t dtype,
                      const int32_t* lengths_dev, int32_t B, int64_t max_indices, void* stream,
                      dpi_plan_t** plan);

/* Borrowed device pointers into the plan, valid until the next build/destroy. Any out-pointer may be NULL.
 *   offsets_dev int32[G+1]; seg_dev int32[2*seg_capacity], interleaved pairs {seg_bag[s], seg_off[s]};
 *   meta_dev int32[12] = {S, N (low 32 bits), C[G] (low 32 bits), overflow flag, K, G, min_len, max_len, N (high 32 bits),
 *   C[G] (high 32 bits), -, -} (min / max bag length of the batch: a1's summary of the workload;
 *   min_len == max_len is the uniform-length flag; the high words are zero unless the plan holds 64-bit offsets). */
dpi_status_t dpi_plan_device_views(const dpi_plan_t* plan, const int32_t** offsets_dev,
                                   const int32_t** seg_dev, const int32_t** meta_dev);

/* Static facts about a plan (host only, no synchronisation). Any out-pointer may be NULL. D is the widest table's
 * dim (the common D when all are equal). */
dpi_status_t dpi_plan_info(const dpi_plan_t* plan, int32_t* T, int32_t* B, int32_t* D, int32_t* dtype,
                           int64_t* G, int32_t* K, int64_t* seg_capacity);

/* Parity/debug: synchronises `stream`, copies the plan to caller-owned host arrays.
 *   offsets_host int32[G+1] (may be NULL); seg_bag_host / seg_off_host int32[seg_cap] receive S+1 entries
 *   each (may be NULL); S, N receive the segment count and total index count (may be NULL).
 * DPI_ERR_INVALID_ARG if seg_cap < S+1 or the last build overflowed max_indices. */
dpi_status_t dpi_plan_export(const dpi_plan_t* plan, int32_t* offsets_host, int32_t* seg_bag_host,
                             int32_t* seg_off_host, int64_t seg_cap, int32_t* S, int64_t* N, void* stream);

/* Parity/debug: a1's summary of the last built batch: min_len = shortest, max_len = longest bag;
 * min_len == max_len is the uniform-length flag (1 / 1 is Alg. 1's one-hot workload). Synchronises `stream`. The device
 * reads the same two words (meta_dev[6], meta_dev[7]) to pick the a3 variant. Either out-pointer may be NULL. */
dpi_status_t dpi_plan_stats(const dpi_plan_t* plan, int32_t* min_len, int32_t* max_len, void* stream);

/*
 * dpi_lookup -- step a3, asynchronous on `stream`, ONE kernel launch for all tables and samples.
 *   table_ptrs_dev device array of T device pointers; table t is row-major [table_rows[t], D] of the
 *                  plan's dtype, 16-byte aligned -- 32-byte aligned when 256-bit row loads are in use (DPI_OPT_VEC_BYTES:
 *                  by default fp32 tables with equal dims and rows >= 256 B) ("Embs", per-table local ids
 *                  PAPER.md:162)
 *   indices_dev    device int32[N], per-table local row ids, bag-contiguous in bag order g
 *   offsets_dev    NULL (use the plan's own offsets) or a device int32[G+1] equal to them
 *   plan           a built plan (same stream, or ordered after dpi_plan_build by an event)
 *   pooling        host uint8[T] of dpi_pool_t (NULL = all SUM)
 *   out_dev        device [B, T*D] row-major in the plan's output dtype (dpi_plan_set_out_dtype; default =
 *                  table dtype), 16-byte aligned (32-byte for fp32 output of 16-bit tables); table t at columns
 *                  [t*D, (t+1)*D); every element is written exactly once
 * Out-of-range indices are a precondition violation (the paper is silent, R12): use
 * dpi_check_indices in tests.
 */
dpi_status_t dpi_lookup(const void* const* table_ptrs_dev, const int32_t* indices_dev,
                        const int32_t* offsets_dev, const dpi_plan_t* plan, const uint8_t* pooling,
                        void* out_dev, void* stream);

/*
 * dpi_forward -- the whole path a1 + a2 + a3 on device-resident inputs in one call: dpi_plan_build followed by dpi_lookup,
 * or -- for small / short-bag batches, where the second launch and the plan's trip through global memory are half of the
 * step (the paper's motivation: 4.75 us of work behind 21.92 us of launch overhead; "a single parallel
 * operation") -- ONE fused launch in which the CTA that scans a run of bags pools those bags right away.
 * Either way the plan is left built exactly as dpi_plan_build leaves it (offsets, segments, meta: bit-identical), so
 * dpi_plan_export / dpi_plan_device_views / later dpi_lookup calls on the same batch work unchanged, and the output block
 * is the one dpi_lookup writes. Which way is taken depends on host-known facts only (DPI_OPT_FUSED).
 * Arguments as in dpi_plan_build + dpi_lookup (plan's own offsets; indices int32 / int64 per the plan's index type).
 * Asynchronous on `stream`.
 */
dpi_status_t dpi_forward(dpi_plan_t* plan, const int32_t* lengths_dev, const void* const* table_ptrs_dev,
                         const void* indices_dev, const uint8_t* pooling, void* out_dev, void* stream);

/*
 * dpi_forward_noalloc -- dpi_forward for callers that cannot allocate device memory. It takes no dpi_plan_t (creating one
 * costs nine cudaMalloc calls) and itself calls no cudaMalloc, cudaFree or any other allocating routine: the working memory
 * of the one-launch path (forward_fused.cu: the offsets it scans, its look-back records and counters) is a fixed array of
 * about 2 MB built into the library image. Meant for
 *   - operators inside a serving runtime whose own arena holds all of the GPU's memory (tables + framework pool), where a
 *     cudaMalloc from the operator fails or takes memory somebody else has budgeted;
 *   - request threads with a latency bound, which cannot afford the driver locks and the device-wide synchronisation that
 *     cudaMalloc / cudaFree may bring;
 *   - stateless callbacks that are handed pointers and a stream and have nowhere to keep a plan handle between calls.
 * The price: the array occupies its ~2 MB on EVERY GPU on which this library's code gets loaded, until the process exits; the
 * batch is limited to DPI_NOALLOC_MAX_BAGS bags; and all calls on one GPU share the array, so calls whose kernels may overlap
 * in time (different streams or host threads, same GPU) race on it and give wrong results -- keep them on one stream, or
 * order them with events. Each call first resets the shared words (a one-CTA kernel), so nothing carries over from the call
 * before, whatever its shape was; then runs the fused forward kernel: two launches, asynchronous on `stream`.
 * The FIRST call on each device (with that device current) also looks up the array's device address and the SM count and
 * caches them; make that first call outside any stream capture. Later calls do no set-up.
 *   T, D, dtype     tables, their common embedding dim and storage type; D*sizeof(dtype) a multiple of 16 B, <= 512 B
 *   B               samples; G = B*T must be <= DPI_NOALLOC_MAX_BAGS, else DPI_ERR_INVALID_ARG with a message naming the limit
 *   lengths_dev     device int32[G], g = b*T + t (sample-major), as in dpi_plan_build; N = sum of lengths must be < 2^30
 *                   (precondition; the host never sees N)
 *   table_ptrs_dev, indices_dev (int32[N]), pooling (host uint8[T] or NULL), out_dev ([B, T*D] in the table dtype, 16-byte
 *                   aligned)   as in dpi_lookup
 * Result: the block dpi_forward writes on its fused path, bit for bit (same kernel). Like that path the chunks are not
 * load-balanced across CTAs: right for the short-bag batches of CTR serving, correct but slower for long bags.
 * Equal dims, int32 ids, sample-major bags, dense output in the table dtype only; everything else needs a dpi_plan_t.
 * No plan is left behind for the caller: the array's contents after a call are unspecified.
 */
#define DPI_NOALLOC_MAX_BAGS 524288   /* 2^19 bags: 4 B of scratch per bag + 11 KB fixed */
dpi_status_t dpi_forward_noalloc(int32_t T, int32_t D, dpi_dtype_t dtype, int32_t B, const int32_t* lengths_dev,
                                 const void* const* table_ptrs_dev, const int32_t* indices_dev, const uint8_t* pooling,
                                 void* out_dev, void* stream);

/*
 * dpi_plan_status -- did any build of this plan since the last call exceed its capacity (N > max_indices)? Such a build
 * leaves S = 0 behind (a fitting batch always has S >= 1), and every a3 kernel launched through dpi_lookup / dpi_lookup_ex /
 * the two-launch dpi_forward returns at once on S = 0: nothing is read through the oversized offsets and the output block
 * is left untouched. The ONE exception is dpi_forward's fused single launch: its CTAs pool their chunk before the batch
 * total N exists anywhere, so an over-capacity batch is pooled and stored like any other (it reads indices[0, N), which the
 * caller must own anyway); only the plan it leaves behind is marked S = 0. The planner also bumps a sticky device
 * counter, which this call reads (synchronises `stream`) and clears. DPI_OK and *overflowed_builds = 0 when all builds
 * fitted, DPI_ERR_INVALID_ARG and the count otherwise. overflowed_builds may be NULL. Off the hot path: call it once per
 * served batch group, not per lookup.
 */
dpi_status_t dpi_plan_status(const dpi_plan_t* plan, int32_t* overflowed_builds, void* stream);

/*
 * dpi_lookup_ex -- step a3 with the interface variants: the same fused gather-and-pool,
 * asynchronous on `stream`, ONE launch. Anything the plan's layout says (mixed dims, table-major bags, int64 ids)
 * plus, per call:
 *   weights_dev  NULL, or device fp32[N]: one weight per index entry, acc += w[j] * row (fp32 fused multiply-add;
 *                with every w = 1 the result is bit-identical to the unweighted sum). Sum pooling only: a
 *                mean-pooled table together with weights -> DPI_ERR_UNSUPPORTED.
 *   out_ld       elements between consecutive output rows; 0 = dense (= dpi_plan_out_width). A larger value writes
 *                this call's [B, width] block into a wider row-major matrix (e.g. next to dense features, or as
 *                one rank's column block of a table-sharded model). The pitch in bytes must keep rows 16-byte
 *                aligned (32-byte for fp32 output of 16-bit tables), else DPI_ERR_INVALID_ARG.
 *   indices_dev  int32 or int64 per the plan's index type; the other fields as in dpi_lookup.
 *   out_peers_dev / n_peers / rows_per_peer
 *                fused lookup + all-to-all for table-wise sharding: when out_peers_dev is
 *                not NULL it is a device array of n_peers output base pointers -- peer-mapped memory of the other
 *                GPUs (CUDA IPC / symmetric memory) or plain local buffers -- and sample b is stored to
 *                out_peers_dev[b / rows_per_peer] at row b % rows_per_peer (same pitch and columns), i.e. every
 *                rank writes its tables' column blocks straight into the batch shard of the rank that owns the
 *                sample, over NVLink, from the same kernel that pools them: no send buffer and no separate
 *                collective. out_dev is then ignored. n_peers*rows_per_peer must cover B. The caller orders
 *                consumers after ALL ranks' kernels (e.g. a barrier on the stream).
 *   flags        DPI_LOOKUP_FORCE_GENERAL runs the general kernel even when the call needs none of the variants
 *                (used by the parity tests to compare the two instantiations).
 * Set struct_size = sizeof(dpi_lookup_args_t); a mismatch -> DPI_ERR_INVALID_ARG. Unused fields must be zero.
 */
#define DPI_LOOKUP_FORCE_GENERAL 1u
typedef struct dpi_lookup_args_s {
    uint32_t struct_size;
    uint32_t flags;
    const void* const* table_ptrs_dev;
    const void* indices_dev;
    const int32_t* offsets_dev;
    const float* weights_dev;
    const uint8_t* pooling; /* host[T] or NULL */
    void* out_dev;
    int64_t out_ld;
    const void* const* out_peers_dev; /* NULL, or device array of n_peers output base pointers */
    int32_t n_peers;
    int32_t rows_per_peer;
} dpi_lookup_args_t;
dpi_status_t dpi_lookup_ex(const dpi_lookup_args_t* args, const dpi_plan_t* plan, void* stream);

/*
 * Peer-visible output blocks for the fused lookup + all-to-all above (NEXT-3; one process per GPU). CUDA IPC plumbing only.
 *   dpi_peer_alloc  allocates `bytes` of device memory on the current device as ONE dedicated allocation (an IPC handle
 *                   names a whole allocation) and writes its DPI_PEER_HANDLE_BYTES-byte handle; the caller ships the handle
 *                   to the other ranks over its control plane (e.g. torch.distributed all_gather, any backend).
 *   dpi_peer_open   maps another PROCESS's block into this process (peer access is enabled on demand when the block lives on
 *                   another GPU); the returned pointer goes into out_peers_dev. Opening a handle in the process that created
 *                   it is an error of the CUDA runtime (DPI_ERR_CUDA): a rank uses its own dpi_peer_alloc pointer.
 *   dpi_peer_close  unmaps a pointer returned by dpi_peer_open;  dpi_peer_free releases a dpi_peer_alloc block (after every
 *                   peer has closed it). NULL is a no-op for both.
 * Ordering is the caller's: a rank may read its block only after ALL ranks' lookups have completed (stream synchronise +
 * a barrier of the control plane, or an interprocess event).
 */
#define DPI_PEER_HANDLE_BYTES 64
dpi_status_t dpi_peer_alloc(int64_t bytes, void** dev_ptr, uint8_t* handle);
dpi_status_t dpi_peer_open(const uint8_t* handle, void** dev_ptr);
dpi_status_t dpi_peer_close(void* dev_ptr);
dpi_status_t dpi_peer_free(void* dev_ptr);

/*
 * dpi_lookup_onehot -- Algorithm 1 itself: the one-hot case, where every (sample, table) bag holds
 * exactly one id. The workload is then pure arithmetic, so this call needs NO built plan (the plan object only supplies
 * T, B, the common dim and the dtype): ONE launch copies row ids_dev[b*T + t] of table t to out[b, t*D .. (t+1)*D).
 * Bit-identical to dpi_plan_build on all-ones lengths + dpi_lookup (sum or mean pooling: a bag of length 1 is its row).
 *   ids_dev  device int32[B*T] (int64 when the plan's index type is DPI_IDX_I64), sample-major, per-table local row ids
 *            in [0, table_rows[t]) (precondition, as in dpi_lookup)
 *   out_dev  device [B, T*D] of the TABLE dtype, 16-byte aligned
 * Equal dims, sample-major bags, default columns and table-dtype output only: anything else -> DPI_ERR_UNSUPPORTED
 * (use dpi_lookup_ex). Asynchronous on `stream`.
 */
dpi_status_t dpi_lookup_onehot(const void* const* table_ptrs_dev, const void* ids_dev, const dpi_plan_t* plan,
                               void* out_dev, void* stream);

/*
 * dpi_lookup_input_first -- ABLATION, not the product path: the same lookup with the paper's strawman
 * "input-first" workload allocation (different samples on different threads, so table reads
 * and output writes of a warp are random), kept to measure the paper's Fig. 11 claim (output-first up to 10.3x
 * faster) on B200. Same arguments, results and error behaviour as dpi_lookup; it uses only the
 * plan's offsets (no segments), one thread per sample.
 */
dpi_status_t dpi_lookup_input_first(const void* const* table_ptrs_dev, const int32_t* indices_dev,
                                    const int32_t* offsets_dev, const dpi_plan_t* plan, const uint8_t* pooling,
                                    void* out_dev, void* stream);

/*
 * dpi_forward_host -- the whole path (a1+a2+a3) for callers whose sparse inputs live in HOST memory
 * (the end-to-end number of bench.py): copies lengths and indices host->device into plan-owned staging,
 * builds the plan, runs the lookup and copies the [B, T*D] block back, then synchronises `stream`. A large batch is
 * cut into chunks of whole samples (DPI_OPT_HOST_CHUNKS); chunk c goes H2D -> plan -> lookup -> D2H on one of three
 * internal streams ordered after `stream`, so both PCIe directions and the SMs are busy at once. Each chunk is an
 * independent sub-batch with its own device plan (bags are independent); the host only adds up how many
 * index entries each chunk owns, to size the copies. The result is identical to the unchunked call.
 * Each chunk runs as dpi_forward does: one fused launch when eligible, else planner + lookup.
 * Tables stay resident on the device (they are the model, not a per-batch input).
 *   lengths_host int32[G]; indices_host int32 / int64 [n_indices] per the plan's index type
 *   (n_indices <= max_indices); out_host [B, sum dims].
 *   Pinned (page-locked) host buffers make the copies asynchronous and faster but are not required.
 *   With dpi_plan_set_columns (a row wider than the tables' blocks) the two output paths differ outside the blocks: the direct
 *   path stores pooled vectors only and leaves every other column of out_host untouched; the staged path copies whole rows
 *   of its device block back, so columns that belong to no table are overwritten with unspecified values.
 */
dpi_status_t dpi_forward_host(dpi_plan_t* plan, const void* const* table_ptrs_dev,
                              const int32_t* lengths_host, const void* indices_host, int64_t n_indices,
                              const uint8_t* pooling, void* out_host, void* stream);

/* Off the hot path: checks the preconditions of dpi_lookup on the last built batch; synchronises. Counts indices outside
 * [0, table_rows[t]) -> DPI_ERR_INDEX_RANGE (and *n_bad > 0) if any; and, when DPI_OPT_MAX_BAG_HINT = L > 0 is set, bags longer
 * than the promised L -> DPI_ERR_INVALID_ARG (results would still be correct, only the kernel choice would be wrong). */
dpi_status_t dpi_check_indices(const dpi_plan_t* plan, const void* indices_dev, int64_t* n_bad,
                               void* stream);

dpi_status_t dpi_plan_destroy(dpi_plan_t* plan);

/* Number of kernels this library has launched in this process (for bench.py's gpu_launches claim). */
int64_t dpi_launch_count(void);

int32_t dpi_version(void);
const char* dpi_status_string(dpi_status_t status);
const char* dpi_last_error(void); /* thread-local detail of the last failing call on this thread */

#ifdef __cplusplus
}
#endif
#endif /* DPI_H_ */
