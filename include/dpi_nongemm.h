/*
 * dpi_nongemm.h -- C ABI of the step AFTER the fused embedding lookup: the fused non-GEMM
 * operators that consume X_embed and the breadth-first two-stream launcher. Same library (libdpi.so), same rules as
 * dpi.h: extern "C", plain pointers and sizes, every call returns dpi_status_t, nothing throws, device work is
 * asynchronous on the `stream` argument (a cudaStream_t passed as void*), no CPU fallback.
 *
 * Source passages:
 *   IV-D "Fusion Mechanism for non-GEMM Operators": "we combine all neighbouring non-GEMM
 *   operators into a single operator ... We traverse the output matrix element by element, assigning the filling tasks
 *   for each matrix element to individual threads, ensuring that data reads and writes are contiguous in memory."
 *   The operators it names: DeepFM's factorization machine ("element-wise square and reduce-sum"),
 *   DCNv2's cross network ("element-wise addition and element-wise multiplication ... besides GEMM"), the MLP's
 *   activation. The paper prints no formulas; DESIGN.md 11.4 (readings N1-N3) fixes them.
 *   IV-E "Stream Scheduling Strategy" + Algorithm 2: operators of the explicit and the implicit
 *   interaction module go to two CUDA streams and are launched in an alternating, breadth-first order, the module
 *   with more operators first.
 * GEMMs are NOT here: they are plain library calls (cuBLAS) made by the caller between these operators.
 *
 * Data layout: all matrices row-major, element type `dtype` (DPI_F32 / DPI_F16 / DPI_BF16 as in dpi.h) unless stated;
 * arithmetic in fp32, one round-to-nearest-even cast at the store. Pointers are DEVICE pointers owned by the caller,
 * 16-byte aligned, rows 16-byte aligned (row pitches are in ELEMENTS and pitch*sizeof(elt) must be a multiple of 16).
 * Errors: NULL / non-positive sizes / misalignment -> DPI_ERR_INVALID_ARG, shapes the kernels do not cover ->
 * DPI_ERR_UNSUPPORTED, both before any launch; launch failures -> DPI_ERR_CUDA with dpi_last_error() text.
 */
#ifndef DPI_NONGEMM_H
#define DPI_NONGEMM_H

#include "dpi.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * dpi_fm_interaction -- DeepFM's FM second-order term, all of its non-GEMM operators (square, reduce-sum over fields,
 * subtract, scale, reduce-sum over the embedding dimension) in ONE launch that reads X_embed once.
 *   x_dev   [B, x_ld] of `dtype`: the lookup's output block, field t at columns [t*D, (t+1)*D)
 *   T, D    number of fields and the common embedding dim; D*sizeof(elt) a multiple of 16 and <= 512 bytes
 *   x_ld    elements between rows; 0 = T*D
 *   y_dev   NULL or fp32[B]:    y[b]   = sum_{t<u} <x[b,t,:], x[b,u,:]> = 1/2 sum_c ((sum_t x_tc)^2 - sum_t x_tc^2)
 *   v_dev   NULL or fp32[B, D]: v[b,c] = 1/2 ((sum_t x_tc)^2 - sum_t x_tc^2)     (the term before the last reduce-sum)
 *           at least one of y_dev / v_dev must be given.
 * One warp (or sub-warp group) per sample, output-first: the lanes of a warp read consecutive 16-byte vectors of one
 * sample's row. fp32 accumulation.
 */
dpi_status_t dpi_fm_interaction(const void* x_dev, dpi_dtype_t dtype, int32_t B, int32_t T, int32_t D, int64_t x_ld,
                                float* y_dev, float* v_dev, void* stream);

/*
 * dpi_forward_fm -- the lookup and its first non-GEMM consumer as one operator ("we combine all neighbouring
 * non-GEMM operators into a single operator"; the embedding lookup is itself non-GEMM and DeepFM's FM reads what it writes,
 * PAPER.md:186): a1 + a2 + a3 exactly as dpi_forward (out_dev receives the [B, T*D] block, the plan is left built) PLUS the
 * FM second-order term of every sample, y_dev fp32[B] and / or v_dev fp32[B, D] as in dpi_fm_interaction.
 * For small / short-bag batches (the dpi_forward rule, DPI_OPT_FUSED) with table-dtype output this is ONE launch: chunks of
 * the fused forward kernel are whole samples, and the CTA that pooled a sample's T bags forms its FM term from the vectors
 * it has just stored (read back through L2 after a CTA barrier) -- no second launch, no second pass over X_embed in HBM.
 * Otherwise it is dpi_forward followed by the FM kernel on the same stream. Either way y / v are bit-identical to
 * dpi_fm_interaction applied to the block this call wrote (the same per-sample code runs in both). One common dim, default columns and
 * sample-major bags only (DPI_ERR_UNSUPPORTED otherwise); y_dev 4-byte, v_dev 16-byte aligned. Asynchronous on `stream`.
 */
dpi_status_t dpi_forward_fm(dpi_plan_t* plan, const int32_t* lengths_dev, const void* const* table_ptrs_dev,
                            const void* indices_dev, const uint8_t* pooling, void* out_dev, float* y_dev, float* v_dev,
                            void* stream);

/*
 * dpi_cross_combine -- the non-GEMM part of one DCNv2 cross layer, x_{l+1} = x_0 * (W x_l + b) + x_l, given
 * u = W x_l from the caller's GEMM: out[b,f] = x0[b,f] * (u[b,f] + bias[f]) + xl[b,f]  (element-wise add, multiply,
 * add fused into one pass).
 *   x0_dev, xl_dev, u_dev, out_dev  [B, F] dense of `dtype` (out_dev may alias xl_dev or u_dev); bias_dev NULL or
 *   fp32[F]; F*sizeof(elt) a multiple of 16.
 */
dpi_status_t dpi_cross_combine(const void* x0_dev, const void* xl_dev, const void* u_dev, const float* bias_dev,
                               void* out_dev, dpi_dtype_t dtype, int32_t B, int32_t F, void* stream);

/*
 * dpi_lr_first_order -- DeepFM's logistic-regression (first-order) term, "table lookup ... and reduce-sum"
 * (DESIGN.md 11.4 N7): one scalar weight per feature,
 *     y[b] = bias + sum_t sum_{j in bag(b,t)} w_t[indices[j]]          (or y[b] += ... when accumulate != 0)
 * fused into ONE launch (T lookups + T-way reduce-sum + bias): one warp per sample, lanes over its T bags.
 *   w_ptrs_dev   device array of T device pointers, w_ptrs_dev[t] = fp32[table_rows[t]]
 *   indices_dev  device int32, sample-major CSR bags exactly as dpi_lookup reads them (per-table local ids, range is a
 *                precondition); offsets_dev device int32[B*T+1] (e.g. the plan's, dpi_plan_device_views), or NULL for
 *                one-hot input (bag g is entry g: indices_dev = IDs[B*T])
 *   y_dev        device fp32[B]; accumulate != 0 adds to what is there (e.g. the FM term), bias included once
 * fp32 accumulation; an empty sample gives bias.
 */
dpi_status_t dpi_lr_first_order(const void* const* w_ptrs_dev, const int32_t* indices_dev, const int32_t* offsets_dev,
                                int32_t B, int32_t T, float bias, float* y_dev, int32_t accumulate, void* stream);

typedef enum { DPI_ACT_IDENTITY = 0, DPI_ACT_RELU = 1, DPI_ACT_SIGMOID = 2 } dpi_act_t;

/*
 * dpi_bias_act -- the non-GEMM part of one MLP layer: out[b,f] = act(u[b,f] + bias[f]) ("GEMM and
 * activation operators"). u_dev, out_dev [B, F] dense of `dtype` (may alias); bias_dev NULL or fp32[F];
 * F*sizeof(elt) a multiple of 16. Sigmoid is 1 / (1 + exp(-s)) in fp32 with the hardware ex2 / rcp approximations
 * (absolute error <= 2^-21 before the output cast; the precise expf + IEEE division made the operator ALU-bound).
 */
dpi_status_t dpi_bias_act(const void* u_dev, const float* bias_dev, void* out_dev, dpi_dtype_t dtype, int32_t B,
                          int32_t F, dpi_act_t act, void* stream);

/* ---- Algorithm 2: breadth-first stream scheduling ------------------------------------------- */

typedef enum { DPI_MODULE_EXPLICIT = 0, DPI_MODULE_IMPLICIT = 1 } dpi_module_t;

/*
 * dpi_bfs_schedule -- the launch queue Q of Algorithm 2 (host, integers only). Writes n_explicit + n_implicit entries:
 * q_module[i] in {DPI_MODULE_EXPLICIT, DPI_MODULE_IMPLICIT}, q_op[i] = index of the operator inside its module.
 * Alternates the two modules starting with the one that has MORE operators (ties: explicit), then appends the rest
 * of the longer one. Host arrays owned by the caller.
 */
dpi_status_t dpi_bfs_schedule(int32_t n_explicit, int32_t n_implicit, int32_t* q_module, int32_t* q_op);

/* One operator of a module: `launch(user, stream)` must enqueue its work on `stream` (a cudaStream_t) and return. */
typedef void (*dpi_op_fn)(void* user, void* stream);
typedef struct dpi_op_s {
    dpi_op_fn launch;
    void* user;
} dpi_op_t;

typedef struct dpi_launcher_s dpi_launcher_t; /* opaque: two non-blocking streams + fork/join events */

dpi_status_t dpi_launcher_create(dpi_launcher_t** launcher);
dpi_status_t dpi_launcher_destroy(dpi_launcher_t* launcher);

/*
 * dpi_launcher_run -- Algorithm 2 end to end: both module streams are ordered after everything already enqueued on
 * `stream` (fork event), the operators are launched in the order of dpi_bfs_schedule, each into its module's stream
 * (lines 5-8), and `stream` is ordered after both modules (join events). Asynchronous; safe inside CUDA stream
 * capture (the fork/join become graph dependencies). n_streams = 1 launches the same queue into `stream` itself
 * (the single-default-stream baseline of PAPER.md:192), n_streams = 2 is the paper's strategy.
 * The callbacks run on the calling thread, in queue order, before the call returns.
 */
dpi_status_t dpi_launcher_run(dpi_launcher_t* launcher, const dpi_op_t* explicit_ops, int32_t n_explicit,
                              const dpi_op_t* implicit_ops, int32_t n_implicit, int32_t n_streams, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DPI_NONGEMM_H */
