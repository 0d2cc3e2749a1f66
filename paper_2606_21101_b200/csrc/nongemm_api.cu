// nongemm_api.cu -- C ABI of include/dpi_nongemm.h: argument validation and launches of the
// fused non-GEMM operators, and Algorithm 2: the breadth-first launch queue and the two-stream
// launcher. Host code only; every number is produced by nongemm_kernels.cu. No CPU fallback.
#include <new>
#include <vector>

#include "dpi_internal.cuh"
#include "../../include/dpi_nongemm.h"

using namespace dpi;

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
bool dtype_ok(int d) { return d == DPI_F32 || d == DPI_F16 || d == DPI_BF16; }
uint32_t elt_bytes(int d) { return d == DPI_F32 ? 4u : 2u; }

dpi_status_t cuda_status(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return DPI_OK;
    (void)cudaGetLastError();
    return report_error(DPI_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

}  // namespace

extern "C" {

dpi_status_t dpi_fm_interaction(const void* x_dev, dpi_dtype_t dtype, int32_t B, int32_t T, int32_t D, int64_t x_ld,
                                float* y_dev, float* v_dev, void* stream) {
    if (!x_dev || (!y_dev && !v_dev)) return report_error(DPI_ERR_INVALID_ARG, "dpi_fm_interaction: NULL x, or neither y nor v given");
    if (!dtype_ok(dtype)) return report_error(DPI_ERR_INVALID_ARG, "dpi_fm_interaction: bad dtype %d", static_cast<int>(dtype));
    if (B < 0 || T <= 0 || D <= 0) return report_error(DPI_ERR_INVALID_ARG, "dpi_fm_interaction: B=%d T=%d D=%d", B, T, D);
    const uint32_t eb = elt_bytes(dtype);
    const uint64_t field_bytes = static_cast<uint64_t>(D) * eb;
    if (field_bytes % 16 != 0 || field_bytes > 512)
        return report_error(DPI_ERR_UNSUPPORTED, "dpi_fm_interaction: D*sizeof(elt) = %llu must be a multiple of 16 and <= 512",
                            static_cast<unsigned long long>(field_bytes));
    const int64_t width = static_cast<int64_t>(T) * D;
    if (x_ld == 0) x_ld = width;
    if (x_ld < width || (static_cast<uint64_t>(x_ld) * eb) % 16 != 0)
        return report_error(DPI_ERR_INVALID_ARG, "dpi_fm_interaction: x_ld = %lld (needs >= T*D and a 16-byte multiple in bytes)",
                            static_cast<long long>(x_ld));
    if (!aligned16(x_dev) || (v_dev && !aligned16(v_dev)) || (y_dev && (reinterpret_cast<uintptr_t>(y_dev) & 3u)))
        return report_error(DPI_ERR_INVALID_ARG, "dpi_fm_interaction: misaligned pointer");
    if (B == 0) return DPI_OK;
    return cuda_status(launch_fm(x_dev, dtype, static_cast<uint32_t>(B), static_cast<uint32_t>(T), static_cast<uint32_t>(D),
                                 static_cast<uint64_t>(x_ld) * eb, y_dev, v_dev, static_cast<cudaStream_t>(stream)),
                       "fm_kernel launch");
}

dpi_status_t dpi_lr_first_order(const void* const* w_ptrs_dev, const int32_t* indices_dev, const int32_t* offsets_dev,
                                int32_t B, int32_t T, float bias, float* y_dev, int32_t accumulate, void* stream) {
    if (!w_ptrs_dev || !indices_dev || !y_dev) return report_error(DPI_ERR_INVALID_ARG, "dpi_lr_first_order: NULL pointer");
    if (B < 0 || T <= 0) return report_error(DPI_ERR_INVALID_ARG, "dpi_lr_first_order: B=%d T=%d", B, T);
    if ((reinterpret_cast<uintptr_t>(w_ptrs_dev) & 7u) || (reinterpret_cast<uintptr_t>(indices_dev) & 3u) ||
        (reinterpret_cast<uintptr_t>(offsets_dev) & 3u) || (reinterpret_cast<uintptr_t>(y_dev) & 3u))
        return report_error(DPI_ERR_INVALID_ARG, "dpi_lr_first_order: misaligned pointer");
    if (static_cast<int64_t>(B) * T > 0x7fffffffll) return report_error(DPI_ERR_UNSUPPORTED, "dpi_lr_first_order: B*T exceeds 2^31 - 1");
    if (B == 0) return DPI_OK;
    return cuda_status(launch_lr(w_ptrs_dev, indices_dev, offsets_dev, static_cast<uint32_t>(B), static_cast<uint32_t>(T), bias, y_dev,
                                 accumulate != 0, static_cast<cudaStream_t>(stream)),
                       "lr_kernel launch");
}

static dpi_status_t check_ew(const char* who, int dtype, int32_t B, int32_t F) {
    if (!dtype_ok(dtype)) return report_error(DPI_ERR_INVALID_ARG, "%s: bad dtype %d", who, dtype);
    if (B < 0 || F <= 0) return report_error(DPI_ERR_INVALID_ARG, "%s: B=%d F=%d", who, B, F);
    if ((static_cast<uint64_t>(F) * elt_bytes(dtype)) % 16 != 0)
        return report_error(DPI_ERR_UNSUPPORTED, "%s: F*sizeof(elt) must be a multiple of 16 (F=%d)", who, F);
    return DPI_OK;
}

dpi_status_t dpi_cross_combine(const void* x0_dev, const void* xl_dev, const void* u_dev, const float* bias_dev,
                               void* out_dev, dpi_dtype_t dtype, int32_t B, int32_t F, void* stream) {
    if (!x0_dev || !xl_dev || !u_dev || !out_dev) return report_error(DPI_ERR_INVALID_ARG, "dpi_cross_combine: NULL pointer");
    const dpi_status_t st = check_ew("dpi_cross_combine", dtype, B, F);
    if (st != DPI_OK) return st;
    if (!aligned16(x0_dev) || !aligned16(xl_dev) || !aligned16(u_dev) || !aligned16(out_dev) || (bias_dev && !aligned16(bias_dev)))
        return report_error(DPI_ERR_INVALID_ARG, "dpi_cross_combine: pointers must be 16-byte aligned");
    if (B == 0) return DPI_OK;
    return cuda_status(launch_cross_combine(x0_dev, xl_dev, u_dev, bias_dev, out_dev, dtype, static_cast<uint32_t>(B),
                                            static_cast<uint32_t>(F), static_cast<cudaStream_t>(stream)),
                       "cross_combine_kernel launch");
}

dpi_status_t dpi_bias_act(const void* u_dev, const float* bias_dev, void* out_dev, dpi_dtype_t dtype, int32_t B,
                          int32_t F, dpi_act_t act, void* stream) {
    if (!u_dev || !out_dev) return report_error(DPI_ERR_INVALID_ARG, "dpi_bias_act: NULL pointer");
    if (act != DPI_ACT_IDENTITY && act != DPI_ACT_RELU && act != DPI_ACT_SIGMOID)
        return report_error(DPI_ERR_INVALID_ARG, "dpi_bias_act: bad activation %d", static_cast<int>(act));
    const dpi_status_t st = check_ew("dpi_bias_act", dtype, B, F);
    if (st != DPI_OK) return st;
    if (!aligned16(u_dev) || !aligned16(out_dev) || (bias_dev && !aligned16(bias_dev)))
        return report_error(DPI_ERR_INVALID_ARG, "dpi_bias_act: pointers must be 16-byte aligned");
    if (B == 0) return DPI_OK;
    return cuda_status(launch_bias_act(u_dev, bias_dev, out_dev, dtype, static_cast<uint32_t>(B), static_cast<uint32_t>(F),
                                       static_cast<int>(act), static_cast<cudaStream_t>(stream)),
                       "bias_act_kernel launch");
}

// ---- Algorithm 2 -----------------------------------------------------------------------------------------------
// The module with more operators goes first and the two alternate while both have operators left; the rest of the
// longer module follows ("The module that has more operators launches first").
dpi_status_t dpi_bfs_schedule(int32_t n_explicit, int32_t n_implicit, int32_t* q_module, int32_t* q_op) {
    if (n_explicit < 0 || n_implicit < 0) return report_error(DPI_ERR_INVALID_ARG, "dpi_bfs_schedule: negative count");
    if ((n_explicit + n_implicit) > 0 && (!q_module || !q_op)) return report_error(DPI_ERR_INVALID_ARG, "dpi_bfs_schedule: NULL queue");
    const int32_t lead = n_implicit > n_explicit ? DPI_MODULE_IMPLICIT : DPI_MODULE_EXPLICIT;
    const int32_t n_lead = lead == DPI_MODULE_IMPLICIT ? n_implicit : n_explicit;
    const int32_t n_other = lead == DPI_MODULE_IMPLICIT ? n_explicit : n_implicit;
    int64_t n = 0;
    for (int32_t i = 0; i < n_lead; ++i) {
        q_module[n] = lead; q_op[n] = i; ++n;
        if (i < n_other) { q_module[n] = 1 - lead; q_op[n] = i; ++n; }
    }
    return DPI_OK;
}

}  // extern "C"

struct dpi_launcher_s {
    cudaStream_t st[2] = {nullptr, nullptr};      // [DPI_MODULE_EXPLICIT], [DPI_MODULE_IMPLICIT]
    cudaEvent_t fork = nullptr, join[2] = {nullptr, nullptr};
};

extern "C" {

dpi_status_t dpi_launcher_create(dpi_launcher_t** launcher) {
    if (!launcher) return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_create: NULL");
    dpi_launcher_t* l = new (std::nothrow) dpi_launcher_t();
    if (!l) return report_error(DPI_ERR_ALLOC, "dpi_launcher_create: out of host memory");
    cudaError_t e = cudaSuccess;
    for (int m = 0; m < 2 && e == cudaSuccess; ++m) {
        e = cudaStreamCreateWithFlags(&l->st[m], cudaStreamNonBlocking);                       // Alg. 2 lines 5-6
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&l->join[m], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&l->fork, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        dpi_launcher_destroy(l);
        return cuda_status(e, "dpi_launcher_create");
    }
    *launcher = l;
    return DPI_OK;
}

dpi_status_t dpi_launcher_destroy(dpi_launcher_t* l) {
    if (!l) return DPI_OK;
    for (int m = 0; m < 2; ++m) {
        if (l->join[m]) (void)cudaEventDestroy(l->join[m]);
        if (l->st[m]) (void)cudaStreamDestroy(l->st[m]);
    }
    if (l->fork) (void)cudaEventDestroy(l->fork);
    delete l;
    return DPI_OK;
}

dpi_status_t dpi_launcher_run(dpi_launcher_t* l, const dpi_op_t* explicit_ops, int32_t n_explicit,
                              const dpi_op_t* implicit_ops, int32_t n_implicit, int32_t n_streams, void* stream) {
    if (!l) return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_run: NULL launcher");
    if (n_explicit < 0 || n_implicit < 0 || (n_explicit > 0 && !explicit_ops) || (n_implicit > 0 && !implicit_ops))
        return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_run: bad operator lists");
    if (n_streams != 1 && n_streams != 2) return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_run: n_streams must be 1 or 2");
    for (int32_t i = 0; i < n_explicit; ++i)
        if (!explicit_ops[i].launch) return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_run: explicit op %d has no launch function", i);
    for (int32_t i = 0; i < n_implicit; ++i)
        if (!implicit_ops[i].launch) return report_error(DPI_ERR_INVALID_ARG, "dpi_launcher_run: implicit op %d has no launch function", i);
    const int32_t n = n_explicit + n_implicit;
    if (n == 0) return DPI_OK;
    std::vector<int32_t> qm(n), qo(n);
    const dpi_status_t st = dpi_bfs_schedule(n_explicit, n_implicit, qm.data(), qo.data());
    if (st != DPI_OK) return st;
    cudaStream_t main = static_cast<cudaStream_t>(stream);
    const bool two = n_streams == 2;
    if (two) {  // both module streams start after everything already enqueued on the caller's stream
        cudaError_t e = cudaEventRecord(l->fork, main);
        for (int m = 0; m < 2 && e == cudaSuccess; ++m) e = cudaStreamWaitEvent(l->st[m], l->fork, 0);
        if (e != cudaSuccess) return cuda_status(e, "dpi_launcher_run: fork");
    }
    for (int32_t i = 0; i < n; ++i) {  // the launch queue Q, in order (Alg. 2 lines 9-26)
        const dpi_op_t& op = qm[i] == DPI_MODULE_EXPLICIT ? explicit_ops[qo[i]] : implicit_ops[qo[i]];
        op.launch(op.user, two ? static_cast<void*>(l->st[qm[i]]) : stream);
    }
    if (two) {
        for (int m = 0; m < 2; ++m) {
            cudaError_t e = cudaEventRecord(l->join[m], l->st[m]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(main, l->join[m], 0);
            if (e != cudaSuccess) return cuda_status(e, "dpi_launcher_run: join");
        }
    }
    return DPI_OK;
}

}  // extern "C"
