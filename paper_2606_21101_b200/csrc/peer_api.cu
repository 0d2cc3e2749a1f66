// peer_api.cu -- peer-visible output blocks for table-wise sharding (
// the paper names multi-GPU embedding only as related work). One process per GPU: every rank allocates
// its [B / n, sum dims] batch shard with dpi_peer_alloc, the 64-byte handles travel over the job's control plane
// (torch.distributed, any backend), every rank maps the others' shards with dpi_peer_open, and dpi_lookup_ex(out_peers_dev)
// stores into them -- over NVLink when the ranks sit on different GPUs, through the same device's memory when they share one.
// Host code only: CUDA IPC plumbing, no arithmetic of the method.
#include <cstring>

#include "dpi_internal.cuh"

using namespace dpi;

namespace {
dpi_status_t cuda_status(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return DPI_OK;
    (void)cudaGetLastError();
    return report_error(e == cudaErrorMemoryAllocation ? DPI_ERR_ALLOC : DPI_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
static_assert(sizeof(cudaIpcMemHandle_t) == DPI_PEER_HANDLE_BYTES, "handle size is part of the ABI");
}  // namespace

extern "C" {

dpi_status_t dpi_peer_alloc(int64_t bytes, void** dev_ptr, uint8_t* handle) {
    if (!dev_ptr || !handle || bytes < 1) return report_error(DPI_ERR_INVALID_ARG, "dpi_peer_alloc: NULL argument or bytes < 1");
    *dev_ptr = nullptr;
    void* p = nullptr;
    // a dedicated cudaMalloc: an IPC handle names a whole allocation, so the block must not be carved out of a pool
    dpi_status_t st = cuda_status(cudaMalloc(&p, static_cast<size_t>(bytes)), "cudaMalloc");
    if (st != DPI_OK) return st;
    cudaIpcMemHandle_t h;
    st = cuda_status(cudaIpcGetMemHandle(&h, p), "cudaIpcGetMemHandle");
    if (st != DPI_OK) {
        (void)cudaFree(p);
        return st;
    }
    std::memcpy(handle, &h, sizeof h);
    *dev_ptr = p;
    return DPI_OK;
}

dpi_status_t dpi_peer_open(const uint8_t* handle, void** dev_ptr) {
    if (!dev_ptr || !handle) return report_error(DPI_ERR_INVALID_ARG, "dpi_peer_open: NULL argument");
    *dev_ptr = nullptr;
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle, sizeof h);
    void* p = nullptr;
    dpi_status_t st = cuda_status(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess), "cudaIpcOpenMemHandle");
    if (st != DPI_OK) return st;
    *dev_ptr = p;
    return DPI_OK;
}

dpi_status_t dpi_peer_close(void* dev_ptr) {
    if (!dev_ptr) return DPI_OK;
    return cuda_status(cudaIpcCloseMemHandle(dev_ptr), "cudaIpcCloseMemHandle");
}

dpi_status_t dpi_peer_free(void* dev_ptr) {
    if (!dev_ptr) return DPI_OK;
    return cuda_status(cudaFree(dev_ptr), "cudaFree");
}

}  // extern "C"
