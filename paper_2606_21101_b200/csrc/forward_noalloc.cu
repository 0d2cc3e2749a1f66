// forward_noalloc.cu -- dpi_forward_noalloc: the one-launch path a1 + a2 + a3 (forward_fused.cu) for callers that must not
// allocate device memory (include/dpi.h has the contract; README "No-allocation entry point").
//
// Every other way into the lookup goes through a dpi_plan_t, and dpi_plan_create calls cudaMalloc nine times. Some callers
// of an embedding lookup cannot do that:
//   * an operator plugged into a serving runtime whose arena already owns all of the GPU's memory -- with 180 GB of HBM
//     handed to the embedding tables and the framework's pool, a cudaMalloc from inside the operator fails or eats into a
//     budget somebody else has planned;
//   * a request thread under a latency bound: cudaMalloc / cudaFree take driver-wide locks and may synchronise the whole
//     device, which stalls every other stream of the process for the duration;
//   * a stateless callback (a custom-op hook that gets pointers and a stream and nothing else): it has no place to keep a
//     plan handle between calls and no create / destroy moment to allocate and free one.
// For them the fused forward kernel's working memory -- the plan it leaves behind (offsets, a stub of segment records, meta)
// and its look-back records and counters -- lives in ONE fixed array inside the library image, g_scratch below. The caller
// passes inputs and the output block, nothing else.
//
// What that costs: kScratchBytes (about 2 MB) of device memory on every GPU on which this library's module gets loaded, held
// until the process exits; a hard ceiling on the batch (DPI_NOALLOC_MAX_BAGS bags); and no concurrency -- all calls on one GPU
// share the array, so two calls whose kernels overlap in time (different streams, different host threads) race on it.
// Calls on ONE stream are ordered and safe.
#include <algorithm>
#include <mutex>

#include "dpi_internal.cuh"

namespace dpi {
namespace {

// ---- layout of the scratch array (byte offsets; every block 256-byte aligned) ----
constexpr size_t kOffState = 0;                                               // unsigned int[kStateWords]   planner counters
constexpr size_t kOffMeta = 256;                                              // int32[kMetaWords]           plan summary
constexpr size_t kOffSeg = 512;                                               // int2[kSegCap]               segment stub
constexpr size_t kOffStatus = 768;                                            // ulonglong2[kStatusRecords]  look-back records
constexpr size_t kOffOffsets = kOffStatus + sizeof(ulonglong2) * kStatusRecords;   // int32[MAX_BAGS + 1]    a1's offsets
constexpr size_t kScratchBytes = (kOffOffsets + sizeof(int32_t) * (static_cast<size_t>(DPI_NOALLOC_MAX_BAGS) + 1) + 255) / 256 * 256;
static_assert(kOffOffsets % 256 == 0, "offsets block must stay 256-byte aligned");
static_assert(sizeof(unsigned int) * kStateWords <= 256 && sizeof(int32_t) * kMetaWords <= 256, "state / meta outgrew their slots");

// The balanced segments are of no use to this entry point (the fused kernel pools chunk by chunk and nobody can ask for the
// plan afterwards), so the quantum is set beyond any reachable cost C[G] <= N + G < 2^30: the kernel then writes exactly
// seg[0] and seg[1] and the stub below is all the segment memory it needs.
constexpr uint32_t kSegCap = 4;
constexpr uint32_t kQuantumShift = 30;
static_assert(sizeof(int2) * kSegCap <= 256, "segment stub outgrew its slot");

// The scratch itself. In HOST code the name g_scratch is only a handle for the runtime's symbol table, not an address a
// kernel could use: device_setup() below asks the runtime for the real device address, once per GPU.
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

// Puts the shared words back to what a fresh plan holds (dpi_plan_create's initial values), whatever the previous call --
// possibly one with a different grid, or one that died half-way -- left in them: ticket / done counters 0, epoch 1, running
// min / max re-armed, every look-back record "not ready", meta zero. Device code may name the array directly.
__global__ void __launch_bounds__(256) noalloc_reset_kernel() {
    unsigned int* state = reinterpret_cast<unsigned int*>(g_scratch + kOffState);
    int32_t* meta = reinterpret_cast<int32_t*>(g_scratch + kOffMeta);
    ulonglong2* status = reinterpret_cast<ulonglong2*>(g_scratch + kOffStatus);
    const unsigned int tid = threadIdx.x;
    if (tid < kStateWords) state[tid] = tid == kStateEpoch ? 1u : (tid == kStateMinLen ? 0xffffffffu : 0u);
    if (tid < kMetaWords) meta[tid] = 0;
    for (unsigned int i = tid; i < static_cast<unsigned int>(kStatusRecords); i += blockDim.x) status[i] = make_ulonglong2(0ull, 0ull);
}

struct DeviceSetup {
    bool ready = false;
    unsigned char* scratch = nullptr;   // device address of g_scratch on this GPU
    int num_sms = 0;
};
constexpr int kMaxDevices = 64;
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

// One-time set-up for the current device: resolve the array's device address and read the SM count. No allocation.
dpi_status_t device_setup(const DeviceSetup** out) {
    int dev = -1, n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev == 0) {
        (void)cudaGetLastError();
        return report_error(DPI_ERR_CUDA, "no CUDA device (%s); libdpi has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return report_error(DPI_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= kMaxDevices) return report_error(DPI_ERR_UNSUPPORTED, "device ordinal %d is outside [0, %d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& s = g_setup[dev];
    if (!s.ready) {
        int major = 0, sms = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return report_error(DPI_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e)); }
        if (major < 10) return report_error(DPI_ERR_UNSUPPORTED, "device compute capability %d.x: libdpi is built for sm_100a only", major);
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);   // the address of g_scratch ON THE CURRENT DEVICE
        if (e != cudaSuccess || p == nullptr) {
            (void)cudaGetLastError();
            return report_error(DPI_ERR_CUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", dev, e != cudaSuccess ? cudaGetErrorString(e) : "null address");
        }
        s.scratch = static_cast<unsigned char*>(p);
        s.num_sms = sms;
        s.ready = true;
    }
    *out = &s;
    return DPI_OK;
}

}  // namespace
}  // namespace dpi

using namespace dpi;

extern "C" dpi_status_t dpi_forward_noalloc(int32_t T, int32_t D, dpi_dtype_t dtype, int32_t B, const int32_t* lengths_dev,
                                            const void* const* table_ptrs_dev, const int32_t* indices_dev, const uint8_t* pooling,
                                            void* out_dev, void* stream) {
    if (T < 1 || B < 1 || D < 1) return report_error(DPI_ERR_INVALID_ARG, "T=%d, B=%d and D=%d must be >= 1", T, B, D);
    if (T > DPI_MAX_TABLES) return report_error(DPI_ERR_UNSUPPORTED, "T=%d exceeds DPI_MAX_TABLES=%d", T, DPI_MAX_TABLES);
    if (dtype != DPI_F32 && dtype != DPI_F16 && dtype != DPI_BF16) return report_error(DPI_ERR_INVALID_ARG, "unknown dtype %d", (int)dtype);
    const int64_t G64 = static_cast<int64_t>(B) * T;
    if (G64 > DPI_NOALLOC_MAX_BAGS)
        return report_error(DPI_ERR_INVALID_ARG, "B*T = %lld bags exceeds DPI_NOALLOC_MAX_BAGS = %d, the size of the library's built-in scratch array; "
                            "split the batch into runs of whole samples or use a dpi_plan_t (dpi_plan_create + dpi_forward)",
                            (long long)G64, (int)DPI_NOALLOC_MAX_BAGS);
    const int64_t row_bytes = static_cast<int64_t>(D) * (dtype == DPI_F32 ? 4 : 2);
    if (row_bytes % 16 != 0) return report_error(DPI_ERR_UNSUPPORTED, "row size %lld B is not a multiple of 16 B", (long long)row_bytes);
    if (row_bytes > 512) return report_error(DPI_ERR_UNSUPPORTED, "row size %lld B exceeds 512 B (one warp-wide 128-bit load)", (long long)row_bytes);
    if (!lengths_dev || !table_ptrs_dev || !indices_dev || !out_dev) return report_error(DPI_ERR_INVALID_ARG, "lengths_dev / table_ptrs_dev / indices_dev / out_dev is NULL");
    if (reinterpret_cast<uintptr_t>(lengths_dev) & 3u) return report_error(DPI_ERR_INVALID_ARG, "lengths_dev is not 4-byte aligned");
    if (reinterpret_cast<uintptr_t>(indices_dev) & 3u) return report_error(DPI_ERR_INVALID_ARG, "indices_dev is not 4-byte aligned");
    if (reinterpret_cast<uintptr_t>(out_dev) & 15u) return report_error(DPI_ERR_INVALID_ARG, "out_dev is not 16-byte aligned");

    const DeviceSetup* dev = nullptr;
    dpi_status_t st = device_setup(&dev);
    if (st != DPI_OK) return st;
    const uint32_t G = static_cast<uint32_t>(G64);
    const int lanes = [&] { int p = 1; while (p < static_cast<int>(row_bytes / 16)) p <<= 1; return p; }();

    // Grid of the fused kernel, by the rule dpi_plan_create applies (prepare_launches in dpi_api.cu): at most one resident
    // wave, at most kFusedMaxChunks chunks, no chunk smaller than one bag per lane group, at most 2048 bags per chunk.
    const int occ = fused_occupancy(dtype, false, lanes, static_cast<uint32_t>(T));
    if (occ <= 0) return report_error(DPI_ERR_UNSUPPORTED, "no fused forward kernel for %d lanes per row", lanes);
    uint64_t chunks = std::min<uint64_t>(kFusedMaxChunks, static_cast<uint64_t>(dev->num_sms) * occ);
    const uint32_t min_bags = static_cast<uint32_t>(kFusedThreads / lanes);
    chunks = std::min<uint64_t>(chunks, (static_cast<uint64_t>(G) + min_bags - 1) / min_bags);
    if (chunks < 1) chunks = 1;
    const uint32_t chunk_bags = static_cast<uint32_t>((G + chunks - 1) / chunks);
    if (chunk_bags > static_cast<uint32_t>(kFusedMaxChunkBags))
        return report_error(DPI_ERR_UNSUPPORTED, "%u bags on a %d-SM device need chunks of %u bags; the fused kernel holds at most %d", G, dev->num_sms, chunk_bags, kFusedMaxChunkBags);

    FusedArgs f{};
    PlanArgs& pa = f.plan;
    pa.len = lengths_dev;
    pa.offsets = reinterpret_cast<int32_t*>(dev->scratch + kOffOffsets);
    pa.seg = reinterpret_cast<int2*>(dev->scratch + kOffSeg);
    pa.meta = reinterpret_cast<int32_t*>(dev->scratch + kOffMeta);
    pa.status = reinterpret_cast<ulonglong2*>(dev->scratch + kOffStatus);
    pa.state = reinterpret_cast<unsigned int*>(dev->scratch + kOffState);
    pa.G = G;
    pa.K = 1u << kQuantumShift;
    pa.seg_cap = kSegCap;
    pa.num_chunks = (G + chunk_bags - 1) / chunk_bags;
    pa.max_indices = 0x7fffffffu;   // N is not known on the host; the precondition N < 2^30 is the caller's (dpi.h)
    f.chunk_bags = chunk_bags;
    f.items = (chunk_bags + kFusedThreads - 1) / kFusedThreads;
    f.k_shift = kQuantumShift;
    LookupArgs& la = f.look;
    la.tables = table_ptrs_dev;
    la.indices = indices_dev;
    la.offsets = pa.offsets;
    la.seg = pa.seg;
    la.meta = pa.meta;
    la.out = out_dev;
    la.G = G;
    la.T = static_cast<uint32_t>(T);
    la.B = static_cast<uint32_t>(B);
    la.nvec = static_cast<uint32_t>(row_bytes / 16);
    if (pooling) {
        for (int t = 0; t < T; ++t) {
            if (pooling[t] > 1) return report_error(DPI_ERR_INVALID_ARG, "pooling[%d] = %d is not a dpi_pool_t", t, pooling[t]);
            if (pooling[t] == DPI_POOL_MEAN) {
                la.pool.w[t >> 5] |= 1u << (t & 31);
                f.any_mean = 1;
            }
        }
    }

    cudaStream_t s = static_cast<cudaStream_t>(stream);
    noalloc_reset_kernel<<<1, 256, 0, s>>>();
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return report_error(DPI_ERR_CUDA, "scratch reset kernel launch: %s", cudaGetErrorString(e));
    // plain launch (no programmatic dependent launch): the kernel must not start before the reset above has finished
    e = launch_fused(f, dtype, false, lanes, false, s);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return report_error(DPI_ERR_CUDA, "fused forward kernel launch: %s", cudaGetErrorString(e)); }
    return DPI_OK;
}
