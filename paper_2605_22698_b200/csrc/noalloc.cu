// e3_graph_prepare_noalloc: graph preparation (readings A11/A14/A15; see e3_graph_prepare) for callers that
// cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The scratch of e3_graph_prepare (4 + N + E + 4 int32: validation flags, the per-sender cursor, the unsorted fill) lives in ONE
// file-scope device array of kScratchBytes; every GPU that loads the library holds that much until the process exits.  All calls
// on a device share the array: calls that overlap on the GPU (two streams, two threads) race on it, and it keeps the contents of
// the previous call.  Nothing in it has to start at zero except the validation flags, which the validating call clears itself;
// the cursor (N entries) and the fill (E entries) are fully overwritten before they are read.
//
// Host code cannot use the array's name as a device address (it is a host-side stand-in): the address is taken once per device,
// with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels receive.
#include <mutex>

#include "e3_internal.h"

namespace {

constexpr size_t kScratchBytes = 32u << 20;      // 32 MiB: E + N <= 8 388 600 (configs 1-5 of BASELINE.json all fit)
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_graph_scratch[kScratchBytes];

std::mutex g_mu;
void *g_scratch_ptr[kMaxDevices] = {};           // device address of g_graph_scratch on each device, 0 = not asked yet

// the device address of the array on the CURRENT device (cudaGetSymbolAddress once per device)
int scratch_of_current_device(void **out)
{
    int dev = -1;
    E3_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { e3::set_error("e3_graph_prepare_noalloc: device ordinal %d not supported", dev); return E3_ERR_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_graph_scratch);
        if (e != cudaSuccess) return e3::cuda_fail(e, "cudaGetSymbolAddress(static graph scratch)");
        if (!p) { e3::set_error("e3_graph_prepare_noalloc: cudaGetSymbolAddress returned a null address"); return E3_ERR_CUDA; }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return E3_OK;
}

}  // namespace

extern "C" size_t e3_graph_noalloc_capacity_bytes(void) { return kScratchBytes; }

extern "C" int e3_graph_prepare_noalloc(const int32_t *senders, const int32_t *receivers, int64_t n_edges, int32_t n_nodes,
                                        int32_t *row_ptr, int32_t *perm_s, int32_t *col_ptr, int validate, e3_stream stream)
{
    using namespace e3;
    if (n_edges < 0 || n_nodes < 0 || n_edges > 0x7fffffffLL || !row_ptr || !col_ptr || (n_edges > 0 && (!senders || !receivers || !perm_s))) {
        set_error("e3_graph_prepare_noalloc: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    const size_t need = graph_workspace_bytes(n_edges, n_nodes);
    if (need > kScratchBytes) {
        set_error("e3_graph_prepare_noalloc: n_edges + n_nodes = %lld needs %zu bytes of scratch, the static array holds %zu "
                  "(n_edges + n_nodes <= %zu); use e3_graph_prepare with a caller-owned workspace",
                  (long long)n_edges + n_nodes, need, kScratchBytes, kScratchBytes / sizeof(int32_t) - 8);
        return E3_ERR_WORKSPACE;
    }
    void *scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != E3_OK) return rc;
    return launch_graph_prepare(senders, receivers, n_edges, n_nodes, row_ptr, perm_s, col_ptr, scratch, kScratchBytes, validate,
                                reinterpret_cast<cudaStream_t>(stream));
}
