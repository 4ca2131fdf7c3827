// qa_static_workspace.cu -- qa_ground_state_open_static: the open-array ground-state search for callers that cannot call
// cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
//
// qa_ground_state_open needs a caller-allocated workspace (qa_workspace_bytes: 664 bytes per pixel at 16 dots; the
// prologue, walk and finish kernels of the three-launch path hand h, E(base), base, N_c and the pass-1 records to each other
// through it).  Here that workspace is a file-scope __device__ array of QA_STATIC_WORKSPACE_BYTES = 16 MiB: every GPU that
// loads the library holds it until the process exits.  The caller still passes V_g and the outputs.
//
// In host code the array's NAME is a host-side stand-in, not a device address (a kernel given it would fault, or use the
// wrong memory where the GPU can reach host memory): the address is fetched once per device, with that device current, by
// cudaGetSymbolAddress (qa_static_workspace_init, also called lazily by the entry point) and that pointer is what the kernels get.
//
// Every call on a device shares the one array and finds the previous call's contents in it.  Nothing the kernels read from
// the workspace has to start at zero except the work counter of the pruned walk, which the prologue kernel of every call
// zeroes itself (qa_kernels_generic.cu); every other field is written by a kernel of the call before a later kernel of the
// same call reads it.  Two calls that overlap on the GPU (different streams, or different host threads) RACE on the
// array: callers serialise them.  The entry point calls no cudaMalloc / cudaFree / allocating library routine (kernel-timing
// aid off: qa_set_kernel_timing(1) creates CUDA events lazily).
#include <cstdio>
#include <mutex>

#include "qa_internal.cuh"

#define QA_STATIC_WS_BYTES ((size_t)16 << 20)
static_assert(QA_STATIC_WS_BYTES == QA_STATIC_WORKSPACE_BYTES, "the header states the size of the array");

static __device__ __align__(256) unsigned char qa_static_workspace[QA_STATIC_WS_BYTES];

namespace {

constexpr int SW_MAX_DEVICES = 64;
std::mutex g_sw_mu;
void *g_sw_ptr[SW_MAX_DEVICES];  // device address of qa_static_workspace on device d (nullptr: not fetched yet)
thread_local char g_sw_err[256] = "";

// Device address of the array on the CURRENT device (fetched once per device, with that device current).
qa_status sw_pointer(void **out)
{
    *out = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        std::snprintf(g_sw_err, sizeof(g_sw_err), "cudaGetDevice: %s", cudaGetErrorString(e));
        return QA_ERR_CUDA;
    }
    if (dev < 0 || dev >= SW_MAX_DEVICES) {
        std::snprintf(g_sw_err, sizeof(g_sw_err), "device ordinal %d outside [0, %d)", dev, SW_MAX_DEVICES);
        return QA_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_sw_mu);
    if (!g_sw_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, qa_static_workspace);
        if (e != cudaSuccess || !p) {
            std::snprintf(g_sw_err, sizeof(g_sw_err), "cudaGetSymbolAddress(qa_static_workspace) on device %d: %s", dev,
                          cudaGetErrorString(e));
            return QA_ERR_CUDA;
        }
        g_sw_ptr[dev] = p;
    }
    *out = g_sw_ptr[dev];
    return QA_OK;
}

}  // namespace

extern "C" {

size_t qa_static_workspace_bytes(void) { return QA_STATIC_WS_BYTES; }

qa_status qa_static_workspace_init(void)
{
    void *p = nullptr;
    return sw_pointer(&p);
}

const char *qa_static_workspace_last_error(void) { return g_sw_err; }

qa_status qa_ground_state_open_static(const qa_model *model, const double *d_Vg, int64_t P, qa_algorithm alg, double t,
                                      int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                                      qa_stats *d_stats, void *cuda_stream)
{
    g_sw_err[0] = '\0';
    if (!model || P < 0) {
        std::snprintf(g_sw_err, sizeof(g_sw_err), "model is NULL or P < 0");
        return QA_ERR_INVALID_ARG;
    }
    const size_t need = qa_workspace_bytes(model, P);
    if (need > QA_STATIC_WS_BYTES) {
        std::snprintf(g_sw_err, sizeof(g_sw_err),
                      "P = %lld pixels need %zu bytes of scratch; the static workspace holds %zu (use qa_ground_state_open "
                      "with a workspace of your own, or split the sweep)",
                      (long long)P, need, (size_t)QA_STATIC_WS_BYTES);
        return QA_ERR_STATIC_WORKSPACE;
    }
    void *ws = nullptr;
    const qa_status st = sw_pointer(&ws);
    if (st != QA_OK) return st;
    return qa_ground_state_open(model, d_Vg, P, alg, t, n_max, d_N, d_E, d_xcont, d_Vsensor, d_stats, ws, QA_STATIC_WS_BYTES,
                                cuda_stream);
}

}  // extern "C"
