// vegas_static.cu -- vegas_refine_static_enqueue: the grid refinement (S7) for callers that have no way to hand the
// library device memory of their own making.
//
// Everything else in this library works inside a workspace the caller allocates (vegas_workspace_bytes ->
// torch.empty / cudaMalloc -> vegas_create).  Some callers cannot do that: code that runs as a plug-in inside another
// program -- a callback of an analysis framework, a custom operator, a step of somebody else's pipeline -- is handed
// device pointers to its inputs and outputs and nothing more.  The host program's pool already holds nearly all of the
// GPU's memory, so a cudaMalloc of their own may simply fail; they have no handle on that pool to ask it instead; and
// cudaMalloc / cudaFree stall the whole device while the host's other streams are busy, which a step in the middle of a
// pipelined loop must not do.  The refinement needs working memory beyond its inputs and outputs (the candidate edges,
// a writable copy of the histogram, the mapping table it rebuilds, the outcome flags), so for these callers that memory
// is compiled into the library: the file-scope array below.  The price is stated in the header: every GPU on which
// the library is loaded holds the array (about 256 KB) until the process exits, all calls on a device share it, and
// sizes beyond its capacity are refused.
//
// The arithmetic is refine_all of vegas_kernels.cuh, unchanged, launched with the geometry vegas_refine uses, so the
// new edges carry the same bits as vegas_refine's.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include <type_traits>

#include <cuda_runtime.h>

#include "../../include/vegas_b200.h"

int vegas_detail_fail(int code, const char* msg);        // vegas_api.cu: records the text vegas_last_error() returns

namespace {

// vegas_kernels.cuh also defines the library's non-template kernels (refine_kernel, build_table_kernel, ...), which
// vegas_api.cu already gives external linkage.  Included inside this unnamed namespace (its system headers are
// included above, so their guards skip them here) this file gets private copies and the link sees no duplicates.
#include "vegas_kernels.cuh"

using namespace vegas;

constexpr int kMaxEdges = VEGAS_STATIC_MAX_EDGES;        // capacity in edges: dim * (nbins + 1)
constexpr int kStatusInts = 64;                          // status words live in the first 256 bytes after the doubles
constexpr size_t kStaticSmemReserve = 1024;              // refine_all's few static shared words, as in vegas_api.cu

// Layout (doubles): hist copy [kMaxEdges] | candidate edges [kMaxEdges] | table (lo, wd) [2 * kMaxEdges] | status ints.
// In HOST code the name g_refine_scratch is only a handle for the runtime (it is not a device address and must never
// be passed to a kernel): static_setup() below asks the runtime for the device address once per device.
static __device__ __align__(256) double g_refine_scratch[4 * kMaxEdges + kStatusInts * sizeof(int) / sizeof(double)];

// The variant of refine_kernel that owns no workspace.  One CTA.  `scratch` is the device address of g_refine_scratch.
//   edges_in [d][N+1], hist_in [d][N]: read only.   edges_out [d][N+1]: the refined grid, or a copy of edges_in when
//   the refinement is rejected (step 7).  status_out[0] = 0 refined / 1 rejected.
// The array still holds whatever the previous call left: the outcome counters are zeroed here (refine_all increments
// one of them); the histogram copy, the candidate edges and the table are overwritten before they are read.
__global__ void refine_static_kernel(const double* edges_in /* may alias edges_out */, const double* hist_in, int N,
                                     double alpha, int d, double* edges_out, int* status_out, double* scratch,
                                     int smem_bytes)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* hist = scratch;
    double* cand = scratch + kMaxEdges;
    double* table = scratch + 2 * kMaxEdges;
    int* status = reinterpret_cast<int*>(scratch + 4 * kMaxEdges);
    if (threadIdx.x < 3) status[threadIdx.x] = 0;
    for (int i = threadIdx.x; i < d * N; i += blockDim.x) hist[i] = hist_in[i];
    if (edges_out != edges_in)
        for (int i = threadIdx.x; i < d * (N + 1); i += blockDim.x) edges_out[i] = edges_in[i];
    __syncthreads();                                     // refine_all reads both through L2 (__ldcg)
    refine_all(edges_out, hist, N, alpha, cand, d, table, /*precision fp64*/ 0, status, smem_raw,
               static_cast<size_t>(smem_bytes), false);
    __syncthreads();
    if (threadIdx.x == 0) status_out[0] = status[2];
}

struct DeviceSetup {
    bool ready = false;
    double* scratch = nullptr;                           // device address of g_refine_scratch on this device
    int smem_optin = 0;
};
constexpr int kMaxDevices = 64;
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

int failf(int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    return vegas_detail_fail(code, buf);
}

#define STATIC_CUDA_TRY(expr)                                                                                   \
    do {                                                                                                        \
        cudaError_t e_ = (expr);                                                                                \
        if (e_ != cudaSuccess) return failf(VEGAS_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// Once per device, with that device current: the device address of the scratch array and the kernel's shared-memory
// opt-in.  Neither call allocates.
int static_setup(int dev, const DeviceSetup** out)
{
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& s = g_setup[dev];
    if (!s.ready) {
        int major = 0, minor = 0, optin = 0;
        STATIC_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        STATIC_CUDA_TRY(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
        if (major != 10 || minor != 0)
            return failf(VEGAS_EUNSUPPORTED, "device sm_%d%d: this library is built for sm_100a (B200) only", major, minor);
        STATIC_CUDA_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        void* p = nullptr;
        STATIC_CUDA_TRY(cudaGetSymbolAddress(&p, g_refine_scratch));
        if (!p) return failf(VEGAS_ECUDA, "cudaGetSymbolAddress returned a NULL address for the scratch array");
        STATIC_CUDA_TRY(cudaFuncSetAttribute(refine_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             optin - static_cast<int>(kStaticSmemReserve)));
        s.scratch = static_cast<double*>(p);
        s.smem_optin = optin;
        s.ready = true;
    }
    *out = &s;
    return VEGAS_OK;
}

}  // namespace

extern "C" int vegas_refine_static_enqueue(int dim, int nbins, double alpha, const double* dev_edges,
                                           const double* dev_hist, double* dev_new_edges, int* dev_status,
                                           void* cuda_stream)
{
    if (dim < 1 || dim > kMaxDim) return failf(VEGAS_EINVAL, "dim %d not in 1..%d", dim, kMaxDim);
    if (nbins < 2 || nbins > 4095) return failf(VEGAS_EINVAL, "nbins %d not in 2..4095", nbins);
    if (static_cast<long long>(dim) * (nbins + 1) > kMaxEdges)
        return failf(VEGAS_EINVAL,
                     "vegas_refine_static_enqueue: dim * (nbins + 1) = %lld edges exceeds the built-in scratch array's capacity "
                     "of %d (VEGAS_STATIC_MAX_EDGES); larger grids need a context with a caller-provided workspace (vegas_create + vegas_refine)",
                     static_cast<long long>(dim) * (nbins + 1), kMaxEdges);
    if (!(alpha >= 0.0)) return failf(VEGAS_EINVAL, "alpha must be >= 0");
    if (!dev_edges || !dev_hist || !dev_new_edges || !dev_status) return failf(VEGAS_EINVAL, "a device pointer is NULL");
    if ((reinterpret_cast<uintptr_t>(dev_edges) | reinterpret_cast<uintptr_t>(dev_hist) | reinterpret_cast<uintptr_t>(dev_new_edges)) & 7u)
        return failf(VEGAS_EINVAL, "dev_edges, dev_hist and dev_new_edges must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(dev_status) & 3u) return failf(VEGAS_EINVAL, "dev_status must be 4-byte aligned");

    int dev = -1;
    STATIC_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return failf(VEGAS_EUNSUPPORTED, "device ordinal %d beyond the %d this entry point keeps set-up for", dev, kMaxDevices);
    const DeviceSetup* s = nullptr;
    const int rc = static_setup(dev, &s);
    if (rc != VEGAS_OK) return rc;

    // the launch geometry of vegas_refine_enqueue: all dimensions in one CTA, as many at a time as fit in shared memory
    // (at most one per warp), ceil((N + 1) / 32) warps per dimension for the per-bin steps when the CTA has them
    const size_t per_dim = 4 * (static_cast<size_t>(nbins) + 1) * sizeof(double);
    const int warps = dim < 32 ? dim : 32;
    int cta_warps = warps * ((nbins + 1 + 31) / 32);
    if (cta_warps > 32) cta_warps = 32;
    const size_t max_smem = static_cast<size_t>(s->smem_optin) - kStaticSmemReserve;
    size_t smem = per_dim * static_cast<size_t>(warps);
    if (smem > max_smem) smem = (max_smem / per_dim) * per_dim;
    if (smem < per_dim) return failf(VEGAS_EINVAL, "nbins %d: one dimension's refinement does not fit in shared memory", nbins);
    refine_static_kernel<<<1, 32 * cta_warps, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
        dev_edges, dev_hist, nbins, alpha, dim, dev_new_edges, dev_status, s->scratch, static_cast<int>(smem));
    STATIC_CUDA_TRY(cudaGetLastError());
    return VEGAS_OK;
}
