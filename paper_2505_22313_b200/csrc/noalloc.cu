// noalloc.cu -- dop_prefilter_noalloc (include/dop.h): the Gaussian pre-filter F0 / A6 (blur.cu: rows into a scratch
// plane, columns out of it) for callers that cannot allocate -- CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  The scratch plane the two stencil kernels exchange is not taken from a workspace but from
// the file-scope device array below, DOP_NOALLOC_MAX_POINTS floats that every GPU which loads libdop.so holds until
// the process exits.  The call enqueues the same two kernels as the plan path (dop::launch_blur) with the taps as
// kernel parameters, so it needs none of the plan's device tables either: no cudaMalloc, cudaFree or allocating
// library routine is reached from here.
//
// In host code `noalloc_scratch` is only a host-side stand-in for the symbol, not a device address (a kernel given
// it would fault, or silently use host memory where the GPU can reach it): the address is looked up once per device,
// with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels receive.
//
// Every call on a device shares the one array and finds the previous call's contents in it.  Nothing has to start at
// zero: the row kernel overwrites all ny * nx floats the column kernel reads before that kernel starts (same stream),
// so no clear is enqueued.  Two calls that overlap on the GPU (different streams, or graph branches without an edge
// between them) race on the array; calls on one stream, or otherwise ordered, are safe.
#include <mutex>

#include "dop_internal.h"

static __device__ __align__(256) float noalloc_scratch[DOP_NOALLOC_MAX_POINTS];

namespace {

constexpr int kMaxDevices = 64;
float* g_scratch[kMaxDevices]; // device address of noalloc_scratch on device i (nullptr = not looked up yet)
std::mutex g_mu;

// device address of the scratch array on the current device (sm_100 only), looked up once per device
dop_status scratch_for_current_device(float** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return DOP_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return DOP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_scratch[dev] == nullptr) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return DOP_ERR_CUDA;
        if (major != 10) return DOP_ERR_ARCH;
        float* ptr = nullptr;
        if (cudaGetSymbolAddress((void**)&ptr, noalloc_scratch) != cudaSuccess || ptr == nullptr) return DOP_ERR_CUDA;
        g_scratch[dev] = ptr;
    }
    *out = g_scratch[dev];
    return DOP_OK;
}

} // namespace

extern "C" dop_status dop_prefilter_noalloc(const dop_plan* p, const float* d_in, float* d_out, void* cuda_stream)
{
    if (p == nullptr || d_in == nullptr || d_out == nullptr) return DOP_ERR_INVALID_ARG;
    if (!p->pre_stencil) return DOP_ERR_INVALID_ARG; // the plan has no stencil form of the pre-filter (see dop.h)
    if (p->desc.ny * p->desc.nx > (long long)DOP_NOALLOC_MAX_POINTS) return DOP_ERR_NOALLOC_LIMIT;
    float* scratch = nullptr;
    dop_status s = scratch_for_current_device(&scratch);
    if (s != DOP_OK) return s;
    cudaError_t e = dop::launch_blur(d_in, scratch, d_out, p->desc.ny, p->desc.nx, p->blur_radius, p->blur_wx.data(),
                                     p->blur_wy.data(), (cudaStream_t)cuda_stream, nullptr, nullptr);
    return e == cudaSuccess ? DOP_OK : DOP_ERR_CUDA;
}
