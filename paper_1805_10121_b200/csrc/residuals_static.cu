// chase_residuals_static (include/chase_filter.h): the residual norms of chase_residuals (Alg. 1 l.8,
// PAPER.md:160; Listing 1 Resd) for callers that have no device memory to hand over as
// scratch and are not allowed to obtain any.
//
// Who that is: a solver that runs inside somebody else's memory budget.  Typical cases are a plug-in of a
// host application whose own pool allocator has already claimed the whole GPU (a cudaMalloc from the
// plug-in then simply fails, or steals memory the host application counts on), a rank of a job whose
// per-process HBM share was fixed at start-up, and a time-critical loop that must not enter the driver's
// allocator because cudaMalloc / cudaFree serialise the whole device while they run.  chase_residuals
// wants an N x ncols scratch block from such a caller, chase_hemm and chase_filter fetch theirs from
// cudaMalloc / cudaMallocAsync; this entry point does neither.
//
// How: the scratch is g_static_scratch below, CHASE_STATIC_SCRATCH_BYTES of zero-initialised device memory
// that belongs to the library image.  Every GPU on which this library's module gets loaded carries that
// array from the moment of loading until the process exits, used or not -- which is why it is kept modest
// and why problems that do not fit are refused (CHASE_ERR_STATIC_LIMIT) rather than served some other way.
//
// In HOST code the identifier g_static_scratch is only a handle of the symbol, not a device address (a
// kernel handed `g_static_scratch` from the host side would fault, or scribble over host memory where the
// GPU can reach it).  The device address differs per GPU; scratch_for_current_device() asks the runtime
// for it with cudaGetSymbolAddress once per device and remembers the answer.
#include <cmath>
#include <mutex>

#include "chase_internal.h"

namespace {

using namespace chase;

static __device__ __align__(256) unsigned char g_static_scratch[CHASE_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_addr_mu;
void *g_addr[kMaxDevices] = {};

// Device address of g_static_scratch on the CURRENT device.  The first call on a device resolves the
// symbol (this is also what makes the runtime load the library's module on that device); later calls
// return the cached pointer without touching the runtime.
cudaError_t scratch_for_current_device(unsigned char **out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_addr_mu);
    if (!g_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_addr[dev] = p;
    }
    *out = (unsigned char *)g_addr[dev];
    return cudaSuccess;
}

size_t elem_size(chase_dtype_t dtype) {
    switch (dtype) {
        case CHASE_F32: return 4;
        case CHASE_F64: return 8;
        case CHASE_C64: return 8;
        case CHASE_C128: return 16;
        default: return 0;
    }
}

}  // namespace

extern "C" int chase_residuals_static(const void *H, int64_t N, const void *V, int64_t ncols, const double *ritzv,
                                      double *resid, chase_dtype_t dtype, void *stream_) {
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t w = elem_size(dtype);
    if (w == 0) return CHASE_ERR_DTYPE;
    if (N <= 0 || ncols < 0 || N > ((int64_t)1 << 30) || ncols > ((int64_t)1 << 30)) return CHASE_ERR_ARG;
    if (!H || (ncols > 0 && (!V || !ritzv || !resid))) return CHASE_ERR_ARG;
    if (ncols == 0) return CHASE_OK;
    for (int64_t j = 0; j < ncols; ++j)
        if (!std::isfinite(ritzv[j])) return CHASE_ERR_ARG;
    if (((uintptr_t)H | (uintptr_t)V) & 15) return CHASE_ERR_ALIGN;

    // Same scratch layout as chase_residuals: [R = H V - V diag(ritzv), vb bytes | control block of the step
    // kernel (stream-K flags + partial tiles on the FP64 tensor path, the 256-byte soft-barrier counter on
    // the tcgen05 path, nothing otherwise) | ritzv as device doubles].  The size test comes before any CUDA
    // call, so an oversized request costs nothing and touches nothing.
    const size_t need = chase_residuals_workspace_bytes(N, ncols, dtype);
    if (need == 0) return CHASE_ERR_ARG;
    if (need > (size_t)CHASE_STATIC_SCRATCH_BYTES) return CHASE_ERR_STATIC_LIMIT;

    unsigned char *scratch = nullptr;
    cudaError_t e = scratch_for_current_device(&scratch);
    if (e != cudaSuccess) return (int)e;

    const size_t vb = ((size_t)N * (size_t)ncols * w + 255) / 256 * 256;
    const size_t r_bytes = chase_filter_workspace_bytes(N, ncols, dtype);
    unsigned char *ctrl = scratch + vb;
    double *d_shift = (double *)(scratch + r_bytes);
    const int path = chase_filter_kernel_path(N, ncols, dtype);

    // The array still holds whatever the previous call (any shape, any dtype) left in it.  R and the shifts
    // are written before they are read; the step kernels' flags and counters are the part that has to start
    // from zero, so that part is cleared here, in stream order, on every call.
    const size_t ctrl_clear = path == 1 ? kSkFlagBytes : (path == 2 ? 256 : 0);
    if (ctrl_clear && (e = cudaMemsetAsync(ctrl, 0, ctrl_clear, stream)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(d_shift, ritzv, (size_t)ncols * sizeof(double), cudaMemcpyHostToDevice, stream)) !=
        cudaSuccess)
        return (int)e;

    int rc;
    if (path == 2 && ncols >= 32) {
        // tcgen05 kernel, as launch_one_step would pick it, except that the soft-barrier counter is the one
        // inside the static array instead of the cudaMalloc'ed process-wide one.
        Tf32Plan plan;
        if ((e = tf32_plan_create(&plan, dtype, H, N, const_cast<void *>(V), scratch, vb, ncols, stream)) != cudaSuccess)
            return (int)e;
        rc = (int)tf32_launch_step(&plan, 0, 0, 1.0, 0.0, 0.0, 0, stream, d_shift);
    } else {
        // FP64 tensor kernel with its stream-K scratch inside the static array (a non-null scratch pointer
        // keeps it away from the library's cudaMalloc'ed cache), or one of the kernels that need no scratch.
        rc = launch_one_step(H, N, V, scratch, ncols, 1.0, 0.0, 0.0, d_shift, 0, dtype, stream,
                             path == 1 ? (void *)ctrl : nullptr);
    }
    if (rc != CHASE_OK) return rc;
    return (int)launch_column_norms(dtype, scratch, N, ncols, resid, stream);
}
