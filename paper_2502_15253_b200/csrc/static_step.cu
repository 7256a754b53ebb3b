/*
 * static_step.cu -- phylino_variable_metric_step_static: the variable-metric step of the minimiser's loop
 * (R30) for callers that must not, or cannot, allocate device memory.
 *
 * Who that is.  phylino_variable_metric_step keeps its 2 N + 2 doubles of scratch (V dg, V grad and the two
 * curvature scalars) in a buffer that the context obtains with cudaMalloc, and the context itself is created with
 * allocations.  Three kinds of users of this library cannot accept that:
 *   - a fit that runs inside a process whose device memory is owned by someone else's pool (a PyTorch or RAPIDS
 *     caching allocator that has already taken the HBM, an MPS / MIG slice with a hard memory limit): a cudaMalloc
 *     from this library can fail there, or fragment the other owner's pool, although the memory "is free";
 *   - a minimiser loop with a latency budget: cudaMalloc and cudaFree synchronise the whole device, so one buffer
 *     that grows in the middle of a fit stalls every other stream of the process;
 *   - hosts that forbid allocation after start-up as a matter of policy (long-running services that must not be
 *     able to run out of memory half-way through a scan).
 * For them the scratch lives in the library image instead: one file-scope __device__ array of fixed size below.
 * The price is stated in phylino.h: a fixed upper limit on N, (2 * PHYLINO_STATIC_MAX_N + 2) * 8 = 32 784 bytes held
 * on every GPU that loads the library until the process exits, and one array shared by all calls.
 *
 * The arithmetic is that of the existing entry point -- the same kernels (launch_variable_metric_step in
 * consumers.cu), handed the address of the static array instead of the context's buffer -- so the two agree bit for bit.
 */
#include "internal.h"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace {

constexpr int kMaxN = PHYLINO_STATIC_MAX_N;
constexpr int kMaxDevices = 64;

/* vg [N] | s [N] | a, b.  In HOST code the name `static_scratch` is only a handle for cudaGetSymbolAddress: it is not a
 * device address and must never be passed to a kernel as one. */
static __device__ __align__(256) double static_scratch[2 * kMaxN + 2];

std::mutex g_lock;
double *g_scratch_of_device[kMaxDevices];      /* the array's address on each device, filled on first use */

void say(char *error, int error_len, const char *fmt, ...)
{
    if (!error || error_len <= 0) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(error, (size_t)error_len, fmt, ap);
    va_end(ap);
}

/* Address of the scratch array on the CURRENT device.  The first call on a device asks the runtime for it (which
 * also makes the runtime load this library's device code there); later calls read the table. */
cudaError_t scratch_here(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> hold(g_lock);
    if (dev >= 0 && dev < kMaxDevices && g_scratch_of_device[dev]) {
        *out = g_scratch_of_device[dev];
        return cudaSuccess;
    }
    double *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < kMaxDevices) g_scratch_of_device[dev] = p;
    *out = p;
    return cudaSuccess;
}

} // namespace

extern "C" phylino_status phylino_variable_metric_step_static(void *cuda_stream, int N, double *V, const double *dx,
                                                              const double *dg, const double *grad, double *direction,
                                                              double *edm, char *error, int error_len)
{
    if (error && error_len > 0) error[0] = '\0';
    if (N < 0 || N > kMaxN) {
        say(error, error_len,
            "N = %d is outside 0..%d (PHYLINO_STATIC_MAX_N): the scratch of this entry point is a fixed array; "
            "use phylino_variable_metric_step for larger problems", N, kMaxN);
        return PHYLINO_ERR_SHAPE;
    }
    if (N == 0) return PHYLINO_OK;
    if (!V || !grad || !direction || !edm) {
        say(error, error_len, "NULL V, grad, direction or edm");
        return PHYLINO_ERR_ARG;
    }
    if ((dx == nullptr) != (dg == nullptr)) {
        say(error, error_len, "dx and dg must both be given or both be NULL");
        return PHYLINO_ERR_ARG;
    }
    double *work = nullptr;
    cudaError_t e = scratch_here(&work);
    if (e != cudaSuccess) {
        say(error, error_len, "cudaGetSymbolAddress(static_scratch): %s", cudaGetErrorString(e));
        return PHYLINO_ERR_CUDA;
    }
    /* nothing in the array has to start at zero: vg, s and (a, b) are each written in full, on the stream, before
     * the kernel that reads them -- what an earlier call left behind is never read */
    e = phylino::launch_variable_metric_step(N, V, dx, dg, grad, direction, edm, work, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) {
        say(error, error_len, "kernel launch: %s", cudaGetErrorString(e));
        return PHYLINO_ERR_CUDA;
    }
    return PHYLINO_OK;
}
