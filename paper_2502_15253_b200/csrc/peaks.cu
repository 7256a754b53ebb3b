/*
 * peaks.cu -- microbenchmark of the pipe that bounds the batched path: fp64 FMA issue rate of
 * the whole chip (the hot loop is ~90 % DFMA/DADD/DMUL, all of which go
 * through the same 64-lane/clk/SM fp64 pipe).  Reported next to the nominal figure by bench.py.
 */
#include <time.h>

#include "internal.h"

namespace phylino {

namespace {

constexpr int CHAINS = 8;

__global__ void __launch_bounds__(256) dfma_kernel(int iters, double seed, double *sink)
{
    double a[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) a[c] = seed + threadIdx.x * 1e-9 + c;
    const double m = 0.999999999, b = 1e-12;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) a[c] = fma(a[c], m, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += a[c];
    if (s == 123.456) sink[0] = s;               /* never true; keeps the chains alive */
}

__global__ void empty_kernel() {}

/* plain coalesced 16-byte loads over [src, src + n16 * 16), four in flight per thread */
__global__ void __launch_bounds__(256) stream_kernel(const double2 *src, size_t n16, double *sink)
{
    double acc = 0.0;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const double2 a = __ldg(src + i), b = __ldg(src + i + stride), c = __ldg(src + i + 2 * stride),
                      d = __ldg(src + i + 3 * stride);
        acc += a.x + b.x + c.x + d.x;
    }
    for (; i < n16; i += stride) acc += __ldg(src + i).x;
    if (acc == 123.456) sink[0] = acc;            /* never true; keeps the loads alive */
}

} // namespace

/* Host wall time of `reps` x (launch of an empty kernel + stream synchronise), in microseconds per
 * repetition: the floor under any single call whose result the host waits for (config 1 is
 * reported against it, not against HBM). */
cudaError_t run_launch_floor(int reps, cudaStream_t st, double *us_per_call)
{
    empty_kernel<<<1, 32, 0, st>>>();
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    for (int i = 0; i < reps; ++i) {
        empty_kernel<<<1, 32, 0, st>>>();
        e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return e;
    }
    clock_gettime(CLOCK_MONOTONIC, &t1);
    *us_per_call = ((double)(t1.tv_sec - t0.tv_sec) * 1e6 + (double)(t1.tv_nsec - t0.tv_nsec) * 1e-3) / reps;
    return cudaGetLastError();
}

/* Device time (CUDA events, best of `reps`) of ONE kernel that only reads `bytes` from HBM with plain coalesced
 * loads, L2 flushed before every repetition: what a call bound by its event bytes can at best take, launch ramp
 * included -- the practical floor beside the bytes / peak-bandwidth figure (a 72 MB read takes about 20 us on a
 * B200 although 72 MB / 6.55 TB/s is 11 us). */
cudaError_t run_hbm_read_floor(size_t bytes, int reps, cudaStream_t st, double *us_best)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const size_t flush_bytes = (size_t)256 << 20;
    char *src = nullptr, *flush = nullptr;
    double *sink = nullptr;
    e = cudaMalloc((void **)&src, bytes + 16);
    if (e == cudaSuccess) e = cudaMalloc((void **)&flush, flush_bytes);
    if (e == cudaSuccess) e = cudaMalloc((void **)&sink, sizeof(double));
    if (e == cudaSuccess) e = cudaMemsetAsync(src, 1, bytes + 16, st);
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    double best = 1e300;
    for (int i = 0; e == cudaSuccess && i < reps + 2; ++i) {
        e = cudaMemsetAsync(flush, i, flush_bytes, st);
        if (e != cudaSuccess) break;
        cudaEventRecord(t0, st);
        stream_kernel<<<sms * 8, 256, 0, st>>>((const double2 *)src, bytes / 16, sink);
        cudaEventRecord(t1, st);
        e = cudaEventSynchronize(t1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
        if (e == cudaSuccess && i >= 2 && ms * 1e3 < best) best = ms * 1e3;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(src); cudaFree(flush); cudaFree(sink);
    if (e != cudaSuccess) return e;
    *us_best = best;
    return cudaSuccess;
}

cudaError_t run_peak_fp64(int iters, cudaStream_t st, double *dfma_per_s)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *sink = nullptr;
    e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = sms * 8;
    dfma_kernel<<<blocks, 256, 0, st>>>(iters / 8 + 1, 1.0, sink);      /* warm-up */
    cudaEventRecord(t0, st);
    dfma_kernel<<<blocks, 256, 0, st>>>(iters, 1.0, sink);
    cudaEventRecord(t1, st);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    double ops = (double)blocks * 256.0 * (double)iters * 4.0 * CHAINS;
    *dfma_per_s = ops / (ms * 1e-3);
    return cudaSuccess;
}

} // namespace phylino
