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
