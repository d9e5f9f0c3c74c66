// Measured fp64 peaks of the device (the roofline denominators bench.py reports against; MEASURED_PEAKS.json has
// no fp64 figure).  Two register-only kernels, each 8 independent accumulator chains per thread:
//   kind 0  DFMA   plain FP64 fused multiply-add pipe           2 flop per thread-instruction
//   kind 1  DMMA   mma.sync.aligned.m8n8k4.row.col.f64          2*8*8*4 = 512 flop per warp-instruction
#include "../../include/epx.h"
#include <cuda_runtime.h>

namespace {

constexpr int PK_THREADS = 256;
constexpr int PK_INNER = 512;

__global__ void __launch_bounds__(PK_THREADS) dfma_peak_kernel(int iters, double seed, double* __restrict__ sink)
{
    double a[8];
#pragma unroll
    for (int i = 0; i < 8; i++) a[i] = seed + threadIdx.x * 1e-9 + i;
    const double m = 1.0 - 1e-9, b = 1e-12;
    for (int it = 0; it < iters; it++) {
#pragma unroll 16
        for (int k = 0; k < PK_INNER / 8; k++) {
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = fma(a[i], m, b);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += a[i];
    if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(PK_THREADS) dmma_peak_kernel(int iters, double seed, double* __restrict__ sink)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = seed + i; c[i][1] = seed - i; }
    const double a = 1e-3 * (threadIdx.x & 31), b = 1e-3;
    for (int it = 0; it < iters; it++) {
#pragma unroll 8
        for (int k = 0; k < PK_INNER / 8; k++) {
#pragma unroll
            for (int i = 0; i < 8; i++)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}

}  // namespace

extern "C" int epx_measure_fp64_peak(int device, int kind, double ms_target, void* dev_scratch, void* cuda_stream,
                                     double* tflops)
{
    if (!tflops || !dev_scratch || kind < 0 || kind > 1 || !(ms_target > 0)) return EPX_E_ARG;
    if (cudaSetDevice(device) != cudaSuccess) return EPX_E_CUDA;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop{};
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return EPX_E_CUDA;
    const int blocks = prop.multiProcessorCount * 8;
    double* sink = (double*)dev_scratch;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    auto run = [&](int iters) -> float {
        cudaEventRecord(e0, s);
        if (kind == 0) dfma_peak_kernel<<<blocks, PK_THREADS, 0, s>>>(iters, 1.0, sink);
        else dmma_peak_kernel<<<blocks, PK_THREADS, 0, s>>>(iters, 1.0, sink);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        return ms;
    };
    run(4);                                  // warm-up
    float ms = run(64);
    int iters = (int)(64.0 * ms_target / (ms > 1e-3f ? ms : 1e-3f));
    if (iters < 64) iters = 64;
    if (iters > (1 << 22)) iters = 1 << 22;
    ms = run(iters);
    const double per_thread_instr = (double)iters * PK_INNER;
    double flops;
    if (kind == 0) flops = per_thread_instr * 2.0 * (double)blocks * PK_THREADS;
    else flops = per_thread_instr * 512.0 * (double)blocks * (PK_THREADS / 32);
    *tflops = flops / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return cudaGetLastError() == cudaSuccess ? EPX_OK : EPX_E_CUDA;
}
