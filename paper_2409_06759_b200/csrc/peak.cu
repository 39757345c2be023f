// peak.cu -- register-resident DMMA.8x8x4 loop: the measured FP64 tensor-core roofline denominator.
// 8 warps per SM, 8 independent accumulator pairs per warp (the pipe needs >= 2 per sub-partition),
// 512 flop per warp-level mma.sync.m8n8k4.f64.
#include "kernels.h"

namespace tcb {

namespace {

__global__ void __launch_bounds__(256) dmma_peak_kernel(double *out, int iters)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = threadIdx.x * 1e-9, b = 1.0 + threadIdx.x * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * 256 + threadIdx.x] = s;
}

// the plain FP64 pipe for comparison: 16 independent DFMA chains per thread, 2 flop per FMA per lane
__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int iters)
{
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-3 + i;
    const double a = 1.0 + threadIdx.x * 1e-12, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    out[blockIdx.x * 256 + threadIdx.x] = s;
}

}  // namespace

cudaError_t run_dfma_peak(double milliseconds, double *tflops, cudaStream_t stream, int64_t *launches)
{
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, sizeof(double) * 256 * nsm * 4);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 20000, ctas = nsm * 4;
    const double flop_per_launch = (double)ctas * 256 * iters * 16 * 2.0;
    dfma_peak_kernel<<<ctas, 256, 0, stream>>>(out, iters);
    cudaStreamSynchronize(stream);
    int n = 0;
    float ms = 0.f;
    cudaEventRecord(e0, stream);
    do {
        for (int j = 0; j < 4; ++j) dfma_peak_kernel<<<ctas, 256, 0, stream>>>(out, iters);
        n += 4;
        if (launches) *launches += 4;
        cudaEventRecord(e1, stream);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        cudaEventElapsedTime(&ms, e0, e1);
    } while (ms < milliseconds);
    if (e == cudaSuccess) *tflops = flop_per_launch * n / (ms * 1e-3) * 1e-12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return e;
}

cudaError_t run_dmma_peak(double milliseconds, double *tflops, cudaStream_t stream, int64_t *launches)
{
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, sizeof(double) * 256 * nsm);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 40000;                      // ~2.6 ms per launch at 37 TFLOP/s
    const double flop_per_launch = (double)nsm * 8 * iters * 8 * 512.0;
    dmma_peak_kernel<<<nsm, 256, 0, stream>>>(out, iters);   // warm-up
    cudaStreamSynchronize(stream);
    int n = 0;
    float ms = 0.f;
    cudaEventRecord(e0, stream);
    do {
        for (int j = 0; j < 4; ++j) dmma_peak_kernel<<<nsm, 256, 0, stream>>>(out, iters);
        n += 4;
        if (launches) *launches += 4;
        cudaEventRecord(e1, stream);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        cudaEventElapsedTime(&ms, e0, e1);
    } while (ms < milliseconds);
    if (e == cudaSuccess) *tflops = flop_per_launch * n / (ms * 1e-3) * 1e-12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return e;
}

}  // namespace tcb
