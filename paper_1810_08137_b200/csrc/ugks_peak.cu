// ugks_peak.cu -- ugks_fp64_peak: measured throughput of the plain FP64 pipe (DFMA), the arithmetic roof of the UGKS step
// (MEASURED_PEAKS.json carries no FP64 figure).  Not on the hot path.
#include "../../include/ugks.h"
#include <cuda_runtime.h>

__global__ void __launch_bounds__(256) k_dfma_peak(double *out, int iters, double a, double b)
{
    double x0 = threadIdx.x * 1e-9, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
    for (int i = 0; i < iters; ++i) {                                // 8 independent chains per thread
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

extern "C" int ugks_fp64_peak(double *thread_dfma_per_s)
{
    if (!thread_dfma_per_s) return UGKS_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return UGKS_ECUDA;
    const int blocks = sms * 8, threads = 256, iters = 1 << 14;
    double *buf = nullptr;
    if (cudaMalloc(&buf, sizeof(double) * blocks * threads) != cudaSuccess) return UGKS_ENOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {                              // first pass warms up; best of the rest
        cudaEventRecord(e0);
        k_dfma_peak<<<blocks, threads>>>(buf, iters, 0.999999, 1e-7);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); return UGKS_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = 8.0 * iters * (double)blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    *thread_dfma_per_s = best;
    return UGKS_OK;
}
