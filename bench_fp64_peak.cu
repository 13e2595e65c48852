// bench_fp64_peak.cu -- bench.py's helper (NOT part of libugks): measured throughput of the plain FP64 pipe (DFMA), the
// arithmetic roof quoted beside the HBM roofline (MEASURED_PEAKS.json carries no FP64 figure).
// bench.py compiles it in-tree with nvcc (sm_100a) into libbench_fp64.so and calls bench_fp64_peak through ctypes.
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

extern "C" int bench_fp64_peak(double *thread_dfma_per_s)
{
    if (!thread_dfma_per_s) return 1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 3;
    const int blocks = sms * 8, threads = 256, iters = 1 << 14;
    double *buf = nullptr;
    if (cudaMalloc(&buf, sizeof(double) * blocks * threads) != cudaSuccess) return 2;
    cudaStream_t st;
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(buf); return 3; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {                              // first pass warms up; best of the rest
        cudaEventRecord(e0, st);
        k_dfma_peak<<<blocks, threads, 0, st>>>(buf, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); cudaStreamDestroy(st); return 3; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = 8.0 * iters * (double)blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaStreamDestroy(st);
    cudaFree(buf);
    *thread_dfma_per_s = best;
    return 0;
}
