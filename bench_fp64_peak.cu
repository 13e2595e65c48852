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

// The same pipe with THREE distinct register operands per DFMA (32 live accumulators, x[i] += x[i+5] * x[i+11]): what a kernel whose
// operands all come from different registers can reach -- the register-operand fetch, not the 16-lane pipe, then sets the rate
// (measured on B200: 1.22e13 against 1.70e13 for x = fma(x, a, b) with two operands held in the reuse cache).
__global__ void __launch_bounds__(128) k_dfma_3op(double *out, int iters, const double *in)
{
    double x[32];
    for (int i = 0; i < 32; ++i) x[i] = in[(threadIdx.x + i * 37) & 1023];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 32; ++i) x[i] = fma(x[(i + 5) % 32], x[(i + 11) % 32], x[i]);
    }
    double s = 0.0;
    for (int i = 0; i < 32; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// which: 0 = two operands reused (the pipe's own rate), 1 = three distinct register operands
static int measure(int which, double *thread_dfma_per_s)
{
    if (!thread_dfma_per_s) return 1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 3;
    const int blocks = sms * 8, threads = which ? 128 : 256, iters = which ? 1 << 12 : 1 << 14;
    double *buf = nullptr, *in = nullptr;
    if (cudaMalloc(&buf, sizeof(double) * blocks * threads) != cudaSuccess) return 2;
    if (cudaMalloc(&in, sizeof(double) * 1024) != cudaSuccess) { cudaFree(buf); return 2; }
    cudaMemset(in, 0, sizeof(double) * 1024);
    cudaStream_t st;
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(buf); cudaFree(in); return 3; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    int rc = 0;
    for (int rep = 0; rep < 5; ++rep) {                              // first pass warms up; best of the rest
        cudaEventRecord(e0, st);
        if (which) k_dfma_3op<<<blocks, threads, 0, st>>>(buf, iters, in);
        else k_dfma_peak<<<blocks, threads, 0, st>>>(buf, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = 3; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (which ? 32.0 : 8.0) * iters * (double)blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaStreamDestroy(st);
    cudaFree(buf); cudaFree(in);
    *thread_dfma_per_s = best;
    return rc;
}

extern "C" int bench_fp64_peak(double *thread_dfma_per_s) { return measure(0, thread_dfma_per_s); }
extern "C" int bench_fp64_peak_3op(double *thread_dfma_per_s) { return measure(1, thread_dfma_per_s); }
