// ugks_noalloc.cu -- ugks_residual_noalloc (include/ugks.h): the L2 residual of a step (RES row, O11) for callers that cannot
// allocate device memory.
//
// Who that is.  The context API never calls cudaMalloc either, but it needs a workspace the CALLER allocates, and the residual's
// per-block partial sums live in that workspace.  Some callers have nothing to allocate from and may not ask the driver:
//   - a convergence monitor or logging hook that is handed two W fields and nothing else, inside a process whose device memory
//     was given to a pool up front (a framework's caching allocator, a solver's arena): a raw cudaMalloc there fails with
//     out-of-memory although the pool has room, and the hook has no handle to the pool;
//   - a time loop that must not stall: cudaMalloc / cudaFree synchronise the whole device, so one call per residual check would
//     serialise every stream of the application.
// For them the partial sums sit in a fixed array inside the library image (below).  The price: the array is there on every GPU
// that loads libugks.so, used or not, until the process exits (UGKS_NOALLOC_SCRATCH_BYTES = 512 KiB), the field size is capped
// (UGKS_NOALLOC_MAX_CELLS), and all calls on one device share the one array.
//
// The arithmetic repeats the context path's (k_cell_scalars' residual partials + k_residual_final in ugks_scalars.cu) with the
// same block size and the same summation order; nothing of that path is changed or called here.
#include "../../include/ugks.h"

#include <cuda_runtime.h>
#include <mutex>
#include <stdio.h>

namespace {

constexpr int CELLS_PER_BLOCK = 128;                                   // as k_cell_scalars: one thread per cell
constexpr long MAX_BLOCKS = (UGKS_NOALLOC_MAX_CELLS + CELLS_PER_BLOCK - 1) / CELLS_PER_BLOCK;
constexpr int MAX_DEVICES = 64;

// [MAX_BLOCKS][8] partial sums: (sum dW_a^2, a = 0..3; sum |W_new_a|, a = 0..3) of one block of 128 cells.
// In HOST code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) double g_residual_scratch[MAX_BLOCKS * 8];
static_assert(sizeof(double) * MAX_BLOCKS * 8 == UGKS_NOALLOC_SCRATCH_BYTES, "ugks.h states the size of the static scratch array");

std::mutex g_mu;
double *g_scratch_dev[MAX_DEVICES];                                    // device address of the array on each device, 0 = not looked up yet

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// stage 1: every block writes its 8 sums to part[blockIdx.x][0..8) -- all slots the second stage reads are overwritten here,
// so nothing the previous call left in the array is ever read and nothing needs clearing
__global__ void __launch_bounds__(CELLS_PER_BLOCK) k_residual_partials_static(const double *__restrict__ W_old,
                                                                               const double *__restrict__ W_new, long ncells,
                                                                               double *__restrict__ part)
{
    const long c = (long)blockIdx.x * blockDim.x + threadIdx.x;
    double p[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
    if (c < ncells) {
        for (int r = 0; r < 4; ++r) {
            const double wn = W_new[c * 4 + r], d = wn - W_old[c * 4 + r];
            p[r] = d * d; p[4 + r] = fabs(wn);
        }
    }
    __shared__ double sh[CELLS_PER_BLOCK / 32][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int v = 0; v < 8; ++v) {
        const double s = warp_sum(p[v]);
        if (lane == 0) sh[warp][v] = s;
    }
    __syncthreads();
    if (threadIdx.x < 8) {
        double s = 0.0;
        for (int w = 0; w < CELLS_PER_BLOCK / 32; ++w) s += sh[w][threadIdx.x];
        part[(size_t)blockIdx.x * 8 + threadIdx.x] = s;
    }
}

// stage 2 (O11): fixed-order sum of the partials, res[a] = sqrt(Nc sum dW_a^2) / (sum |W_new_a| + 1e-300)
__global__ void __launch_bounds__(256) k_residual_final_static(const double *__restrict__ part, int nblocks, double ncells,
                                                               double *__restrict__ res)
{
    __shared__ double sh[8][8];
    const int v = threadIdx.x & 7, g = threadIdx.x >> 3;
    double s = 0.0;
    for (int b = g; b < nblocks; b += 32) s += part[(size_t)b * 8 + v];
    s += __shfl_xor_sync(0xffffffffu, s, 8);
    s += __shfl_xor_sync(0xffffffffu, s, 16);
    if ((threadIdx.x & 31) < 8) sh[threadIdx.x >> 5][v] = s;
    __syncthreads();
    if (threadIdx.x < 8) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[w][threadIdx.x];
        sh[0][threadIdx.x] = t;
    }
    __syncthreads();
    if (threadIdx.x < 4) res[threadIdx.x] = sqrt(ncells * sh[0][threadIdx.x]) / (sh[0][4 + threadIdx.x] + 1e-300);
}

int fail(char *err, size_t err_bytes, int code, const char *msg, const char *detail = "")
{
    if (err && err_bytes) snprintf(err, err_bytes, "ugks_residual_noalloc: %s%s", msg, detail);
    return code;
}

}   // namespace

extern "C" int ugks_residual_noalloc(const double *W_old, const double *W_new, long ncells, double *res, void *cuda_stream,
                                     char *err, size_t err_bytes)
{
    if (err && err_bytes) err[0] = 0;
    if (!W_old || !W_new || !res) return fail(err, err_bytes, UGKS_EINVAL, "NULL pointer");
    if (ncells < 1) return fail(err, err_bytes, UGKS_EINVAL, "ncells must be >= 1");
    if (ncells > UGKS_NOALLOC_MAX_CELLS) {
        char buf[256];
        snprintf(buf, sizeof buf, "%ld cells exceed UGKS_NOALLOC_MAX_CELLS = %ld, the size the library's static scratch array was "
                 "built for (use a context and ugks_residual for larger meshes)", ncells, (long)UGKS_NOALLOC_MAX_CELLS);
        return fail(err, err_bytes, UGKS_EINVAL, buf);
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(err, err_bytes, UGKS_ECUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(err, err_bytes, UGKS_EINVAL, "device ordinal out of range");
    double *scratch;
    {
        // once per device, with that device current: ask the runtime where THIS device keeps its copy of the array
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_dev[dev]) {
            double *p = nullptr;
            e = cudaGetSymbolAddress((void **)&p, g_residual_scratch);
            if (e != cudaSuccess || !p)
                return fail(err, err_bytes, UGKS_ECUDA, "cudaGetSymbolAddress(static scratch): ", cudaGetErrorString(e));
            g_scratch_dev[dev] = p;
        }
        scratch = g_scratch_dev[dev];
    }
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nblocks = (int)((ncells + CELLS_PER_BLOCK - 1) / CELLS_PER_BLOCK);
    k_residual_partials_static<<<nblocks, CELLS_PER_BLOCK, 0, st>>>(W_old, W_new, ncells, scratch);
    k_residual_final_static<<<1, 256, 0, st>>>(scratch, nblocks, (double)ncells, res);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(err, err_bytes, UGKS_ECUDA, "kernel launch: ", cudaGetErrorString(e));
    return UGKS_OK;
}
