// ugks_jit.h -- host interface of the run-time specialised kernels (ugks_jit.cu).  Not part of the C ABI.
#pragma once
#include "ugks_common.cuh"

#include <string>
#include <vector>

struct KArgs_h {                     // host mirror of KArgs (ugks_jit_common.cuh): device pointers only
    const double *fcur; double *fnew; double *cmom; const double *frec0, *frec1, *crec, *ghost, *wallg;
};

enum { JIT_MOMENTS = 0, JIT_UPDATE = 1 };

// Launch geometry of ONE of the two f-sized kernels (each has its own: k_cell_moments likes more points per thread than
// k_flux_update).  Velocity-row chunks are sorted [v < 0][v > 0][mixed]; (m0, mc, sign, 0) each.
struct KGeom {
    int nneg = 0, npos = 0, nmix = 0, cmax = 0, R = 1, npt = 1, strip = 32;
    std::vector<int4> chunks;
    int nchunk() const { return (int)chunks.size(); }
    bool ragged() const { for (const int4 &c : chunks) if (c.y != cmax) return true; return false; }
};

struct JitKernel {
    std::vector<char> image;         // cubin (kept alive for the library)
    cudaLibrary_t lib = nullptr;
    cudaKernel_t k = nullptr, kx = nullptr;      // the kernel; for JIT_MOMENTS also the variant for mixed-sign chunks
    int threads = 0, smem = 0, smemx = 0;
    int users = 0;                   // contexts holding this kernel (jit_get takes a reference, jit_release drops it)
    unsigned long last_used = 0;     // for the eviction order of unused kernels
};

// dynamic shared memory of a kernel of this geometry (the larger of its variants)
size_t jit_smem(int kind, const UgksParams &P, const KGeom &G);
std::string jit_prelude(int kind, const UgksParams &P, const KGeom &G, const double *u, const double *wu, const double *v, const double *wv);
int jit_compile(int kind, const std::string &prelude, std::vector<char> *cubin, std::string *log, bool verbose);
// kernel for this geometry (compiled once per process and prelude); sets the shared-memory opt-in on the current device
int jit_get(int kind, const UgksParams &P, const KGeom &G, const double *u, const double *wu, const double *v, const double *wv,
            JitKernel **out, char *err, size_t errlen);
// drop the reference jit_get took.  Kernels nobody holds stay cached for the next context of that geometry, up to JIT_CACHE_MAX
// of them; beyond that the least recently used ones are unloaded (cudaLibraryUnload) and freed.
void jit_release(JitKernel *m);
constexpr int JIT_CACHE_MAX = 32;
int jit_ctas_per_sm(const JitKernel *m);
// CTAs per SM the kernel of this geometry is compiled for (__launch_bounds__): min(shared memory, 128 registers per thread);
// known without compiling, a lower bound of jit_ctas_per_sm
int jit_ctas_estimate(int kind, const UgksParams &P, const KGeom &G);
int jit_launch_cell_moments(const JitKernel *m, const UgksParams &P, const KGeom &G, int cur, cudaStream_t st);
int jit_launch_flux_update(const JitKernel *m, const UgksParams &P, const KGeom &G, int cur, cudaStream_t st);
