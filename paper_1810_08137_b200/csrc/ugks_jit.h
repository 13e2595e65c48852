// ugks_jit.h -- host interface of the run-time specialised kernels (ugks_jit.cu).  Not part of the C ABI.
#pragma once
#include "ugks_common.cuh"

#include <string>
#include <vector>

struct KArgs_h {                     // host mirror of KArgs (ugks_jit_common.cuh): device pointers only
    const double *fcur; double *fnew; double *cmom; const double *frec0, *frec1, *crec, *ghost, *wallg;
};

struct JitModule {
    std::vector<char> image;         // cubin (kept alive for the library)
    cudaLibrary_t lib = nullptr;
    cudaKernel_t k_mom = nullptr, k_momx = nullptr, k_upd = nullptr;
    int threads = 0, smem_mom = 0, smem_momx = 0, smem_upd = 0;
};

size_t jit_smem_cell_moments(const UgksParams &P);
size_t jit_smem_flux_update(const UgksParams &P);
std::string jit_prelude(const UgksParams &P, const int4 *chunks, const double *u, const double *wu, const double *v, const double *wv);
int jit_compile(const std::string &prelude, std::vector<char> *cubin, std::string *log, bool verbose);
// module for this geometry (compiled once per process and prelude); sets the shared-memory opt-in on the current device
int jit_get(const UgksParams &P, const int4 *chunks, const double *u, const double *wu, const double *v, const double *wv,
            JitModule **out, char *err, size_t errlen);
int jit_launch_cell_moments(const JitModule *m, const UgksParams &P, int cur, cudaStream_t st);
int jit_launch_flux_update(const JitModule *m, const UgksParams &P, int cur, cudaStream_t st);
