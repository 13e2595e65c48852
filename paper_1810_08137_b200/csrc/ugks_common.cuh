// ugks_common.cuh -- shared declarations of the CUDA path (sm_100a).  Not part of the C ABI.
// Notation follows DESIGN.md / include/ugks.h: cells (i,j), velocity point q = m*Nu + k,
// local face frame (n,t) = (u,v) on x-faces and (v,u) on y-faces (AMB-21).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define UGKS_PI 3.14159265358979323846264338327950288

enum { BC_PERIODIC = 0, BC_FIXED = 1, BC_WALL = 2 };

constexpr int NMOM = 12;    // per-(face,chunk) raw moments: 11 used, padded to 12
constexpr int NCOEF = 24;   // per-face coefficients consumed by the flux/update kernel
constexpr int NCELL = 12;   // per-cell coefficients consumed by the flux/update kernel
constexpr int RINGX = 6;    // face_moments: stencil ring slots (4 live rows + 2 in flight)
constexpr int NSX = 4;      // flux_update: x-ring slots (2 live rows + 2 in flight; older rows live in registers)

// coefficient record written by k_face_scalars (S2..S5) and read by k_flux_update (S6, S8)
// P(n,t) = Mt1 + Mt2 (n a.psi + t b.psi) + Mt3 A.psi = sum c_ab n^a t^b (total degree <= 3); the five coefficients that
// contain a (c10, c20, c30, c11, c12) come in an L (n > 0, a_L) and an R (n < 0, a_R) variant.
enum { CF_C0 = 0, CF_U = 1, CF_V = 2, CF_LAM = 3, CF_MT4 = 4, CF_MT5 = 5, CF_RHOW = 6, CF_TYPE = 7,
       CF_C00 = 8, CF_C01 = 9, CF_C02 = 10, CF_C03 = 11, CF_C21 = 12, CF_L = 13, CF_R = 18 };
// per-cell record written by k_cell_scalars (U1, U2) and read by k_flux_update (U3)
enum { CC_GN = 0, CC_UN = 1, CC_VN = 2, CC_LN = 3, CC_GP = 4, CC_UP = 5, CC_VP = 6, CC_LP = 7, CC_KF = 8, CC_KD = 9 };

struct UgksParams {
    int I, J, Nu, Nv, N, Npad;
    double dx, dy, dt, omega, mu_ref;
    int bc[4];                       // xmin, xmax, ymin, ymax
    const double *u, *wu, *v, *wv;   // device copies of the velocity nodes / weights
    const double *ghost;             // [4][Npad] FIXED ghost rows f_b (O0)
    const double *wallg;             // [4][Npad] wall Maxwellians of (1,Uw,Vw,1/Tw) (O0)
    const double *Wb;                // [4][4]   cons(prim_b) of FIXED sides
    const double *wallG;             // [4][4]   sum_{outgoing} w n psi_loc g_w per wall side (local frame)
    double *f[2];                    // ping-pong copies of f, rows padded to Npad
    double *W[2];                    // ping-pong copies of W [cells][4]
    double *mom[2];                  // [faces][nchunk][NMOM], x then y faces
    double *coef[2];                 // [faces][NCOEF]
    double *fw[2];                   // [faces][4] time-integrated macroscopic flux, global frame
    double *cellc;                   // [cells][NCELL]
    double *respart;                 // [resblocks][8] partial residual sums
    int *status;                     // [2]: non-physical-state flags
    int strip;                       // faces / cells per CTA march
    int chunk_m;                     // velocity rows (m) per chunk
    int nchunk;                      // chunks per row of f
    int R;                           // m-rows processed in parallel by one CTA (blockDim = Nu*R)
    int npt;                         // velocity points per thread = ceil(chunk_m / R), 1..8 (template parameter)
};

static __host__ __device__ inline int nfaces_x(const UgksParams &P) { return (P.I + 1) * P.J; }
static __host__ __device__ inline int nfaces_y(const UgksParams &P) { return P.I * (P.J + 1); }

// ---------------------------------------------------------------------------------------------
// row lookup (O1): returns the row of cell `pos` on the line (dir 0: (pos,line), dir 1: (line,pos)),
// resolving PERIODIC wrap and FIXED ghosts.  A WALL neighbour is "missing": *missing = 1 and a valid
// (clamped) row is returned so that staging stays uniform; its values are never used.
template <int DIR>
__device__ __forceinline__ const double *row_ptr(const UgksParams &P, const double *f, int pos, int line, int *missing)
{
    const int n = DIR == 0 ? P.I : P.J;
    const int lo = DIR == 0 ? 0 : 2, hi = lo + 1;
    *missing = 0;
    if (pos < 0) {
        if (P.bc[lo] == BC_PERIODIC) pos += n;
        else if (P.bc[lo] == BC_FIXED) return P.ghost + (size_t)lo * P.Npad;
        else { *missing = 1; pos = 0; }
    } else if (pos >= n) {
        if (P.bc[hi] == BC_PERIODIC) pos -= n;
        else if (P.bc[hi] == BC_FIXED) return P.ghost + (size_t)hi * P.Npad;
        else { *missing = 1; pos = n - 1; }
    }
    const size_t cell = DIR == 0 ? (size_t)line * P.I + pos : (size_t)pos * P.I + line;
    return f + cell * P.Npad;
}

// ---------------------------------------------------------------------------------------------
// mbarrier + 1-D TMA bulk copy (cp.async.bulk; SASS UBLKCP)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n .reg .pred p;\n WAIT_%=:\n"
                 " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// ---------------------------------------------------------------------------------------------
// h*sigma of the van Leer limiter (AMB-4) from un-normalised differences dm = f_c - f_{c-1},
// dp = f_{c+1} - f_c:  h*sigma = (dx/2) * 2 (dm/dx)(dp/dx)/((dm+dp)/dx) = dm dp / (dm + dp).
__device__ __forceinline__ double vl_half(double dm, double dp)
{
    const double pr = dm * dp;
    return pr > 0.0 ? pr / (dm + dp) : 0.0;
}

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// launchers (one per translation unit); each returns the number of kernels it enqueued
int launch_face_moments(const UgksParams &P, int cur, int dir, cudaStream_t st);
int launch_face_scalars(const UgksParams &P, int cur, cudaStream_t st);
int launch_cell_scalars(const UgksParams &P, int cur, int resblocks, cudaStream_t st);
int launch_flux_update(const UgksParams &P, int cur, cudaStream_t st);
int launch_setup(const UgksParams &P, const double *bc_prims /*dev [4][4]*/, double *ghost, double *wallg,
                 double *Wb, double *wallG, cudaStream_t st);
int launch_residual_final(const UgksParams &P, int resblocks, double *res_dev, cudaStream_t st);
int launch_moments_of_f(const UgksParams &P, const double *f, double *Wf, cudaStream_t st);
int setup_moments_attributes(const UgksParams &P);
int setup_update_attributes(const UgksParams &P);
size_t smem_face_moments(const UgksParams &P);
size_t smem_flux_update(const UgksParams &P);
