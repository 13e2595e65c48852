// ugks_common.cuh -- shared declarations of the CUDA path (sm_100a).  Not part of the C ABI.
// Notation follows DESIGN.md / include/ugks.h: cells (i,j), velocity point q = m*Nu + k,
// local face frame (n,t) = (u,v) on x-faces and (v,u) on y-faces (AMB-21).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define UGKS_PI 3.14159265358979323846264338327950288

enum { BC_PERIODIC = 0, BC_FIXED = 1, BC_WALL = 2 };

// ---------------------------------------------------------------------------------------------
// Per-(cell, chunk) half-range moment sets written by k_cell_moments and summed per face by k_face_scalars.
// A cell contributes (f_c + h sigma_c) to its plus-side face where n > 0 and (f_c - h sigma_c) to its minus-side face
// where n < 0 (O3 written cell by cell); sets: 0 = x+, 1 = x-, 2 = y+, 3 = y-.  13 raw sums per set, local frame,
// M_ab = sum w n^a t^b f0, S_ab = sum w n^a t^b (h sigma0):
// With the tangential reconstruction of f (option "tangential", O3t/O8t) five more, T_ab = sum w n^a t^b (h_t theta0), h_t = half
// the tangential spacing; the storage always has room for them.
constexpr int NSET = 4, NRAW = 18, NRAW_BASE = 13, CMS = NSET * NRAW;
enum { RW_M00 = 0, RW_M10, RW_M20, RW_M30, RW_M01, RW_M11, RW_M02, RW_M12, RW_S20, RW_S30, RW_S40, RW_S21, RW_S22,
       RW_T11, RW_T21, RW_T12, RW_T31, RW_T13 };

// Face record written by k_face_scalars (S2..S5; 24 coefficients) and k_tables (separable Maxwellian factors):
//   [0, FR_NCOEF)                        coefficients, see FR_*
//   [FR_NCOEF, FR_NCOEF + NuP)           E_k[k] = exp(-lam (u_k - c_u)^2)   (c_u = U0 on x-faces, V0 (tangential) on y-faces)
//   [FR_NCOEF + NuP, FR_NCOEF + NuP+NvP) E_m[m] = exp(-lam (v_m - c_v)^2)
// Flux polynomial  ell C0 [Mt1 + Mt2 (n a.psi + t b.psi) + Mt3 A.psi] = sum c_ab n^a t^b (total degree <= 3); the five
// coefficients that contain a (c10, c20, c30, c11, c12) come in an L (n > 0, a_L) and an R (n < 0, a_R) variant.
constexpr int FR_NCOEF = 24;
enum { FR_LAM = 0, FR_U = 1, FR_V = 2, FR_TYPE = 3, FR_RHOW = 4, FR_MT4 = 5 /* ell Mt4 */, FR_MT5 = 6 /* -ell Mt5 2/Delta */,
       FR_TAU = 7, FR_C00 = 8, FR_C01 = 9, FR_C02 = 10, FR_C03 = 11, FR_C21 = 12, FR_L = 13, FR_R = 18,
       FR_MT5T = 23 /* -ell Mt5 2/Delta_t (tangential spacing); 0 unless option "tangential" */ };
// offsets inside FR_L / FR_R
enum { LR_C10 = 0, LR_C20 = 1, LR_C30 = 2, LR_C11 = 3, LR_C12 = 4 };

// Cell record written by k_cell_scalars (U1, U2 scalars) and k_tables:
//   [0, CR_NCOEF)                          see CR_*
//   [CR_NCOEF, +NuP)                       gn_u[k] = GN exp(-lam_n (u_k - U_n)^2)    (relaxation prefactors folded in)
//   [CR_NCOEF + NuP, +NuP)                 gp_u[k] = GP exp(-lam_p (u_k - U_p)^2)
//   [CR_NCOEF + 2 NuP, +NvP)               gn_v[m] = exp(-lam_n (v_m - V_n)^2)
//   [CR_NCOEF + 2 NuP + NvP, +NvP)         gp_v[m] = exp(-lam_p (v_m - V_p)^2)
constexpr int CR_NCOEF = 12;
enum { CR_KF = 0, CR_KD = 1, CR_GN = 2, CR_GP = 3, CR_UN = 4, CR_VN = 5, CR_LN = 6, CR_UP = 7, CR_VP = 8, CR_LP = 9 };

struct UgksParams {
    int I, J, Nu, Nv, N, Npad;
    int NuP, NvP;                    // Nu, Nv rounded up to even (16-byte aligned table segments)
    int frs, crs;                    // record strides in doubles: FR_NCOEF + NuP + NvP, CR_NCOEF + 2 NuP + 2 NvP
    double dx, dy, dt, omega, mu_ref;
    double hu, hv;                   // spacing of the u / v nodes if they are equally spaced (to a few ulp), else 0 (k_tables)
    int bc[4];                       // xmin, xmax, ymin, ymax
    int tangential;                  // option "tangential" (NEXT-1, O3t/O8t): f is reconstructed in the tangential direction too
    const double *u, *wu, *v, *wv;   // device copies of the velocity nodes / weights
    const double *ghost;             // [4][Npad] FIXED ghost rows f_b (O0)
    const double *wallg;             // [4][Npad] wall Maxwellians of (1,Uw,Vw,1/Tw) (O0)
    const double *Wb;                // [4][4]   cons(prim_b) of FIXED sides
    const double *wallG;             // [4][4]   sum_{outgoing} w n psi_loc g_w per wall side (local frame)
    const double *ghostmom;          // [4][NRAW] half-range raw moments of the ghost row toward the domain (FIXED sides)
    const int4 *chunks;              // [nchunk] (m0, mc, sign of v over the chunk: +1 / -1 / 0 = mixed, 1 if row m0 is a v = 0 row of a +1 chunk)
    double *f[2];                    // ping-pong copies of f, rows padded to Npad
    double *W[2];                    // ping-pong copies of W [cells][4]
    double *cmom;                    // [cells][nchunk][CMS]: 4 sets x 13 base sums, then 4 sets x 5 T sums
    double *frec[2];                 // [faces][frs], x then y faces
    double *fw[2];                   // [faces][4] time-integrated macroscopic flux, global frame
    double *crec;                    // [cells][crs]
    double *respart;                 // [resblocks][8] partial residual sums
    int *status;                     // [2]: non-physical-state flags
    int strip;                       // cells per CTA march
    int nchunk;                      // velocity-row chunks (sign-uniform where possible), sorted [v < 0][v > 0][mixed]
    int nneg, npos, nmix;            // chunks per class
    int cmax;                        // rows of the largest chunk
    int R;                           // velocity rows processed in parallel by one CTA (threads = Nu*R rounded up to 32)
    int npt;                         // velocity points per thread = ceil(cmax / R), 1..16 (compile-time constant of the JIT kernels)
    int kxm_end, kxp_begin;          // columns with u_k <= 0 are [0, kxm_end), with u_k >= 0 [kxp_begin, Nu) (sorted nodes; else 0..Nu)
};

static __host__ __device__ inline int nfaces_x(const UgksParams &P) { return (P.I + 1) * P.J; }
static __host__ __device__ inline int nfaces_y(const UgksParams &P) { return P.I * (P.J + 1); }
static __host__ __device__ inline int pad2(int x) { return (x + 1) & ~1; }

// ---------------------------------------------------------------------------------------------
// row lookup (O1): returns the row of cell `pos` on the line (dir 0: (pos,line), dir 1: (line,pos)),
// resolving PERIODIC wrap and FIXED ghosts.  A WALL neighbour is "missing": a valid (clamped) row is returned so
// that staging stays uniform; its values are never used.
template <int DIR>
__device__ __forceinline__ const double *row_ptr(const UgksParams &P, const double *f, int pos, int line)
{
    const int n = DIR == 0 ? P.I : P.J;
    const int lo = DIR == 0 ? 0 : 2, hi = lo + 1;
    if (pos < 0) {
        if (P.bc[lo] == BC_PERIODIC) pos += n;
        else if (P.bc[lo] == BC_FIXED) return P.ghost + (size_t)lo * P.Npad;
        else pos = 0;
    } else if (pos >= n) {
        if (P.bc[hi] == BC_PERIODIC) pos -= n;
        else if (P.bc[hi] == BC_FIXED) return P.ghost + (size_t)hi * P.Npad;
        else pos = n - 1;
    }
    const size_t cell = DIR == 0 ? (size_t)line * P.I + pos : (size_t)pos * P.I + line;
    return f + cell * P.Npad;
}
// y-neighbour row `pos` of column 0 and its stride (doubles) from cell to cell along x: Npad, or 0 for a ghost row
__device__ __forceinline__ const double *yrow_base(const UgksParams &P, const double *f, int pos, int *stride)
{
    *stride = P.Npad;
    if (pos < 0) {
        if (P.bc[2] == BC_PERIODIC) pos += P.J;
        else if (P.bc[2] == BC_FIXED) { *stride = 0; return P.ghost + (size_t)2 * P.Npad; }
        else pos = 0;
    } else if (pos >= P.J) {
        if (P.bc[3] == BC_PERIODIC) pos -= P.J;
        else if (P.bc[3] == BC_FIXED) { *stride = 0; return P.ghost + (size_t)3 * P.Npad; }
        else pos = P.J - 1;
    }
    return f + (size_t)pos * P.I * P.Npad;
}
// shared-memory load at a byte offset from a (warp-uniform) base: LDS R, [Roff + URbase]
__device__ __forceinline__ double ldsd(const unsigned char *base, int off) { return *reinterpret_cast<const double *>(base + off); }
__device__ __forceinline__ double2 ldsd2(const unsigned char *base, int off) { return *reinterpret_cast<const double2 *>(base + off); }

// is cell `pos` of a line beyond a WALL side?
template <int DIR>
__device__ __forceinline__ bool beyond_wall(const UgksParams &P, int pos)
{
    const int n = DIR == 0 ? P.I : P.J, lo = DIR == 0 ? 0 : 2;
    return (pos < 0 && P.bc[lo] == BC_WALL) || (pos >= n && P.bc[lo + 1] == BC_WALL);
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
// h*sigma of the van Leer limiter (AMB-4) from un-normalised differences dm = f_c - f_{c-1}, dp = f_{c+1} - f_c:
//   h*sigma = (Delta/2) * 2 (dm/Delta)(dp/Delta)/((dm+dp)/Delta) = dm dp / (dm + dp)   if dm dp > 0, else 0.
// The reciprocal is MUFU.RCP64H (rel. error 2^-23) refined by one cubic step r (1 + e + e^2), e = 1 - s r: error
// e^3 ~ 2^-69, i.e. r is within ~1 ulp.  When dm dp > 0 (as a normal double) the sum is a normal number.  The sign test reads
// the high word: a product that underflowed to a denormal counts as 0, as in AMB-4's "underflow gives sigma = 0".
__device__ __forceinline__ double vl_half(double dm, double dp)
{
    const double pr = dm * dp, s = dm + dp;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));
    const double e = fma(-s, r, 1.0);
    const double t = fma(e, e, e);
    r = fma(r, t, r);
    const double hs = pr * r;
    return __double2hiint(pr) > 0 ? hs : 0.0;
}

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// launchers of the O(faces) / O(cells) kernels (ugks_scalars.cu); each returns the number of kernels it enqueued.  The two
// f-sized kernels are compiled at run time and launched through ugks_jit.h.
int launch_face_scalars(const UgksParams &P, int cur, cudaStream_t st);
int launch_cell_scalars(const UgksParams &P, int cur, int resblocks, cudaStream_t st);
int launch_tables(const UgksParams &P, cudaStream_t st);
int launch_setup(const UgksParams &P, const double *bc_prims /*dev [4][4]*/, double *ghost, double *wallg,
                 double *Wb, double *wallG, double *ghostmom, cudaStream_t st);
int launch_residual_final(const UgksParams &P, int resblocks, double *res_dev, cudaStream_t st);
int launch_moments_of_f(const UgksParams &P, const double *f, double *Wf, cudaStream_t st);
int launch_poison_smem(cudaStream_t st);
