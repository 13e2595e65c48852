// ugks_jit_common.cuh -- device-side declarations shared by the two f-sized kernels (k_cell_moments, k_flux_update).
//
// These kernels are compiled at ugks_init by NVRTC for sm_100a with the whole geometry of the context baked in as
// compile-time constants (the G_* macros of a generated prelude: mesh and velocity-grid sizes, boundary types, the
// velocity-row chunking, R / NPT, strip length, record strides; the velocity nodes, weights and the chunk table come as
// __constant__ arrays).  Every stride, trip count and job table below is therefore an immediate: the per-cell control code of
// the marching CTAs (about half of all executed instructions with run-time geometry: round 1, see the history row of profiles/r3_kernels.md) folds away.
// ugks_jit_check (include/ugks.h) compiles them for a geometry without a device: the offline build / SASS check.
//
// Notation follows DESIGN.md / include/ugks.h: cells (i,j), velocity point q = m*Nu + k, local face frame (n,t) = (u,v) on
// x-faces and (v,u) on y-faces (AMB-21).
#pragma once

#ifdef __CUDACC_RTC__
typedef unsigned int uint32_t;
typedef unsigned long long uint64_t;
#else
#include <stdint.h>
#endif

enum { BC_PERIODIC = 0, BC_FIXED = 1, BC_WALL = 2 };

// ---- geometry (all compile-time) ---------------------------------------------------------------------------------------
constexpr int GI = G_I, GJ = G_J, NU = G_NU, NV = G_NV, NPAD = G_NPAD, NUP = G_NUP, NVP = G_NVP;
constexpr int FRS = G_FRS, CRS = G_CRS;                              // face / cell record strides (doubles)
constexpr int BCX0 = G_BC0, BCX1 = G_BC1, BCY0 = G_BC2, BCY1 = G_BC3;
constexpr int NCHUNK = G_NCHUNK, MC = G_MC, R = G_R, NPT = G_NPT, STRIP = G_STRIP;
constexpr int NSTRIP = (GI + STRIP - 1) / STRIP;
constexpr int BT = ((NU * R + 31) / 32) * 32;                         // threads of a CTA: one per (column, parallel row); lane 0 of a rotating warp issues the bulk copies
constexpr int KXM_END = G_KXM_END, KXP_BEGIN = G_KXP_BEGIN;          // columns with u_k <= 0: [0, KXM_END); u_k >= 0: [KXP_BEGIN, NU)
constexpr int pad2c(int x) { return (x + 1) & ~1; }
constexpr int QB = G_QB;                                              // doubles per staged chunk of a row: >= MC*NU + 1 (shift of an odd start), even;
                                                                      // a 128-byte multiple where that costs no resident CTA (a warp's 256 contiguous
                                                                      // bytes then span two shared-memory lines, not three)
static_assert(QB >= MC * NU + 1 && QB % 2 == 0, "slot size");
constexpr int QBB = QB * 8;

// per-(cell, chunk) half-range raw moment sets (see ugks_common.cuh): sets 0 = x+, 1 = x-, 2 = y+, 3 = y-
// TG: option "tangential" (NEXT-1, O3t/O8t): five more raw sums per set, T_ab = sum w n^a t^b (h_t theta0)
constexpr bool TG = G_TANGENTIAL != 0;
constexpr int NSET = 4, NRAW = 18, NRK = TG ? 18 : 13, CMS = NSET * NRAW;       // storage stride / sums a kernel computes
enum { RW_M00 = 0, RW_M10, RW_M20, RW_M30, RW_M01, RW_M11, RW_M02, RW_M12, RW_S20, RW_S30, RW_S40, RW_S21, RW_S22,
       RW_T11, RW_T21, RW_T12, RW_T31, RW_T13 };
// face / cell record layout (see ugks_common.cuh)
constexpr int FR_NCOEF = 24;
enum { FR_LAM = 0, FR_U = 1, FR_V = 2, FR_TYPE = 3, FR_RHOW = 4, FR_MT4 = 5, FR_MT5 = 6, FR_TAU = 7, FR_C00 = 8, FR_C01 = 9,
       FR_C02 = 10, FR_C03 = 11, FR_C21 = 12, FR_L = 13, FR_R = 18, FR_MT5T = 23 };
enum { LR_C10 = 0, LR_C20 = 1, LR_C30 = 2, LR_C11 = 3, LR_C12 = 4 };
constexpr int CR_NCOEF = 12;
enum { CR_KF = 0, CR_KD = 1 };

// kernel arguments: device pointers only
struct KArgs {
    const double *fcur;              // f^n, rows padded to NPAD
    double *fnew;                    // f^{n+1}
    double *cmom;                    // [cells][NCHUNK][NSET][NRAW]
    const double *frec0, *frec1;     // face records, x / y faces
    const double *crec;              // cell records
    const double *ghost;             // [4][NPAD] FIXED ghost rows
    const double *wallg;             // [4][NPAD] wall Maxwellians
};

// ---- rows --------------------------------------------------------------------------------------------------------------
// row of cell `pos` on x-line j, resolving PERIODIC wrap and FIXED ghosts (O1); a WALL neighbour is "missing": a valid
// (clamped) row is returned so that staging stays uniform; its values are never used.
__device__ __forceinline__ const double *xrow_ptr(const double *f, const double *ghost, int pos, int j)
{
    if (pos < 0) {
        if (BCX0 == BC_PERIODIC) pos += GI;
        else if (BCX0 == BC_FIXED) return ghost;
        else pos = 0;
    } else if (pos >= GI) {
        if (BCX1 == BC_PERIODIC) pos -= GI;
        else if (BCX1 == BC_FIXED) return ghost + NPAD;
        else pos = GI - 1;
    }
    return f + ((size_t)j * GI + pos) * NPAD;
}
// y-neighbour row `pos` of column 0 and its stride (doubles) from cell to cell along x: NPAD, or 0 for a ghost row
__device__ __forceinline__ const double *yrow_base(const double *f, const double *ghost, int pos, int *stride)
{
    *stride = NPAD;
    if (pos < 0) {
        if (BCY0 == BC_PERIODIC) pos += GJ;
        else if (BCY0 == BC_FIXED) { *stride = 0; return ghost + 2 * NPAD; }
        else pos = 0;
    } else if (pos >= GJ) {
        if (BCY1 == BC_PERIODIC) pos -= GJ;
        else if (BCY1 == BC_FIXED) { *stride = 0; return ghost + 3 * NPAD; }
        else pos = GJ - 1;
    }
    return f + (size_t)pos * GI * NPAD;
}
// row of cell (i, jj) with BOTH directions resolved the way the neighbour lookup of O1 does (x first): PERIODIC wraps, a FIXED
// side returns its ghost row, a WALL neighbour is "missing" (a clamped valid row whose values are never used)
__device__ __forceinline__ const double *cell_row_ptr(const double *f, const double *ghost, int i, int jj)
{
    if (i < 0) {
        if (BCX0 == BC_PERIODIC) i += GI;
        else if (BCX0 == BC_FIXED) return ghost;
        else i = 0;
    } else if (i >= GI) {
        if (BCX1 == BC_PERIODIC) i -= GI;
        else if (BCX1 == BC_FIXED) return ghost + NPAD;
        else i = GI - 1;
    }
    if (jj < 0) {
        if (BCY0 == BC_PERIODIC) jj += GJ;
        else if (BCY0 == BC_FIXED) return ghost + 2 * NPAD;
        else jj = 0;
    } else if (jj >= GJ) {
        if (BCY1 == BC_PERIODIC) jj -= GJ;
        else if (BCY1 == BC_FIXED) return ghost + 3 * NPAD;
        else jj = GJ - 1;
    }
    return f + ((size_t)jj * GI + i) * NPAD;
}
__device__ __forceinline__ bool beyond_wall_x(int pos) { return (pos < 0 && BCX0 == BC_WALL) || (pos >= GI && BCX1 == BC_WALL); }
__device__ __forceinline__ bool beyond_wall_y(int pos) { return (pos < 0 && BCY0 == BC_WALL) || (pos >= GJ && BCY1 == BC_WALL); }

// shared-memory load at a byte offset from a (warp-uniform) base: LDS R, [Roff + URbase]
__device__ __forceinline__ double ldsd(const unsigned char *base, int off) { return *reinterpret_cast<const double *>(base + off); }
__device__ __forceinline__ double2 ldsd2(const unsigned char *base, int off) { return *reinterpret_cast<const double2 *>(base + off); }

// ---- mbarrier + 1-D TMA bulk copy (cp.async.bulk; SASS UBLKCP) ------------------------------------------------------------
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
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n .reg .pred p;\n WAIT_%=:\n"
                 " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

struct true_c { static constexpr bool value = true; };
struct false_c { static constexpr bool value = false; };

// ---- limiter ----------------------------------------------------------------------------------------------------------
// h*sigma of the van Leer limiter (AMB-4) from un-normalised differences dm = f_c - f_{c-1}, dp = f_{c+1} - f_c:
//   h*sigma = (Delta/2) * 2 (dm/Delta)(dp/Delta)/((dm+dp)/Delta) = dm dp / (dm + dp)   if dm dp > 0, else 0.
// The reciprocal is MUFU.RCP64H (rel. error 2^-23) refined by one cubic step (1 + e + e^2), e = 1 - s r: error e^3 ~ 2^-69,
// applied to the quotient q0 = pr r: hs = q0 (1 + e + e^2) is within ~1 ulp of pr / s.  The sign test reads the high word: a product that underflowed to a denormal counts as 0, as in
// AMB-4's "underflow gives sigma = 0".
__device__ __forceinline__ double vl_half(double dm, double dp)
{
    const double pr = dm * dp, s = dm + dp;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));
    // q0 = pr r0 is formed beside e = 1 - s r0, so the chain after s is MUFU, e, t = e + e^2, q0 (1 + t): four deep, not five.
    // The sign test acts on the seed: its low word is zero by construction (MUFU.RCP64H), so "no slope" is one 32-bit select of
    // the high word; with r0 = 0 the chain gives q0 = 0, e = 1, t = 2, hs = fma(0, 2, 0) = 0 exactly.
    r = __hiloint2double(__double2hiint(pr) > 0 ? __double2hiint(r) : 0, 0);
    const double q0 = pr * r;
    const double e = fma(-s, r, 1.0);
    const double t = fma(e, e, e);
    return fma(q0, t, q0);
}
