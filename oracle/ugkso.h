/* ugkso.h -- CPU ORACLE for the 2-D BGK-UGKS time step (arXiv:1810.08137).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, header, table or helper with the CUDA path (paper_1810_08137_b200/csrc,
 * include/ugks.h); neither includes the other.
 *
 * What it computes follows /root/reference/PAPER.md ("P:Lnn"):
 *   model + Maxwellian      P:L27-32  Eq. (1)
 *   integral face solution  P:L34-37  Eq. (2)
 *   f and W updates         P:L39-46  Eq. (3)(4)
 *   order of sub-steps      P:L76-86  S1..S8
 * The flux construction itself is delegated by the paper to its refs [1,2]
 * (P:L48); the concrete formulas are the readings O0..O12 / AMB-1..22 listed in
 * DESIGN.md ("Readings of the paper").
 *
 * Plain C99, fp64, single-threaded by default (UGKSO_THREADS env / ugkso_set_threads
 * enables OpenMP over rows/columns/cells; per-face and per-cell arithmetic and its
 * order are unchanged, so results are bit-identical to the single-thread run).
 * All pointers are HOST pointers.  Every call returns 0 on success, nonzero on error.
 *
 * Parity pins: tests/test_oracle_*.py (P1..P15, P17..P19 of DESIGN.md; P17..P19 pin the
 * equilibrium-slope bracket of S5/S8 and cell_gradW against the exact Euler solution, the
 * Navier-Stokes shear-wave decay rate and the S5-vs-S8 consistency of every face).  Field
 * values of a full channel step are "parity unpinned" against the paper: PAPER.md prints no
 * flow-field number (only wall-clock times); they are pinned by invariants instead.
 */
#ifndef UGKSO_H
#define UGKSO_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ugkso_ctx ugkso_ctx;

enum { UGKSO_OK = 0, UGKSO_EINVAL = 1, UGKSO_ENOMEM = 2, UGKSO_ESTATE = 4 };
enum { UGKSO_BC_PERIODIC = 0, UGKSO_BC_FIXED = 1, UGKSO_BC_WALL = 2 };

typedef struct { int I, J; double x0, x1, y0, y1; } ugkso_mesh;
typedef struct { int Nu, Nv; const double *u, *wu, *v, *wv; } ugkso_vgrid;
typedef struct { double omega, mu_ref, Kn, Pr; int K_int; } ugkso_gas;
typedef struct { int type; double rho, U, V, T; } ugkso_bc;
typedef struct { ugkso_bc xmin, xmax, ymin, ymax; } ugkso_bcs;

int  ugkso_init(ugkso_ctx **out, const ugkso_mesh *, const ugkso_vgrid *, const ugkso_gas *,
                const ugkso_bcs *, double cfl);
int  ugkso_set_state(ugkso_ctx *, const double *W /*[J][I][4]*/, const double *f /*[J][I][Nv][Nu]*/);
int  ugkso_step(ugkso_ctx *, int n);
int  ugkso_moments(ugkso_ctx *, double *W_stored /*[J][I][4] or NULL*/, double *W_of_f /*or NULL*/);
int  ugkso_get_f(ugkso_ctx *, double *f);
int  ugkso_residual(ugkso_ctx *, double res[4]);
double ugkso_dt(const ugkso_ctx *);
long ugkso_step_count(const ugkso_ctx *);
double ugkso_mu_ref(const ugkso_ctx *);
void ugkso_set_threads(ugkso_ctx *, int nthreads);
/* NEXT-1 (O3t/O8t): 1 = reconstruct f in the tangential direction too (limited slope theta of the upwind cell)
 * and add -Mt5 t theta0 to the free-transport part of the face solution; default 0 (normal-direction reconstruction only). */
void ugkso_set_tangential(ugkso_ctx *, int on);
void ugkso_destroy(ugkso_ctx *);

/* ---- one-by-one access (full-size sampled parity; stage-wise debugging) ---- */

/* Time-integrated flux through one face from the CURRENT state (O2..O9).
 * dir 0: x-face between cells (i-1,j) and (i,j), i in [0,I];  dir 1: y-face between
 * (i,j-1) and (i,j), j in [0,J].  FW[4] and Ff[Nv*Nu] are signed along +x / +y.
 * stage (may be NULL) receives 40 doubles:
 *   [0..3] W0 (local frame)  [4..7] prim0  [8..11] a_L  [12..15] a_R  [16..19] b
 *   [20..23] A  [24..28] Mt1..Mt5  [29] tau0  [30..33] F_g  [34..37] F_f^W  [38] rho_w (walls) */
int  ugkso_face_flux(ugkso_ctx *, int dir, int i, int j, double FW[4], double *Ff, double *stage);

/* One cell of O10 from the CURRENT state: W^{n+1}[4] and f^{n+1}[Nv*Nu] of cell (i,j). */
int  ugkso_cell_update(ugkso_ctx *, int i, int j, double Wnew[4], double *fnew);

/* ---- closed-form pieces exposed for the pin tests (no state) ---- */
void ugkso_prim_of_W(const double W[4], double prim[4]);
void ugkso_W_of_prim(const double prim[4], double W[4]);
double ugkso_maxwellian(const double prim[4], double u, double v);
/* O4: ML[7], MR[7], Mu[7] (normal, half/half/full range), Mv[7] (tangential) of M[prim]. */
void ugkso_gauss_moments(const double prim[4], double ML[7], double MR[7], double Mu[7], double Mv[7]);
/* O4: T_X[c](alpha,beta) with X = 0:Mu 1:ML 2:MR ; c may be NULL meaning "m(alpha,beta)" itself. */
void ugkso_moment_T(const double prim[4], int X, const double *c, int alpha, int beta, double out[4]);
/* O6: micro-slope c with rho <psi (c.psi)> = s. */
void ugkso_micro_slope(const double prim[4], const double s[4], double c[4]);
/* O5: Mt[5] = Mt1..Mt5 for given dt, tau. */
void ugkso_time_coeffs(double dt, double tau, double Mt[5]);
/* AMB-4: van Leer limiter. */
double ugkso_van_leer(double sm, double sp);
/* AMB-7: tau(rho, lambda) and mu_ref from Kn. */
double ugkso_tau(double mu_ref, double omega, double rho, double lambda);
double ugkso_mu_ref_from_kn(double Kn, double omega);

#ifdef __cplusplus
}
#endif
#endif
