/* ugkso.c -- CPU ORACLE for the 2-D BGK-UGKS time step.  See ugkso.h for the role of
 * this file (test infrastructure; shares nothing with the CUDA path).
 *
 * Every function cites the passage of /root/reference/PAPER.md ("P:Lnn") it follows and
 * the reading (O0..O12, AMB-n of DESIGN.md) that fills in what the paper delegates to
 * its refs [1,2].  The arithmetic is the direct formula in the paper's order:
 * no separable-exponential trick, no tables, no blocking or fusion.  Velocity-space sums
 * run in index order q = m*Nu + k = 0..N-1 with Neumaier compensation.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC ugkso.c -o libugkso.so -lm
 */
#include "ugkso.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------ */
/* compensated sum (Neumaier), used for every velocity-space sum       */
typedef struct { double s, c; } ksum;
static void ks_add(ksum *k, double x)
{
    double t = k->s + x;
    if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x;
    else                       k->c += (x - t) + k->s;
    k->s = t;
}
static double ks_val(const ksum *k) { return k->s + k->c; }

/* ------------------------------------------------------------------ */
/* P:L29 Eq. (1) with lambda = m/(2kT); K_int = 0 (AMB-2): gamma = 2,  */
/* rhoE = rho(U^2+V^2)/2 + rho/(2 lambda).                             */
void ugkso_prim_of_W(const double W[4], double prim[4])
{
    double rho = W[0], U = W[1] / rho, V = W[2] / rho;
    prim[0] = rho; prim[1] = U; prim[2] = V;
    prim[3] = rho / (2.0 * (W[3] - 0.5 * rho * (U * U + V * V)));
}
void ugkso_W_of_prim(const double prim[4], double W[4])
{
    double rho = prim[0], U = prim[1], V = prim[2], lam = prim[3];
    W[0] = rho; W[1] = rho * U; W[2] = rho * V;
    W[3] = 0.5 * rho * (U * U + V * V) + rho / (2.0 * lam);
}
/* P:L29 Eq. (1): g = rho (lambda/pi) exp(-lambda((u-U)^2+(v-V)^2)). */
double ugkso_maxwellian(const double prim[4], double u, double v)
{
    double du = u - prim[1], dv = v - prim[2];
    return prim[0] * (prim[3] / PI) * exp(-prim[3] * (du * du + dv * dv));
}
/* AMB-7: tau = mu/p, mu = mu_ref T^omega, p = rho/(2 lambda), T = 1/lambda. */
double ugkso_tau(double mu_ref, double omega, double rho, double lambda)
{
    return 2.0 * mu_ref * pow(lambda, 1.0 - omega) / rho;
}
/* AMB-7: variable-hard-sphere mean free path, alpha = 1. */
double ugkso_mu_ref_from_kn(double Kn, double omega)
{
    double alpha = 1.0;
    return 5.0 * (alpha + 1.0) * (alpha + 2.0) * sqrt(PI)
         / (4.0 * alpha * (5.0 - 2.0 * omega) * (7.0 - 2.0 * omega)) * Kn;
}
/* AMB-4: van Leer limiter, no epsilon. */
double ugkso_van_leer(double sm, double sp)
{
    double p = sm * sp;
    if (!(p > 0.0)) return 0.0;
    return 2.0 * p / (sm + sp);
}

/* ------------------------------------------------------------------ */
/* O4 (S2): moments <n^p> of the Maxwellian, half and full   */
/* range in the normal velocity, full range in the tangential one.     */
void ugkso_gauss_moments(const double prim[4], double ML[7], double MR[7], double Mu[7], double Mv[7])
{
    double U = prim[1], V = prim[2], lam = prim[3];
    double sl = sqrt(lam);
    double e = 0.5 * exp(-lam * U * U) / sqrt(PI * lam);
    ML[0] = 0.5 * erfc(-sl * U);  ML[1] = U * ML[0] + e;
    MR[0] = 0.5 * erfc( sl * U);  MR[1] = U * MR[0] - e;
    for (int p = 0; p <= 4; ++p) {
        ML[p + 2] = U * ML[p + 1] + (p + 1) / (2.0 * lam) * ML[p];
        MR[p + 2] = U * MR[p + 1] + (p + 1) / (2.0 * lam) * MR[p];
    }
    for (int p = 0; p < 7; ++p) Mu[p] = ML[p] + MR[p];
    Mv[0] = 1.0; Mv[1] = V;
    for (int p = 0; p <= 4; ++p) Mv[p + 2] = V * Mv[p + 1] + (p + 1) / (2.0 * lam) * Mv[p];
}
/* m(alpha,beta) = <n^alpha t^beta psi> over the range of X; Mxi = (1,0,0) for K_int=0. */
static void mom_m(const double *X, const double *Mv, int a, int b, double out[4])
{
    const double Mxi1 = 0.0;
    out[0] = X[a] * Mv[b];
    out[1] = X[a + 1] * Mv[b];
    out[2] = X[a] * Mv[b + 1];
    out[3] = 0.5 * (X[a + 2] * Mv[b] + X[a] * Mv[b + 2] + X[a] * Mv[b] * Mxi1);
}
/* T_X[c](alpha,beta) = <n^alpha t^beta psi (c.psi)>, c.psi = c1 + c2 n + c3 t + c4 (n^2+t^2)/2. */
static void mom_T(const double *X, const double *Mv, const double c[4], int a, int b, double out[4])
{
    double m0[4], m1[4], m2[4], m3[4], m4[4];
    mom_m(X, Mv, a, b, m0);
    mom_m(X, Mv, a + 1, b, m1);
    mom_m(X, Mv, a, b + 1, m2);
    mom_m(X, Mv, a + 2, b, m3);
    mom_m(X, Mv, a, b + 2, m4);
    for (int r = 0; r < 4; ++r)   /* m_xi = 0 for K_int = 0 */
        out[r] = c[0] * m0[r] + c[1] * m1[r] + c[2] * m2[r] + 0.5 * c[3] * (m3[r] + m4[r] + 0.0);
}
void ugkso_moment_T(const double prim[4], int Xsel, const double *c, int a, int b, double out[4])
{
    /* note: needs a+4 <= 8 only through X[a+2] of m(a+2,b); callers use a<=2, b<=1 */
    double ML[9], MR[9], Mu[9], Mv[9];
    double U = prim[1], V = prim[2], lam = prim[3];
    ugkso_gauss_moments(prim, ML, MR, Mu, Mv);
    for (int p = 5; p <= 6; ++p) {           /* two more orders so that any a,b <= 2 is safe */
        ML[p + 2] = U * ML[p + 1] + (p + 1) / (2.0 * lam) * ML[p];
        MR[p + 2] = U * MR[p + 1] + (p + 1) / (2.0 * lam) * MR[p];
        Mu[p + 2] = ML[p + 2] + MR[p + 2];
        Mv[p + 2] = V * Mv[p + 1] + (p + 1) / (2.0 * lam) * Mv[p];
    }
    const double *X = Xsel == 1 ? ML : Xsel == 2 ? MR : Mu;
    if (c) mom_T(X, Mv, c, a, b, out); else mom_m(X, Mv, a, b, out);
}
/* O6 (S4): micro-slope c with rho <psi (c.psi)> = s. */
void ugkso_micro_slope(const double prim[4], const double s[4], double c[4])
{
    double rho = prim[0], U = prim[1], V = prim[2], lam = prim[3];
    c[3] = (2.0 * lam * lam / rho) * (2.0 * s[3] - 2.0 * U * s[1] - 2.0 * V * s[2]
                                      + s[0] * (U * U + V * V - 1.0 / lam));
    c[2] = (2.0 * lam / rho) * (s[2] - V * s[0]) - V * c[3];
    c[1] = (2.0 * lam / rho) * (s[1] - U * s[0]) - U * c[3];
    c[0] = s[0] / rho - U * c[1] - V * c[2] - 0.5 * (U * U + V * V + 1.0 / lam) * c[3];
}
/* O5 (S3): time integrals over [0,dt] of the integral solution Eq. (2).
 * Mt1: weight of g0; Mt2: of (a n + b t) g0; Mt3: of A g0; Mt4: of f0; Mt5: of -n sigma0. AMB-11. */
void ugkso_time_coeffs(double dt, double tau, double Mt[5])
{
    double x = dt / tau;
    if (x >= 1e-3) {
        double em = -expm1(-x), E = 1.0 - em;
        Mt[3] = tau * em;
        Mt[4] = tau * (Mt[3] - dt * E);
        Mt[0] = dt - Mt[3];
        Mt[1] = -tau * Mt[0] + Mt[4];
        Mt[2] = 0.5 * dt * dt - tau * Mt[0];
    } else {
        double x2 = x * x, x3 = x2 * x, x4 = x3 * x, d2 = dt * dt;
        Mt[3] = dt * (1.0 - x / 2.0 + x2 / 6.0 - x3 / 24.0 + x4 / 120.0);
        Mt[0] = dt * (x / 2.0 - x2 / 6.0 + x3 / 24.0 - x4 / 120.0);
        Mt[4] = d2 * (0.5 - x / 3.0 + x2 / 8.0 - x3 / 30.0 + x4 / 144.0);
        Mt[2] = d2 * (x / 6.0 - x2 / 24.0 + x3 / 120.0 - x4 / 720.0);
        Mt[1] = d2 * (-x / 6.0 + x2 / 12.0 - x3 / 40.0 + x4 / 180.0);
    }
}

/* ------------------------------------------------------------------ */
struct ugkso_ctx {
    int I, J, Nu, Nv, N;
    double dx, dy, dt, omega, mu_ref;
    ugkso_bc bc[4];                 /* 0 xmin, 1 xmax, 2 ymin, 3 ymax */
    double *u, *wu, *v, *wv;        /* 1-D nodes and weights */
    double *fb[4], Wb[4][4];        /* FIXED ghost rows and their W  (O0) */
    double *gw[4];                  /* WALL: Maxwellian of (1,Uw,Vw,1/Tw) (O0) */
    double *f, *D;                  /* state f[J][I][N]; flux-divergence accumulator */
    double *W, *Wn, *FWd;           /* W^n, W^{n+1}, accumulated macroscopic flux [J][I][4] */
    double res[4];
    long steps; int have_state, have_res, nthreads;
    int tangential;                 /* O3t/O8t (NEXT-1): tangential slope theta of f in the free-transport part; default 0 */
};

enum { K_CELL = 0, K_GHOST = 1, K_WALL = 2 };

/* O1 neighbour lookup: PERIODIC wraps; FIXED returns the ghost at any depth; WALL = missing. */
static int lookup(const ugkso_ctx *c, int i, int j, const double **frow, const double **Wrow)
{
    int side = -1;
    if (i < 0)          { if (c->bc[0].type == UGKSO_BC_PERIODIC) i += c->I; else side = 0; }
    else if (i >= c->I) { if (c->bc[1].type == UGKSO_BC_PERIODIC) i -= c->I; else side = 1; }
    if (side < 0) {
        if (j < 0)          { if (c->bc[2].type == UGKSO_BC_PERIODIC) j += c->J; else side = 2; }
        else if (j >= c->J) { if (c->bc[3].type == UGKSO_BC_PERIODIC) j -= c->J; else side = 3; }
    }
    if (side >= 0) {
        if (c->bc[side].type == UGKSO_BC_WALL) { *frow = NULL; *Wrow = NULL; return K_WALL; }
        *frow = c->fb[side]; *Wrow = c->Wb[side]; return K_GHOST;
    }
    size_t cell = (size_t)j * c->I + i;
    *frow = c->f + cell * c->N; *Wrow = c->W + cell * 4;
    return K_CELL;
}

/* O1: limited slope of f in direction dir (0:x, 1:y) at cell (i,j), all velocity points. */
static void cell_slope(const ugkso_ctx *c, int dir, int i, int j, double *sig)
{
    const double *f0, *fm, *fp, *Wd;
    int k0 = lookup(c, i, j, &f0, &Wd);
    if (k0 != K_CELL) { for (int q = 0; q < c->N; ++q) sig[q] = 0.0; return; }   /* ghost rows: sigma = 0 */
    int km = lookup(c, i - (dir == 0), j - (dir == 1), &fm, &Wd);
    int kp = lookup(c, i + (dir == 0), j + (dir == 1), &fp, &Wd);
    double D = dir == 0 ? c->dx : c->dy;
    for (int q = 0; q < c->N; ++q) {
        double sm = km != K_WALL ? (f0[q] - fm[q]) / D : 0.0;
        double sp = kp != K_WALL ? (fp[q] - f0[q]) / D : 0.0;
        if (km != K_WALL && kp != K_WALL) sig[q] = ugkso_van_leer(sm, sp);
        else if (km == K_WALL && kp != K_WALL) sig[q] = sp;                    /* AMB-13 */
        else if (kp == K_WALL && km != K_WALL) sig[q] = sm;
        else sig[q] = 0.0;
    }
}

/* O1 / AMB-14: unlimited gradient of W in direction dir at cell (i,j); 0 for a ghost. */
static void cell_gradW(const ugkso_ctx *c, int dir, int i, int j, double g[4])
{
    const double *fd, *W0, *Wm, *Wp;
    int k0 = lookup(c, i, j, &fd, &W0);
    for (int r = 0; r < 4; ++r) g[r] = 0.0;
    if (k0 != K_CELL) return;
    int km = lookup(c, i - (dir == 0), j - (dir == 1), &fd, &Wm);
    int kp = lookup(c, i + (dir == 0), j + (dir == 1), &fd, &Wp);
    double D = dir == 0 ? c->dx : c->dy;
    for (int r = 0; r < 4; ++r) {
        if (km != K_WALL && kp != K_WALL) g[r] = (Wp[r] - Wm[r]) / (2.0 * D);
        else if (km == K_WALL && kp != K_WALL) g[r] = (Wp[r] - W0[r]) / D;
        else if (kp == K_WALL && km != K_WALL) g[r] = (W0[r] - Wm[r]) / D;
    }
}

static void swap12(double w[4]) { double t = w[1]; w[1] = w[2]; w[2] = t; }

/* O9 (BW): diffuse isothermal wall face.  (ci,cj) is the fluid cell, side the wall's side. */
static void wall_face(const ugkso_ctx *c, int side, int ci, int cj, double FW[4], double *Ff,
                      double *scratch, double *stage)
{
    int N = c->N, Nu = c->Nu, dir = side >= 2;
    double sgn = (side == 1 || side == 3) ? 1.0 : -1.0;        /* n_out = sgn * e_dir */
    double h = 0.5 * (dir == 0 ? c->dx : c->dy), ell = dir == 0 ? c->dy : c->dx;
    const double *fc, *Wd, *gw = c->gw[side];
    lookup(c, ci, cj, &fc, &Wd);
    double *sig = scratch;
    cell_slope(c, dir, ci, cj, sig);
    ksum num = {0, 0}, den = {0, 0};
    for (int q = 0; q < N; ++q) {
        int k = q % Nu, m = q / Nu;
        double w = c->wu[k] * c->wv[m];
        double vn = sgn * (dir == 0 ? c->u[k] : c->v[m]);
        double H = vn > 0.0 ? 1.0 : (vn < 0.0 ? 0.0 : 0.5);
        double fface = fc[q] + (sgn * h) * sig[q];
        ks_add(&num, w * vn * fface * H);
        ks_add(&den, w * vn * gw[q] * (1.0 - H));
    }
    double rho_w = -ks_val(&num) / ks_val(&den);
    ksum FWs[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
    for (int q = 0; q < N; ++q) {
        int k = q % Nu, m = q / Nu;
        double u = c->u[k], v = c->v[m], w = c->wu[k] * c->wv[m];
        double vn = sgn * (dir == 0 ? u : v);
        double H = vn > 0.0 ? 1.0 : (vn < 0.0 ? 0.0 : 0.5);
        double fface = fc[q] + (sgn * h) * sig[q];
        double fw = H * fface + (1.0 - H) * rho_w * gw[q];
        double Fq = ell * c->dt * vn * fw;                      /* along n_out */
        Fq *= sgn;                                              /* signed along +x / +y */
        Ff[q] = Fq;
        ks_add(&FWs[0], w * Fq);
        ks_add(&FWs[1], w * u * Fq);
        ks_add(&FWs[2], w * v * Fq);
        ks_add(&FWs[3], w * 0.5 * (u * u + v * v) * Fq);
    }
    for (int r = 0; r < 4; ++r) FW[r] = ks_val(&FWs[r]);
    if (stage) { memset(stage, 0, 40 * sizeof(double)); stage[38] = rho_w; }
}

/* O2..O8: flux through one face.  scratch: 7*N doubles. */
static int face_flux(const ugkso_ctx *c, int dir, int i, int j, double FW[4], double *Ff,
                     double *scratch, double *stage)
{
    int N = c->N, Nu = c->Nu;
    int iL = i - (dir == 0), jL = j - (dir == 1), iR = i, jR = j;
    const double *fL, *fR, *WL, *WR;
    int kL = lookup(c, iL, jL, &fL, &WL), kR = lookup(c, iR, jR, &fR, &WR);
    if (kL == K_WALL && kR == K_WALL) return UGKSO_EINVAL;
    if (kL == K_WALL) { wall_face(c, dir == 0 ? 0 : 2, iR, jR, FW, Ff, scratch, stage); return 0; }
    if (kR == K_WALL) { wall_face(c, dir == 0 ? 1 : 3, iL, jL, FW, Ff, scratch, stage); return 0; }

    double h = 0.5 * (dir == 0 ? c->dx : c->dy), ell = dir == 0 ? c->dy : c->dx, dt = c->dt;
    double *sigL = scratch, *sigR = scratch + N, *f0 = scratch + 2 * N, *s0 = scratch + 3 * N;
    double *thL = scratch + 5 * N, *thR = scratch + 6 * N;          /* (scratch + 4N is used by wall_face) */
    cell_slope(c, dir, iL, jL, sigL);
    cell_slope(c, dir, iR, jR, sigR);
    if (c->tangential) {
        /* O3t (NEXT-1; "b (tangential)", ref [2]): the initial state is reconstructed in BOTH directions,
         * f0(x,y) = f0 + sigma0 x + theta0 y on the upwind side, theta = the limited slope (O1) of the upwind cell in the
         * TANGENTIAL direction.  At the face centre (y = 0) f0 and W0 are unchanged; free transport along the
         * characteristic (x, y) = (-n t', -t t') adds -t t' theta0 under the time integral of Eq. (2). */
        cell_slope(c, 1 - dir, iL, jL, thL);
        cell_slope(c, 1 - dir, iR, jR, thR);
    }

    /* O3 (S0/S1): upwind reconstruction at the face and its moments W0 */
    ksum W0s[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
    for (int q = 0; q < N; ++q) {
        int k = q % Nu, m = q / Nu;
        double n = dir == 0 ? c->u[k] : c->v[m], t = dir == 0 ? c->v[m] : c->u[k];
        double w = c->wu[k] * c->wv[m];
        double H = n > 0.0 ? 1.0 : (n < 0.0 ? 0.0 : 0.5);                     /* AMB-5 */
        f0[q] = H * (fL[q] + h * sigL[q]) + (1.0 - H) * (fR[q] - h * sigR[q]);
        s0[q] = H * sigL[q] + (1.0 - H) * sigR[q];
        ks_add(&W0s[0], w * f0[q]);
        ks_add(&W0s[1], w * n * f0[q]);
        ks_add(&W0s[2], w * t * f0[q]);
        ks_add(&W0s[3], w * 0.5 * (n * n + t * t) * f0[q]);
    }
    double W0[4], prim0[4];
    for (int r = 0; r < 4; ++r) W0[r] = ks_val(&W0s[r]);
    ugkso_prim_of_W(W0, prim0);
    if (!(prim0[0] > 0.0) || !(prim0[3] > 0.0)) return UGKSO_ESTATE;
    double rho0 = prim0[0];

    /* O4 (S2) */
    double ML[7], MR[7], Mu[7], Mv[7];
    ugkso_gauss_moments(prim0, ML, MR, Mu, Mv);
    /* O5 (S3) */
    double tau0 = ugkso_tau(c->mu_ref, c->omega, prim0[0], prim0[3]), Mt[5];
    ugkso_time_coeffs(dt, tau0, Mt);

    /* O6 (S4): micro-slopes from the stored cell averages W^n (AMB-8) */
    double wl[4], wr[4], sL[4], sR[4], sb[4], gL[4], gR[4], aL[4], aR[4], b[4], A[4];
    memcpy(wl, WL, sizeof wl); memcpy(wr, WR, sizeof wr);
    cell_gradW(c, 1 - dir, iL, jL, gL);
    cell_gradW(c, 1 - dir, iR, jR, gR);
    if (dir == 1) { swap12(wl); swap12(wr); swap12(gL); swap12(gR); }        /* P (AMB-21) */
    for (int r = 0; r < 4; ++r) {
        sL[r] = (W0[r] - wl[r]) / h;
        sR[r] = (wr[r] - W0[r]) / h;
        sb[r] = 0.5 * (gL[r] + gR[r]);
    }
    ugkso_micro_slope(prim0, sL, aL);
    ugkso_micro_slope(prim0, sR, aR);
    ugkso_micro_slope(prim0, sb, b);
    double t1[4], t2[4], t3[4], sA[4];
    mom_T(ML, Mv, aL, 1, 0, t1); mom_T(MR, Mv, aR, 1, 0, t2); mom_T(Mu, Mv, b, 0, 1, t3);
    for (int r = 0; r < 4; ++r) sA[r] = -rho0 * (t1[r] + t2[r] + t3[r]);     /* AMB-20 */
    ugkso_micro_slope(prim0, sA, A);

    /* O7 (S5): hydrodynamic part of the macroscopic flux, analytic (AMB-9) */
    double Fg[4], m10[4], t4[4];
    mom_m(Mu, Mv, 1, 0, m10);
    mom_T(ML, Mv, aL, 2, 0, t1); mom_T(MR, Mv, aR, 2, 0, t2); mom_T(Mu, Mv, b, 1, 1, t3);
    mom_T(Mu, Mv, A, 1, 0, t4);
    for (int r = 0; r < 4; ++r)
        Fg[r] = rho0 * (Mt[0] * m10[r] + Mt[1] * (t1[r] + t2[r] + t3[r]) + Mt[2] * t4[r]);

    /* O8 (S6/S7/S8) */
    ksum Ffs[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
    for (int q = 0; q < N; ++q) {
        int k = q % Nu, m = q / Nu;
        double n = dir == 0 ? c->u[k] : c->v[m], t = dir == 0 ? c->v[m] : c->u[k];
        double w = c->wu[k] * c->wv[m];
        double H = n > 0.0 ? 1.0 : (n < 0.0 ? 0.0 : 0.5);
        double e = 0.5 * (n * n + t * t);
        double g0 = ugkso_maxwellian(prim0, n, t);
        double r = Mt[3] * f0[q] - Mt[4] * n * s0[q];
        if (c->tangential)                                                    /* O8t: ... - Mt5 t theta0, theta0 upwind */
            r -= Mt[4] * t * (H * thL[q] + (1.0 - H) * thR[q]);
        ks_add(&Ffs[0], w * n * r);
        ks_add(&Ffs[1], w * n * n * r);
        ks_add(&Ffs[2], w * n * t * r);
        ks_add(&Ffs[3], w * n * e * r);
        double aLp = aL[0] + aL[1] * n + aL[2] * t + aL[3] * e;
        double aRp = aR[0] + aR[1] * n + aR[2] * t + aR[3] * e;
        double bp  = b[0] + b[1] * n + b[2] * t + b[3] * e;
        double Ap  = A[0] + A[1] * n + A[2] * t + A[3] * e;
        Ff[q] = ell * n * ((Mt[0] + Mt[1] * (n * (H * aLp + (1.0 - H) * aRp) + t * bp) + Mt[2] * Ap) * g0 + r);
    }
    double FfW[4];
    for (int r = 0; r < 4; ++r) { FfW[r] = ks_val(&Ffs[r]); FW[r] = ell * (Fg[r] + FfW[r]); }
    if (dir == 1) swap12(FW);
    if (stage) {
        memcpy(stage, W0, 32); memcpy(stage + 4, prim0, 32); memcpy(stage + 8, aL, 32);
        memcpy(stage + 12, aR, 32); memcpy(stage + 16, b, 32); memcpy(stage + 20, A, 32);
        memcpy(stage + 24, Mt, 40); stage[29] = tau0; memcpy(stage + 30, Fg, 32);
        memcpy(stage + 34, FfW, 32); stage[38] = 0.0; stage[39] = 0.0;
    }
    return 0;
}

/* O10 (U2/U3, Eq. (3)): implicit BGK relaxation of one cell given its flux divergence
 * Dq = F^{x,i-1/2} - F^{x,i+1/2} + F^{y,j-1/2} - F^{y,j+1/2}; in-place safe (fout may equal fin). */
static int relax_cell(const ugkso_ctx *c, const double Wn[4], const double Wnew[4],
                      const double *fin, const double *Dq, double *fout)
{
    double pn[4], pp[4];
    ugkso_prim_of_W(Wn, pn); ugkso_prim_of_W(Wnew, pp);
    if (!(pp[0] > 0.0) || !(pp[3] > 0.0)) return UGKSO_ESTATE;
    double taun = ugkso_tau(c->mu_ref, c->omega, pn[0], pn[3]);
    double taup = ugkso_tau(c->mu_ref, c->omega, pp[0], pp[3]);
    double Om = c->dx * c->dy, dt = c->dt;
    for (int q = 0; q < c->N; ++q) {
        double u = c->u[q % c->Nu], v = c->v[q / c->Nu];
        double gn = ugkso_maxwellian(pn, u, v), gp = ugkso_maxwellian(pp, u, v);
        fout[q] = (fin[q] + Dq[q] / Om + 0.5 * dt * (gp / taup + (gn - fin[q]) / taun))
                / (1.0 + 0.5 * dt / taup);
    }
    return 0;
}

/* ------------------------------------------------------------------ */
static void free_ctx(ugkso_ctx *c)
{
    if (!c) return;
    free(c->u); free(c->wu); free(c->v); free(c->wv);
    for (int s = 0; s < 4; ++s) { free(c->fb[s]); free(c->gw[s]); }
    free(c->f); free(c->D); free(c->W); free(c->Wn); free(c->FWd);
    free(c);
}
static double *dupd(const double *p, int n)
{
    double *r = (double *)malloc(sizeof(double) * (size_t)n);
    if (r) memcpy(r, p, sizeof(double) * (size_t)n);
    return r;
}

/* O0: setup.  dt = CFL / (max|u|/dx + max|v|/dy) (AMB-6); ghost rows; wall Maxwellians. */
int ugkso_init(ugkso_ctx **out, const ugkso_mesh *m, const ugkso_vgrid *vg, const ugkso_gas *gas,
               const ugkso_bcs *bcs, double cfl)
{
    if (!out || !m || !vg || !gas || !bcs) return UGKSO_EINVAL;
    *out = NULL;
    if (m->I < 2 || m->J < 2 || !(m->x1 > m->x0) || !(m->y1 > m->y0)) return UGKSO_EINVAL;
    if (vg->Nu < 1 || vg->Nv < 1 || !vg->u || !vg->wu || !vg->v || !vg->wv) return UGKSO_EINVAL;
    if (gas->Pr != 1.0 || gas->K_int != 0 || !(cfl > 0.0)) return UGKSO_EINVAL;
    const ugkso_bc *b[4] = { &bcs->xmin, &bcs->xmax, &bcs->ymin, &bcs->ymax };
    for (int s = 0; s < 4; ++s) {
        if (b[s]->type < 0 || b[s]->type > 2) return UGKSO_EINVAL;
        if (b[s]->type != UGKSO_BC_PERIODIC && !(b[s]->T > 0.0)) return UGKSO_EINVAL;
        if (b[s]->type == UGKSO_BC_FIXED && !(b[s]->rho > 0.0)) return UGKSO_EINVAL;
    }
    if ((b[0]->type == UGKSO_BC_PERIODIC) != (b[1]->type == UGKSO_BC_PERIODIC)) return UGKSO_EINVAL;
    if ((b[2]->type == UGKSO_BC_PERIODIC) != (b[3]->type == UGKSO_BC_PERIODIC)) return UGKSO_EINVAL;
    double swu = 0, swv = 0, umax = 0, vmax = 0;
    for (int k = 0; k < vg->Nu; ++k) { swu += vg->wu[k]; if (fabs(vg->u[k]) > umax) umax = fabs(vg->u[k]); }
    for (int k = 0; k < vg->Nv; ++k) { swv += vg->wv[k]; if (fabs(vg->v[k]) > vmax) vmax = fabs(vg->v[k]); }
    if (!(swu > 0.0) || !(swv > 0.0) || !(umax + vmax > 0.0)) return UGKSO_EINVAL;

    ugkso_ctx *c = (ugkso_ctx *)calloc(1, sizeof *c);
    if (!c) return UGKSO_ENOMEM;
    c->I = m->I; c->J = m->J; c->Nu = vg->Nu; c->Nv = vg->Nv; c->N = vg->Nu * vg->Nv;
    c->dx = (m->x1 - m->x0) / m->I; c->dy = (m->y1 - m->y0) / m->J;
    c->omega = gas->omega;
    c->mu_ref = gas->mu_ref > 0.0 ? gas->mu_ref : ugkso_mu_ref_from_kn(gas->Kn, gas->omega);
    if (!(c->mu_ref > 0.0)) { free(c); return UGKSO_EINVAL; }
    c->dt = cfl / (umax / c->dx + vmax / c->dy);
    c->nthreads = 1;
    const char *env = getenv("UGKSO_THREADS");
    if (env && atoi(env) > 0) c->nthreads = atoi(env);
    c->u = dupd(vg->u, c->Nu); c->wu = dupd(vg->wu, c->Nu);
    c->v = dupd(vg->v, c->Nv); c->wv = dupd(vg->wv, c->Nv);
    size_t cells = (size_t)c->I * c->J;
    c->f = (double *)malloc(sizeof(double) * cells * c->N);
    c->D = (double *)malloc(sizeof(double) * cells * c->N);
    c->W = (double *)malloc(sizeof(double) * cells * 4);
    c->Wn = (double *)malloc(sizeof(double) * cells * 4);
    c->FWd = (double *)malloc(sizeof(double) * cells * 4);
    int ok = c->u && c->wu && c->v && c->wv && c->f && c->D && c->W && c->Wn && c->FWd;
    for (int s = 0; s < 4 && ok; ++s) {
        c->bc[s] = *b[s];
        if (b[s]->type == UGKSO_BC_PERIODIC) continue;
        double prim[4] = { b[s]->type == UGKSO_BC_FIXED ? b[s]->rho : 1.0, b[s]->U, b[s]->V, 1.0 / b[s]->T };
        double *row = (double *)malloc(sizeof(double) * c->N);
        if (!row) { ok = 0; break; }
        for (int q = 0; q < c->N; ++q)
            row[q] = ugkso_maxwellian(prim, c->u[q % c->Nu], c->v[q / c->Nu]);
        if (b[s]->type == UGKSO_BC_FIXED) { c->fb[s] = row; ugkso_W_of_prim(prim, c->Wb[s]); }
        else c->gw[s] = row;
    }
    if (!ok) { free_ctx(c); return UGKSO_ENOMEM; }
    *out = c;
    return UGKSO_OK;
}

void ugkso_destroy(ugkso_ctx *c) { free_ctx(c); }
void ugkso_set_threads(ugkso_ctx *c, int n) { if (c && n > 0) c->nthreads = n; }
void ugkso_set_tangential(ugkso_ctx *c, int on) { if (c) c->tangential = on != 0; }
double ugkso_dt(const ugkso_ctx *c) { return c ? c->dt : 0.0; }
long ugkso_step_count(const ugkso_ctx *c) { return c ? c->steps : -1; }
double ugkso_mu_ref(const ugkso_ctx *c) { return c ? c->mu_ref : 0.0; }

int ugkso_set_state(ugkso_ctx *c, const double *W, const double *f)
{
    if (!c || !W || !f) return UGKSO_EINVAL;
    size_t cells = (size_t)c->I * c->J;
    memcpy(c->W, W, sizeof(double) * cells * 4);
    memcpy(c->f, f, sizeof(double) * cells * c->N);
    c->have_state = 1; c->have_res = 0; c->steps = 0;
    return UGKSO_OK;
}
int ugkso_get_f(ugkso_ctx *c, double *f)
{
    if (!c || !f) return UGKSO_EINVAL;
    if (!c->have_state) return UGKSO_ESTATE;
    memcpy(f, c->f, sizeof(double) * (size_t)c->I * c->J * c->N);
    return UGKSO_OK;
}

/* O12 (MOM): W_of_f[c] = sum_q w_q psi_q f[c][q]. */
int ugkso_moments(ugkso_ctx *c, double *W_stored, double *W_of_f)
{
    if (!c) return UGKSO_EINVAL;
    if (!c->have_state) return UGKSO_ESTATE;
    size_t cells = (size_t)c->I * c->J;
    if (W_stored) memcpy(W_stored, c->W, sizeof(double) * cells * 4);
    if (W_of_f) {
        for (size_t cell = 0; cell < cells; ++cell) {
            const double *fr = c->f + cell * c->N;
            ksum s[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
            for (int q = 0; q < c->N; ++q) {
                double u = c->u[q % c->Nu], v = c->v[q / c->Nu], w = c->wu[q % c->Nu] * c->wv[q / c->Nu];
                ks_add(&s[0], w * fr[q]);
                ks_add(&s[1], w * u * fr[q]);
                ks_add(&s[2], w * v * fr[q]);
                ks_add(&s[3], w * 0.5 * (u * u + v * v) * fr[q]);
            }
            for (int r = 0; r < 4; ++r) W_of_f[cell * 4 + r] = ks_val(&s[r]);
        }
    }
    return UGKSO_OK;
}

int ugkso_face_flux(ugkso_ctx *c, int dir, int i, int j, double FW[4], double *Ff, double *stage)
{
    if (!c || !FW || !Ff || dir < 0 || dir > 1) return UGKSO_EINVAL;
    if (!c->have_state) return UGKSO_ESTATE;
    if (dir == 0 && (i < 0 || i > c->I || j < 0 || j >= c->J)) return UGKSO_EINVAL;
    if (dir == 1 && (i < 0 || i >= c->I || j < 0 || j > c->J)) return UGKSO_EINVAL;
    double *scratch = (double *)malloc(sizeof(double) * 7 * (size_t)c->N);
    if (!scratch) return UGKSO_ENOMEM;
    int rc = face_flux(c, dir, i, j, FW, Ff, scratch, stage);
    free(scratch);
    return rc;
}

/* O10 for one cell from the current state (Jacobi: everything from f^n, W^n). */
int ugkso_cell_update(ugkso_ctx *c, int i, int j, double Wnew[4], double *fnew)
{
    if (!c || !Wnew || !fnew || i < 0 || i >= c->I || j < 0 || j >= c->J) return UGKSO_EINVAL;
    if (!c->have_state) return UGKSO_ESTATE;
    int N = c->N;
    double *buf = (double *)malloc(sizeof(double) * 9 * (size_t)N);
    if (!buf) return UGKSO_ENOMEM;
    double *Ff = buf, *Dq = buf + N, *scratch = buf + 2 * N, FW[4], FWd[4] = {0, 0, 0, 0};
    int rc = 0;
    for (int q = 0; q < N; ++q) Dq[q] = 0.0;
    for (int face = 0; face < 4 && !rc; ++face) {
        int dir = face >> 1, plus = face & 1;
        rc = face_flux(c, dir, i + (dir == 0 && plus), j + (dir == 1 && plus), FW, Ff, scratch, NULL);
        double sg = plus ? -1.0 : 1.0;
        for (int q = 0; q < N; ++q) Dq[q] += sg * Ff[q];
        for (int r = 0; r < 4; ++r) FWd[r] += sg * FW[r];
    }
    if (!rc) {
        size_t cell = (size_t)j * c->I + i;
        double Om = c->dx * c->dy;
        for (int r = 0; r < 4; ++r) Wnew[r] = c->W[cell * 4 + r] + FWd[r] / Om;     /* P:L45 Eq. (4) */
        rc = relax_cell(c, c->W + cell * 4, Wnew, c->f + cell * N, Dq, fnew);
    }
    free(buf);
    return rc;
}

/* one full step: O2 face loop (x then y), O10 cell loop, O11 residual */
static int step_once(ugkso_ctx *c)
{
    const int I = c->I, J = c->J, N = c->N;
    const size_t cells = (size_t)I * J;
    int nth = c->nthreads, err = 0;
    (void)nth;
    memset(c->D, 0, sizeof(double) * cells * N);
    memset(c->FWd, 0, sizeof(double) * cells * 4);

    /* x-faces: rows are independent (a face touches only cells of its row) */
    #pragma omp parallel num_threads(nth)
    {
        double *buf = (double *)malloc(sizeof(double) * 8 * (size_t)N), FW[4];
        int lerr = buf ? 0 : UGKSO_ENOMEM;
        #pragma omp for schedule(static)
        for (int j = 0; j < J; ++j) {
            for (int i = 0; i <= I && !lerr; ++i) {
                int rc = face_flux(c, 0, i, j, FW, buf, buf + N, NULL);
                if (rc) { lerr = rc; break; }
                int iL = i - 1, iR = i;                                     /* periodic: wrap to owners */
                if (c->bc[0].type == UGKSO_BC_PERIODIC) { if (i == I) continue; if (iL < 0) iL += I; }
                if (iR < I) {
                    double *D = c->D + ((size_t)j * I + iR) * N, *G = c->FWd + ((size_t)j * I + iR) * 4;
                    for (int q = 0; q < N; ++q) D[q] += buf[q];
                    for (int r = 0; r < 4; ++r) G[r] += FW[r];
                }
                if (iL >= 0) {
                    double *D = c->D + ((size_t)j * I + iL) * N, *G = c->FWd + ((size_t)j * I + iL) * 4;
                    for (int q = 0; q < N; ++q) D[q] -= buf[q];
                    for (int r = 0; r < 4; ++r) G[r] -= FW[r];
                }
            }
        }
        #pragma omp critical
        { if (lerr && !err) err = lerr; }
        #pragma omp barrier
        /* y-faces: columns are independent */
        #pragma omp for schedule(static)
        for (int i = 0; i < I; ++i) {
            for (int j = 0; j <= J && !lerr && buf; ++j) {
                int rc = face_flux(c, 1, i, j, FW, buf, buf + N, NULL);
                if (rc) { lerr = rc; break; }
                int jL = j - 1, jR = j;
                if (c->bc[2].type == UGKSO_BC_PERIODIC) { if (j == J) continue; if (jL < 0) jL += J; }
                if (jR < J) {
                    double *D = c->D + ((size_t)jR * I + i) * N, *G = c->FWd + ((size_t)jR * I + i) * 4;
                    for (int q = 0; q < N; ++q) D[q] += buf[q];
                    for (int r = 0; r < 4; ++r) G[r] += FW[r];
                }
                if (jL >= 0) {
                    double *D = c->D + ((size_t)jL * I + i) * N, *G = c->FWd + ((size_t)jL * I + i) * 4;
                    for (int q = 0; q < N; ++q) D[q] -= buf[q];
                    for (int r = 0; r < 4; ++r) G[r] -= FW[r];
                }
            }
        }
        #pragma omp critical
        { if (lerr && !err) err = lerr; }
        free(buf);
    }
    if (err) return err;

    /* O10: W update (Eq. (4)) then implicit f update (Eq. (3)) */
    double Om = c->dx * c->dy;
    #pragma omp parallel for schedule(static) num_threads(nth)
    for (long cell = 0; cell < (long)cells; ++cell) {
        double *Wn = c->Wn + cell * 4;
        for (int r = 0; r < 4; ++r) Wn[r] = c->W[cell * 4 + r] + c->FWd[cell * 4 + r] / Om;
        int rc = relax_cell(c, c->W + cell * 4, Wn, c->f + cell * N, c->D + cell * N, c->f + cell * N);
        if (rc) {
            #pragma omp critical
            { if (!err) err = rc; }
        }
    }
    /* O11 (RES, AMB-15) */
    for (int r = 0; r < 4; ++r) {
        ksum d2 = {0, 0}, ab = {0, 0};
        for (size_t cell = 0; cell < cells; ++cell) {
            double d = c->Wn[cell * 4 + r] - c->W[cell * 4 + r];
            ks_add(&d2, d * d); ks_add(&ab, fabs(c->Wn[cell * 4 + r]));
        }
        c->res[r] = sqrt((double)cells * ks_val(&d2)) / (ks_val(&ab) + 1e-300);
    }
    double *t = c->W; c->W = c->Wn; c->Wn = t;
    c->have_res = 1; c->steps += 1;
    return err;
}

int ugkso_step(ugkso_ctx *c, int n)
{
    if (!c || n < 0) return UGKSO_EINVAL;
    if (!c->have_state) return UGKSO_ESTATE;
    for (int s = 0; s < n; ++s) { int rc = step_once(c); if (rc) return rc; }
    return UGKSO_OK;
}
int ugkso_residual(ugkso_ctx *c, double res[4])
{
    if (!c || !res) return UGKSO_EINVAL;
    if (!c->have_res) return UGKSO_ESTATE;
    memcpy(res, c->res, sizeof c->res);
    return UGKSO_OK;
}
