// ugks_update.cu -- k_flux_update: S6 + S8 at the four faces of every cell fused with the
// updates U3 (Eq. (3)); U1/U2 come precomputed per cell from k_cell_scalars.
//
// One CTA marches along a strip of cells of row j for one chunk of velocity rows.  The x-stencil rows
// (i-2..i+2, j) live in a TMA-fed shared-memory ring; the four y-stencil rows (i, j-2), (i, j-1), (i, j+1),
// (i, j+2) of each cell are double-buffered.  The x-face flux is evaluated once per face and carried to the
// next cell; the two y-faces of a cell are evaluated by the cell itself.  f^{n+1} is written straight from
// registers: f is read from HBM once (plus L2-served stencil re-reads) and written once.
#include "ugks_common.cuh"

struct FaceCoef {
    double C0, U, V, lam, Mt1, Mt2, Mt3, Mt4, Mt5, aL[4], aR[4], b[4], A[4], rho_w;
};
__device__ __forceinline__ FaceCoef load_coef(const double *cf)
{
    FaceCoef c;
    c.C0 = cf[CF_C0]; c.U = cf[CF_U]; c.V = cf[CF_V]; c.lam = cf[CF_LAM];
    c.Mt1 = cf[CF_MT1]; c.Mt2 = cf[CF_MT2]; c.Mt3 = cf[CF_MT3]; c.Mt4 = cf[CF_MT4]; c.Mt5 = cf[CF_MT5];
#pragma unroll
    for (int r = 0; r < 4; ++r) { c.aL[r] = cf[CF_AL + r]; c.aR[r] = cf[CF_AR + r]; c.b[r] = cf[CF_B + r]; c.A[r] = cf[CF_A + r]; }
    c.rho_w = cf[CF_RHOW];
    return c;
}

// Time-integrated flux of f through one face at one velocity point (O3 + O8), signed along +x / +y.
// ms: bit0 LL missing, bit1 L missing, bit2 R missing, bit3 RR missing.  gw: wall Maxwellian at this point.
__device__ __forceinline__ double point_flux(const FaceCoef &c, double n, double t, double fLL, double fL, double fR,
                                             double fRR, int ms, double gw, double ell, double inv_h)
{
    double f0, hs;
    if (n > 0.0) {
        if (ms & 2) { f0 = c.rho_w * gw; hs = 0.0; }
        else {
            double dp = fR - fL, dm = fL - fLL;
            if (ms & 1) dm = dp;
            if (ms & 4) dp = dm;
            hs = vl_half(dm, dp);
            f0 = fL + hs;
        }
    } else if (n < 0.0) {
        if (ms & 4) { f0 = c.rho_w * gw; hs = 0.0; }
        else {
            double dm = fR - fL, dp = fRR - fR;
            if (ms & 2) dm = dp;
            if (ms & 8) dp = dm;
            hs = vl_half(dm, dp);
            f0 = fR - hs;
        }
    } else return 0.0;
    const double e = 0.5 * (n * n + t * t);
    const double *a = n > 0.0 ? c.aL : c.aR;
    const double ap = a[0] + a[1] * n + a[2] * t + a[3] * e;
    const double bp = c.b[0] + c.b[1] * n + c.b[2] * t + c.b[3] * e;
    const double Ap = c.A[0] + c.A[1] * n + c.A[2] * t + c.A[3] * e;
    const double dn = n - c.U, dtg = t - c.V;
    const double g0 = c.C0 * exp(-c.lam * (dn * dn + dtg * dtg));
    const double Pq = c.Mt1 + c.Mt2 * (n * ap + t * bp) + c.Mt3 * Ap;
    return ell * n * (Pq * g0 + c.Mt4 * f0 - c.Mt5 * n * (hs * inv_h));
}

template <int DIR>
__device__ __forceinline__ int miss_mask(const UgksParams &P, int a)
{
    const int n = DIR == 0 ? P.I : P.J, lo = DIR == 0 ? 0 : 2;
    const bool wlo = P.bc[lo] == BC_WALL, whi = P.bc[lo + 1] == BC_WALL;
    int ms = 0;
    for (int d = 0; d < 4; ++d) {
        const int pos = a - 2 + d;
        if ((pos < 0 && wlo) || (pos >= n && whi)) ms |= 1 << d;
    }
    return ms;
}

template <int MAXT>
__global__ void __launch_bounds__(MAXT) k_flux_update(const UgksParams P, const int cur)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    int b = blockIdx.x;
    const int j = b % P.J; b /= P.J;
    const int s = b % nstrip;
    const int chunk = b / nstrip;
    const int c0 = s * P.strip, c1 = min(c0 + P.strip, P.I);         // cells [c0, c1) of row j
    const int m0 = chunk * P.chunk_m, mc = min(P.chunk_m, P.Nv - m0);
    const int Nu = P.Nu, Q = mc * Nu, q0 = m0 * Nu;
    const int Qs = (P.chunk_m * Nu + 1) & ~1;
    const uint32_t bytes = (uint32_t)(((Q + 1) & ~1) * sizeof(double));

    double *ring = reinterpret_cast<double *>(smem_raw);             // [RINGX][Qs]
    double *ybuf = ring + (size_t)RINGX * Qs;                        // [2][4][Qs]
    double *Fprev = ybuf + (size_t)8 * Qs;                           // [Qs]
    double *Dacc = Fprev + Qs;                                       // [Qs]
    double *vt = Dacc + Qs;                                          // [chunk_m]
    uint64_t *bars = reinterpret_cast<uint64_t *>(vt + P.chunk_m);   // [RINGX] x-ring, [2] y buffers

    const int tid = threadIdx.x;
    const bool active = tid < Nu * P.R;
    const int k = tid % Nu, r = tid / Nu;
    const double *fcur = P.f[cur];
    double *fnew = P.f[cur ^ 1];
    const int rows_first = c0 - 2, rows_last = c1 + 1;

    if (tid == 0) {
        for (int i = 0; i < RINGX + 2; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    for (int i = tid; i < mc; i += blockDim.x) vt[i] = P.v[m0 + i];
    __syncthreads();

    auto issue_x = [&](int idx) {
        int miss;
        const double *src = row_ptr<0>(P, fcur, rows_first + idx, j, &miss) + q0;
        mbar_expect_tx(&bars[idx % RINGX], bytes);
        tma_load_1d(ring + (size_t)(idx % RINGX) * Qs, src, bytes, &bars[idx % RINGX]);
    };
    auto issue_y = [&](int cell) {
        const int buf = (cell - c0) & 1;
        mbar_expect_tx(&bars[RINGX + buf], 4 * bytes);
        const int dj[4] = { -2, -1, 1, 2 };
        for (int d = 0; d < 4; ++d) {
            int miss;
            const double *src = row_ptr<1>(P, fcur, j + dj[d], cell, &miss) + q0;
            tma_load_1d(ybuf + (size_t)(buf * 4 + d) * Qs, src, bytes, &bars[RINGX + buf]);
        }
    };
    if (tid == 0) {
        for (int idx = 0; idx < RINGX && rows_first + idx <= rows_last; ++idx) issue_x(idx);
        issue_y(c0);
        if (c0 + 1 < c1) issue_y(c0 + 1);
    }
    const double uk = active ? P.u[k] : 0.0;
    const double ihx = 2.0 / P.dx, ihy = 2.0 / P.dy;
    const int msy0 = miss_mask<1>(P, j), msy1 = miss_mask<1>(P, j + 1);
    const int wsy0 = (msy0 & 2) ? 2 : 3, wsy1 = (msy1 & 2) ? 2 : 3;  // which wall row a missing-upwind point reads
    const double *gwy0 = P.wallg + (size_t)wsy0 * P.Npad + q0, *gwy1 = P.wallg + (size_t)wsy1 * P.Npad + q0;

    for (int a = c0; a <= c1; ++a) {                                 // x-face a; then cell a-1
        const int idxN = a - c0 + 3;
        if (a == c0) for (int idx = 0; idx < 3; ++idx) mbar_wait(&bars[idx], 0);
        mbar_wait(&bars[idxN % RINGX], (idxN / RINGX) & 1);
        const double *rLL = ring + (size_t)((idxN - 3) % RINGX) * Qs;
        const double *rL = ring + (size_t)((idxN - 2) % RINGX) * Qs;
        const double *rR = ring + (size_t)((idxN - 1) % RINGX) * Qs;
        const double *rRR = ring + (size_t)(idxN % RINGX) * Qs;
        {
            const int ms = miss_mask<0>(P, a);
            const FaceCoef cf = load_coef(P.coef[0] + ((size_t)j * (P.I + 1) + a) * NCOEF);
            const double *gw = P.wallg + (size_t)((ms & 2) ? 0 : 1) * P.Npad + q0;
            if (active)
                for (int mm = r; mm < mc; mm += P.R) {
                    const int q = mm * Nu + k;
                    const double gwq = (ms & 6) ? gw[q] : 0.0;
                    const double F = point_flux(cf, uk, vt[mm], rLL[q], rL[q], rR[q], rRR[q], ms, gwq, P.dy, ihx);
                    if (a > c0) Dacc[q] = Fprev[q] - F;
                    Fprev[q] = F;
                }
        }
        if (a > c0) {
            const int cell = a - 1, buf = (cell - c0) & 1;
            mbar_wait(&bars[RINGX + buf], ((cell - c0) >> 1) & 1);
            const double *y0 = ybuf + (size_t)(buf * 4 + 0) * Qs, *y1 = y0 + Qs, *y3 = y1 + Qs, *y4 = y3 + Qs;
            const double *y2 = rL;                                   // the cell's own row: L of x-face a
            {
                const FaceCoef cf = load_coef(P.coef[1] + ((size_t)j * P.I + cell) * NCOEF);
                if (active)
                    for (int mm = r; mm < mc; mm += P.R) {
                        const int q = mm * Nu + k;
                        const double gwq = (msy0 & 6) ? gwy0[q] : 0.0;
                        Dacc[q] += point_flux(cf, vt[mm], uk, y0[q], y1[q], y2[q], y3[q], msy0, gwq, P.dx, ihy);
                    }
            }
            {
                const FaceCoef cf = load_coef(P.coef[1] + ((size_t)(j + 1) * P.I + cell) * NCOEF);
                const double *cc = P.cellc + ((size_t)j * P.I + cell) * NCELL;
                const double GN = cc[CC_GN], UN = cc[CC_UN], VN = cc[CC_VN], LN = cc[CC_LN];
                const double GP = cc[CC_GP], UP = cc[CC_UP], VP = cc[CC_VP], LP = cc[CC_LP];
                const double KF = cc[CC_KF], KD = cc[CC_KD];
                double *out = fnew + ((size_t)j * P.I + cell) * P.Npad + q0;
                if (active)
                    for (int mm = r; mm < mc; mm += P.R) {
                        const int q = mm * Nu + k;
                        const double v = vt[mm];
                        const double gwq = (msy1 & 6) ? gwy1[q] : 0.0;
                        const double D = Dacc[q] - point_flux(cf, v, uk, y1[q], y2[q], y3[q], y4[q], msy1, gwq, P.dx, ihy);
                        const double dun = uk - UN, dvn = v - VN, dup = uk - UP, dvp = v - VP;
                        const double gn = GN * exp(-LN * (dun * dun + dvn * dvn));
                        const double gp = GP * exp(-LP * (dup * dup + dvp * dvp));
                        out[q] = KF * y2[q] + KD * D + gp + gn;      // P:L41 Eq. (3), solved for f^{n+1}
                    }
            }
        }
        __syncthreads();
        if (tid == 0) {
            const int idx = a - c0 + RINGX;
            if (rows_first + idx <= rows_last && a < c1) issue_x(idx);
            if (a > c0 && a - 1 + 2 < c1) issue_y(a + 1);
        }
    }
}

size_t smem_flux_update(const UgksParams &P)
{
    const size_t Qs = ((size_t)P.chunk_m * P.Nu + 1) & ~(size_t)1;
    return ((RINGX + 8 + 2) * Qs + (size_t)P.chunk_m) * sizeof(double) + (RINGX + 2) * sizeof(uint64_t);
}

int launch_flux_update(const UgksParams &P, int cur, cudaStream_t st)
{
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    const int threads = ((P.Nu * P.R + 31) / 32) * 32;
    if (threads <= 256) k_flux_update<256><<<P.J * nstrip * P.nchunk, threads, smem_flux_update(P), st>>>(P, cur);
    else k_flux_update<1024><<<P.J * nstrip * P.nchunk, threads, smem_flux_update(P), st>>>(P, cur);
    return 1;
}

int setup_update_attributes(const UgksParams &P)
{
    const int smem = (int)smem_flux_update(P);
    cudaError_t e = cudaFuncSetAttribute(k_flux_update<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_flux_update<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    return e == cudaSuccess ? 0 : 1;
}
