// ugks_update.cu -- k_flux_update: S6 + S8 at the faces of every cell fused with the update U3
// (Eq. (3)); U1/U2 come precomputed per cell from k_cell_scalars.
//
// One CTA marches along a strip of cells of row j for one chunk of velocity rows.  Thread (k, r) owns velocity
// column k and the NPT rows m = r + p*R: everything that depends on the face and on u_k only (the cubic of the
// flux polynomial in the other velocity, the separable Maxwellian factor) is formed once per face per thread.
//   * x-stencil: each thread keeps its two upwind-side rows in registers and reads ONE new row per face from a
//     4-slot shared-memory ring fed by 1-D TMA bulk copies (two rows in flight).
//   * y-stencil: the rows (i, j-2), (i, j-1), (i, j+1), (i, j+2) of the cell are TMA-staged, double-buffered.
//   * the face Maxwellian is separable on the tensor-product grid: exp(-lam((n-U)^2+(t-V)^2)) = E_n[k] E_t[m]; the
//     5 (Nu + chunk) exponentials a step needs are computed cooperatively one step ahead into shared memory.
//   * the x-face flux is evaluated once per face and carried in registers to the next cell; the two y-faces of
//     a cell are evaluated by the cell.  f^{n+1} is written straight from registers: f crosses HBM once each way.
#include "ugks_common.cuh"

constexpr int REC_X = 0, REC_YL = NCOEF, REC_YU = 2 * NCOEF, REC_CC = 3 * NCOEF, REC_SIZE = 3 * NCOEF + NCELL;   // 84
constexpr int NREC = 3;                                              // record slots: records arrive two steps ahead
// per-step table buffer (doubles): k-tables [6 x-face][7 y-lower][7 y-upper][2 relaxation] x Nu, then
// m-tables [x-face Et][y-lower En][y-upper En][g^n][g^{n+1}] x chunk_m
constexpr int TK_X = 0, TK_YL = 6, TK_YU = 13, TK_G = 20, NKT = 22, NMT = 5;

// h*sigma of the van Leer limiter from un-normalised differences, with a Newton-refined MUFU reciprocal
// (rcp.approx.ftz.f64 gives ~2^-23; two FMA iterations reach ~1 ulp).  When dm*dp > 0 the sum is a normal number.
__device__ __forceinline__ double vl_half_fast(double dm, double dp)
{
    const double pr = dm * dp, s = dm + dp;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));
    double e = fma(-s, r, 1.0);
    r = fma(r, e, r);
    e = fma(-s, r, 1.0);
    r = fma(r, e, r);
    return pr > 0.0 ? pr * r : 0.0;
}

// upwind reconstruction at a face from the upwind cell c and its neighbours: f0 = f_c + sg * h sigma_c (O3).
// FLAGS: mm / mp = the minus / plus neighbour is a wall (one-sided slope, AMB-13); mc = the upwind cell itself is a
// wall: the incoming distribution is the wall Maxwellian fwall = rho_w g_w (O9).
template <bool FLAGS>
__device__ __forceinline__ void recon(double fm, double fc, double fp, double sg, bool mm, bool mc, bool mp, double fwall,
                                      double &f0, double &hs)
{
    double dm = fc - fm, dp = fp - fc;
    if (FLAGS) { if (mm) dm = dp; if (mp) dp = dm; }
    hs = vl_half_fast(dm, dp);
    f0 = fma(sg, hs, fc);
    if (FLAGS && mc) { f0 = fwall; hs = 0.0; }
}

template <int DIR>
__device__ __forceinline__ int miss_mask(const UgksParams &P, int a)
{
    const int n = DIR == 0 ? P.I : P.J, lo = DIR == 0 ? 0 : 2;
    const bool wlo = P.bc[lo] == BC_WALL, whi = P.bc[lo + 1] == BC_WALL;
    int ms = 0;
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        const int pos = a - 2 + d;
        if ((pos < 0 && wlo) || (pos >= n && whi)) ms |= 1 << d;
    }
    return ms;
}

template <int NPT, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_flux_update(const UgksParams P, const int cur)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    int b = blockIdx.x;
    const int j = b % P.J; b /= P.J;
    const int s = b % nstrip;
    const int chunk = b / nstrip;
    const int c0 = s * P.strip, c1 = min(c0 + P.strip, P.I);         // cells [c0, c1) of row j
    const int m0 = chunk * P.chunk_m, mc = min(P.chunk_m, P.Nv - m0);
    const int Nu = P.Nu, R = P.R, CM = P.chunk_m, Q = mc * Nu, q0 = m0 * Nu;
    const int Qs = (CM * Nu + 1) & ~1;
    const uint32_t bytes = (uint32_t)(((Q + 1) & ~1) * sizeof(double));
    const int tabsz = (NKT * Nu + NMT * CM + 1) & ~1;                // one table buffer, doubles

    double *ring = reinterpret_cast<double *>(smem_raw);             // [NSX][Qs]
    double *ybuf = ring + (size_t)NSX * Qs;                          // [2][4][Qs]
    double *tabs = ybuf + (size_t)8 * Qs;                            // [2][tabsz]
    double *recs = tabs + 2 * tabsz;                                 // [NREC][REC_SIZE]
    uint64_t *bars = reinterpret_cast<uint64_t *>(recs + NREC * REC_SIZE);   // [NSX] x-ring, [2] y buffers, [NREC] records

    const int tid = threadIdx.x;
    const bool active = tid < Nu * R;
    const int k = tid % Nu, r = tid / Nu;
    const double *fcur = P.f[cur];
    double *fnew = P.f[cur ^ 1];
    const int rows_first = c0 - 2, rows_last = c1 + 1;
    const double ihx = 2.0 / P.dx, ihy = 2.0 / P.dy;

    auto issue_x = [&](int row) {
        int miss;
        const int sl = (row - rows_first) % NSX;
        const double *src = row_ptr<0>(P, fcur, row, j, &miss) + q0;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(ring + (size_t)sl * Qs, src, bytes, &bars[sl]);
    };
    auto wait_x = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSX], (idx / NSX) & 1);
    };
    auto issue_y = [&](int cell) {
        const int buf = (cell - c0) & 1;
        mbar_expect_tx(&bars[NSX + buf], 4 * bytes);
        const int dj[4] = { -2, -1, 1, 2 };
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            int miss;
            const double *src = row_ptr<1>(P, fcur, j + dj[d], cell, &miss) + q0;
            tma_load_1d(ybuf + (size_t)(buf * 4 + d) * Qs, src, bytes, &bars[NSX + buf]);
        }
    };
    // records of step st: x-face st, and for cell st-1 its two y-faces and its relaxation coefficients
    auto issue_rec = [&](int st) {
        const int sl = (st - c0) % NREC;
        double *dst = recs + sl * REC_SIZE;
        const bool have_cell = st > c0;
        const int cell = st - 1;
        mbar_expect_tx(&bars[NSX + 2 + sl], (uint32_t)((have_cell ? REC_SIZE : NCOEF) * sizeof(double)));
        tma_load_1d(dst + REC_X, P.coef[0] + ((size_t)j * (P.I + 1) + st) * NCOEF, NCOEF * 8, &bars[NSX + 2 + sl]);
        if (have_cell) {
            tma_load_1d(dst + REC_YL, P.coef[1] + ((size_t)j * P.I + cell) * NCOEF, NCOEF * 8, &bars[NSX + 2 + sl]);
            tma_load_1d(dst + REC_YU, P.coef[1] + ((size_t)(j + 1) * P.I + cell) * NCOEF, NCOEF * 8, &bars[NSX + 2 + sl]);
            tma_load_1d(dst + REC_CC, P.cellc + ((size_t)j * P.I + cell) * NCELL, NCELL * 8, &bars[NSX + 2 + sl]);
        }
    };
    // tables of step st -> buffer st&1.  One work item = one velocity node of one table group:
    //   items [0,3Nu): (face f, k): separable factor E[k] and the flux polynomial column of that face at u_k
    //   items [3Nu,5Nu): relaxation factors of g^n, g^{n+1} in u;  items [5Nu, 5Nu+5mc): the five m-tables
    auto make_tables = [&](int st) {
        const int sl = (st - c0) % NREC;
        mbar_wait(&bars[NSX + 2 + sl], ((st - c0) / NREC) & 1);
        const double *rec = recs + sl * REC_SIZE;
        double *T = tabs + (size_t)(st & 1) * tabsz, *Tm = T + NKT * Nu;
        const bool have_cell = st > c0;
        const int nitem = 5 * Nu + 5 * mc;
        for (int e = tid; e < nitem; e += blockDim.x) {
            if (e < 3 * Nu) {
                const int f = e / Nu, kk = e - f * Nu;
                if (f > 0 && !have_cell) continue;
                const double *g = rec + f * NCOEF;
                const double c = P.u[kk];
                if (f == 0) {                                        // x-face: n = u_k, cubic in t
                    const double *LR = g + (c > 0.0 ? CF_L : CF_R);
                    const double d = c - g[CF_U];
                    const double sc = P.dy * c * g[CF_C0] * exp(-g[CF_LAM] * d * d);
                    double *o = T + TK_X * Nu + kk;
                    o[0] = sc * fma(c, fma(c, fma(c, LR[2], LR[1]), LR[0]), g[CF_C00]);
                    o[Nu] = sc * fma(c, fma(c, g[CF_C21], LR[3]), g[CF_C01]);
                    o[2 * Nu] = sc * fma(c, LR[4], g[CF_C02]);
                    o[3 * Nu] = sc * g[CF_C03];
                    o[4 * Nu] = P.dy * c * g[CF_MT4];
                    o[5 * Nu] = -P.dy * c * c * g[CF_MT5] * ihx;
                } else {                                             // y-face: t = u_k, cubic in n (L and R variants)
                    const double d = c - g[CF_V];
                    const double sc = P.dx * exp(-g[CF_LAM] * d * d);
                    const double *L = g + CF_L, *Rr = g + CF_R;
                    double *o = T + (f == 1 ? TK_YL : TK_YU) * Nu + kk;
                    o[0] = sc * fma(c, fma(c, fma(c, g[CF_C03], g[CF_C02]), g[CF_C01]), g[CF_C00]);
                    o[Nu] = sc * fma(c, fma(c, L[4], L[3]), L[0]);
                    o[2 * Nu] = sc * fma(c, g[CF_C21], L[1]);
                    o[3 * Nu] = sc * L[2];
                    o[4 * Nu] = sc * fma(c, fma(c, Rr[4], Rr[3]), Rr[0]);
                    o[5 * Nu] = sc * fma(c, g[CF_C21], Rr[1]);
                    o[6 * Nu] = sc * Rr[2];
                }
            } else if (e < 5 * Nu) {
                if (!have_cell) continue;
                const int w = (e - 3 * Nu) / Nu, kk = e - (3 + w) * Nu;
                const double *cc = rec + REC_CC + (w == 0 ? CC_GN : CC_GP);
                const double d = P.u[kk] - cc[1];
                T[(TK_G + w) * Nu + kk] = cc[0] * exp(-cc[3] * d * d);
            } else {
                const int e2 = e - 5 * Nu, tab = e2 / mc, mi = e2 - tab * mc;
                if (tab > 0 && !have_cell) continue;
                const double vv = P.v[m0 + mi];
                double pref, lam, cen;
                if (tab == 0) { pref = 1.0; lam = rec[REC_X + CF_LAM]; cen = rec[REC_X + CF_V]; }
                else if (tab <= 2) { const double *g = rec + tab * NCOEF; pref = g[CF_C0]; lam = g[CF_LAM]; cen = g[CF_U]; }
                else { const double *cc = rec + REC_CC + (tab == 3 ? CC_GN : CC_GP); pref = 1.0; lam = cc[3]; cen = cc[2]; }
                const double d = vv - cen;
                Tm[tab * CM + mi] = pref * exp(-lam * d * d);
            }
        }
    };

    if (tid == 0) {
        for (int i = 0; i < NSX + 2 + NREC; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        issue_rec(c0);
        issue_rec(c0 + 1);
        for (int row = rows_first; row < rows_first + NSX && row <= rows_last; ++row) issue_x(row);
        issue_y(c0);
        if (c0 + 1 < c1) issue_y(c0 + 1);
    }
    make_tables(c0);

    const double uk = active ? P.u[k] : 0.0;
    const bool posx = uk > 0.0;
    const double sgx = posx ? 1.0 : -1.0;
    double vreg[NPT], fm[NPT], fc[NPT], Fprev[NPT];
    bool valid[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        valid[p] = active && mm < mc;
        vreg[p] = valid[p] ? P.v[m0 + mm] : 0.0;
        Fprev[p] = 0.0;
    }
    const int qbase = r * Nu + k, qstep = R * Nu;
    {   // prologue: the two oldest rows of each thread's x-window go to registers
        wait_x(c0 - 2); wait_x(c0 - 1); wait_x(c0);
        const double *ra = ring + (size_t)(posx ? 0 : 1) * Qs, *rb = ring + (size_t)(posx ? 1 : 2) * Qs;
#pragma unroll
        for (int p = 0; p < NPT; ++p) {
            fm[p] = valid[p] ? ra[qbase + p * qstep] : 0.0;
            fc[p] = valid[p] ? rb[qbase + p * qstep] : 0.0;
        }
    }
    __syncthreads();                                                 // tables of step c0 complete; rows c0-2, c0-1 consumed
    if (tid == 0) {
        if (c0 + 2 <= rows_last) issue_x(c0 + 2);
        if (c0 + 3 <= rows_last) issue_x(c0 + 3);
    }
    const int msy0 = miss_mask<1>(P, j), msy1 = miss_mask<1>(P, j + 1);
    const bool anyms = (msy0 | msy1) != 0;
    const double *gwy0 = P.wallg + (size_t)2 * P.Npad + q0, *gwy1 = P.wallg + (size_t)3 * P.Npad + q0;

    for (int a = c0; a <= c1; ++a) {                                 // x-face a, then cell a-1
        const double *T = tabs + (size_t)(a & 1) * tabsz, *Tm = T + NKT * Nu;
        const double *rec = recs + ((a - c0) % NREC) * REC_SIZE;
        if (a + 1 <= c1) make_tables(a + 1);                         // next step's tables: off the critical path
        wait_x(a + 1);
        double own[NPT], D[NPT];
        {
            const int ms = miss_mask<0>(P, a);
            const int sh = posx ? 0 : 1;
            const bool mm_ = (ms >> sh) & 1, mc_ = (ms >> (sh + 1)) & 1, mp_ = (ms >> (sh + 2)) & 1;
            const double *rn = ring + (size_t)((a + sh - rows_first) % NSX) * Qs;
            const double *tk = T + TK_X * Nu + k;
            const double p0 = tk[0], p1 = tk[Nu], p2 = tk[2 * Nu], p3 = tk[3 * Nu], c4 = tk[4 * Nu], c5 = tk[5 * Nu];
            const double rw = rec[REC_X + CF_RHOW];
            const double *gw = P.wallg + (size_t)(posx ? 0 : 1) * P.Npad + q0;
#pragma unroll
            for (int p = 0; p < NPT; ++p) {
                if (valid[p]) {
                    const int q = qbase + p * qstep;
                    const double fn = rn[q], t = vreg[p];
                    double f0, hs;
                    if (ms == 0) recon<false>(fm[p], fc[p], fn, sgx, false, false, false, 0.0, f0, hs);
                    else recon<true>(fm[p], fc[p], fn, sgx, mm_, mc_, mp_, mc_ ? rw * gw[q] : 0.0, f0, hs);
                    const double X = fma(t, fma(t, fma(t, p3, p2), p1), p0) * Tm[p * R + r];
                    const double F = fma(c4, f0, fma(c5, hs, X));
                    D[p] = Fprev[p] - F;
                    Fprev[p] = F;
                    own[p] = posx ? fc[p] : fm[p];                   // row of cell a-1
                    fm[p] = fc[p]; fc[p] = fn;
                }
            }
        }
        if (a > c0) {
            const int cell = a - 1, buf = (cell - c0) & 1;
            mbar_wait(&bars[NSX + buf], ((cell - c0) >> 1) & 1);
            const double *y0 = ybuf + (size_t)(buf * 4) * Qs, *y1 = y0 + Qs, *y3 = y1 + Qs, *y4 = y3 + Qs;
            {   // lower face j
                const double *tk = T + TK_YL * Nu + k;
                const double q0_ = tk[0], q1L = tk[Nu], q2L = tk[2 * Nu], q3L = tk[3 * Nu], q1R = tk[4 * Nu], q2R = tk[5 * Nu], q3R = tk[6 * Nu];
                const double c4 = P.dx * rec[REC_YL + CF_MT4], c5 = -P.dx * rec[REC_YL + CF_MT5] * ihy, rw = rec[REC_YL + CF_RHOW];
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    if (valid[p]) {
                        const int q = qbase + p * qstep;
                        const double n = vreg[p], o = own[p], a1 = y1[q];
                        const bool pos = n > 0.0;
                        double f0, hs;
                        if (pos) {
                            const double a0 = y0[q];
                            if (!anyms) recon<false>(a0, a1, o, 1.0, false, false, false, 0.0, f0, hs);
                            else recon<true>(a0, a1, o, 1.0, msy0 & 1, msy0 & 2, msy0 & 4, (msy0 & 2) ? rw * gwy0[q] : 0.0, f0, hs);
                        } else {
                            const double a3 = y3[q];
                            if (!anyms) recon<false>(a1, o, a3, -1.0, false, false, false, 0.0, f0, hs);
                            else recon<true>(a1, o, a3, -1.0, msy0 & 2, msy0 & 4, msy0 & 8, 0.0, f0, hs);
                        }
                        const double q1 = pos ? q1L : q1R, q2 = pos ? q2L : q2R, q3 = pos ? q3L : q3R;
                        const double poly = fma(n, fma(n, fma(n, q3, q2), q1), q0_);
                        D[p] += n * fma(c4, f0, fma(c5 * n, hs, poly * Tm[CM + p * R + r]));
                    }
                }
            }
            {   // upper face j+1, then the update of the cell
                const double *tk = T + TK_YU * Nu + k;
                const double q0_ = tk[0], q1L = tk[Nu], q2L = tk[2 * Nu], q3L = tk[3 * Nu], q1R = tk[4 * Nu], q2R = tk[5 * Nu], q3R = tk[6 * Nu];
                const double c4 = P.dx * rec[REC_YU + CF_MT4], c5 = -P.dx * rec[REC_YU + CF_MT5] * ihy, rw = rec[REC_YU + CF_RHOW];
                const double gnu = T[TK_G * Nu + k], gpu = T[(TK_G + 1) * Nu + k];
                const double KF = rec[REC_CC + CC_KF], KD = rec[REC_CC + CC_KD];
                double *out = fnew + ((size_t)j * P.I + cell) * P.Npad + q0;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    if (valid[p]) {
                        const int q = qbase + p * qstep, mi = p * R + r;
                        const double n = vreg[p], o = own[p], a3 = y3[q];
                        const bool pos = n > 0.0;
                        double f0, hs;
                        if (pos) {
                            const double a1 = y1[q];
                            if (!anyms) recon<false>(a1, o, a3, 1.0, false, false, false, 0.0, f0, hs);
                            else recon<true>(a1, o, a3, 1.0, msy1 & 1, msy1 & 2, msy1 & 4, 0.0, f0, hs);
                        } else {
                            const double a4 = y4[q];
                            if (!anyms) recon<false>(o, a3, a4, -1.0, false, false, false, 0.0, f0, hs);
                            else recon<true>(o, a3, a4, -1.0, msy1 & 2, msy1 & 4, msy1 & 8, (msy1 & 4) ? rw * gwy1[q] : 0.0, f0, hs);
                        }
                        const double q1 = pos ? q1L : q1R, q2 = pos ? q2L : q2R, q3 = pos ? q3L : q3R;
                        const double poly = fma(n, fma(n, fma(n, q3, q2), q1), q0_);
                        const double Dq = D[p] - n * fma(c4, f0, fma(c5 * n, hs, poly * Tm[2 * CM + mi]));
                        const double g = fma(Tm[4 * CM + mi], gpu, Tm[3 * CM + mi] * gnu);
                        out[q] = fma(KF, o, fma(KD, Dq, g));         // P:L41 Eq. (3), solved for f^{n+1}
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 0) {
            if (a + NSX <= rows_last) issue_x(a + NSX);              // row a is consumed, its slot takes row a+4
            if (a > c0 && a + 1 < c1) issue_y(a + 1);
            if (a + 2 <= c1) issue_rec(a + 2);
        }
    }
}

size_t smem_flux_update(const UgksParams &P)
{
    const size_t Qs = ((size_t)P.chunk_m * P.Nu + 1) & ~(size_t)1;
    const size_t tabsz = ((size_t)NKT * P.Nu + (size_t)NMT * P.chunk_m + 1) & ~(size_t)1;
    return ((NSX + 8) * Qs + 2 * tabsz + NREC * REC_SIZE) * sizeof(double) + (NSX + 2 + NREC) * sizeof(uint64_t);
}

// thread-count classes: <=128 threads (4 CTAs/SM by registers), <=256 (2 CTAs/SM), <=1024 (1 CTA/SM)
template <int MAXT, int MINB>
static bool launch_npt(const UgksParams &P, int cur, int grid, int threads, size_t smem, cudaStream_t st)
{
    switch (P.npt) {
#define CASE(N) case N: k_flux_update<N, MAXT, MINB><<<grid, threads, smem, st>>>(P, cur); return true;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    }
    return false;
}

int launch_flux_update(const UgksParams &P, int cur, cudaStream_t st)
{
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    const int threads = ((P.Nu * P.R + 31) / 32) * 32;
    const int grid = P.J * nstrip * P.nchunk;
    const size_t smem = smem_flux_update(P);
    if (threads <= 128) launch_npt<128, 4>(P, cur, grid, threads, smem, st);
    else if (threads <= 256) launch_npt<256, 2>(P, cur, grid, threads, smem, st);
    else launch_npt<1024, 1>(P, cur, grid, threads, smem, st);
    return 1;
}

template <int MAXT, int MINB>
static cudaError_t set_attr_all(int smem)
{
    cudaError_t e = cudaSuccess;
#define ATTR(N) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_flux_update<N, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    ATTR(1) ATTR(2) ATTR(3) ATTR(4) ATTR(5) ATTR(6) ATTR(7) ATTR(8)
#undef ATTR
    return e;
}

int setup_update_attributes(const UgksParams &P)
{
    const int smem = (int)smem_flux_update(P);
    cudaError_t e = set_attr_all<128, 4>(smem);
    if (e == cudaSuccess) e = set_attr_all<256, 2>(smem);
    if (e == cudaSuccess) e = set_attr_all<1024, 1>(smem);
    return e == cudaSuccess ? 0 : 1;
}
