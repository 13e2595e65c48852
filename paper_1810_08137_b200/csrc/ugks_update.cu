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
#include <type_traits>

constexpr int REC_X = 0, REC_YL = NCOEF, REC_YU = 2 * NCOEF, REC_CC = 3 * NCOEF, REC_SIZE = 3 * NCOEF + NCELL;   // 84
constexpr int NREC = 4;                                              // record slots: records arrive three steps ahead
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
    double *un = recs + NREC * REC_SIZE;                             // [Nu] velocity nodes u_k
    double *vn = un + ((Nu + 1) & ~1);                               // [CM] velocity nodes v_m of this chunk
    uint64_t *bars = reinterpret_cast<uint64_t *>(vn + ((CM + 1) & ~1));     // [NSX] x-ring, [2] y buffers, [NREC] records

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
    // tables of step st -> buffer st&1, two warp-uniform groups of work items:
    //   A (threads from the front): one item per (face f, k): E[k] and the flux-polynomial column of that face at u_k
    //   B (threads from the back): one item per plain separable factor: g^n, g^{n+1} in u (2 Nu) and the five m-tables
    auto make_tables = [&](int st) {
        const int sl = (st - c0) % NREC;
        mbar_wait(&bars[NSX + 2 + sl], ((st - c0) / NREC) & 1);
        const double *rec = recs + sl * REC_SIZE;
        double *T = tabs + (size_t)(st & 1) * tabsz, *Tm = T + NKT * Nu;
        const bool have_cell = st > c0;
        const int nA = (have_cell ? 3 : 1) * Nu;
        for (int e = tid; e < nA; e += blockDim.x) {
            const int f = (e >= Nu) + (e >= 2 * Nu), kk = e - f * Nu;
            const double *g = rec + f * NCOEF;
            const double c = un[kk];
            const double d = c - (f == 0 ? g[CF_U] : g[CF_V]);
            const double E = exp(-g[CF_LAM] * d * d);
            if (f == 0) {                                            // x-face: n = u_k, cubic in t
                const double *LR = g + (c > 0.0 ? CF_L : CF_R);
                const double sc = P.dy * c * g[CF_C0] * E;
                double *o = T + TK_X * Nu + kk;
                o[0] = sc * fma(c, fma(c, fma(c, LR[2], LR[1]), LR[0]), g[CF_C00]);
                o[Nu] = sc * fma(c, fma(c, g[CF_C21], LR[3]), g[CF_C01]);
                o[2 * Nu] = sc * fma(c, LR[4], g[CF_C02]);
                o[3 * Nu] = sc * g[CF_C03];
                o[4 * Nu] = P.dy * c * g[CF_MT4];
                o[5 * Nu] = -P.dy * c * c * g[CF_MT5] * ihx;
            } else {                                                 // y-face: t = u_k, cubic in n (L and R variants)
                const double sc = P.dx * E;
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
        }
        // B items: [0, mc): x-face Et[m];  then (cell only) y-lower En[m], y-upper En[m], g^n v, g^{n+1} v, g^n u, g^{n+1} u
        const int nB = have_cell ? 5 * mc + 2 * Nu : mc;
        for (int e = (int)blockDim.x - 1 - tid; e < nB; e += blockDim.x) {
            const bool isk = e >= 5 * mc;
            const int e2 = isk ? e - 5 * mc : e;
            const int len = isk ? Nu : mc;
            int tab = 0;
            tab += e2 >= len; tab += e2 >= 2 * len; tab += e2 >= 3 * len; tab += e2 >= 4 * len;
            const int idx = e2 - tab * len;
            const double node = isk ? un[idx] : vn[idx];
            // (pref, lam, centre) of the factor
            const bool relax = isk || tab >= 3;
            const int w = isk ? tab : tab - 3;                       // 0: g^n, 1: g^{n+1}
            const double *g = relax ? rec + REC_CC + (w == 0 ? CC_GN : CC_GP) : rec + tab * NCOEF;
            const double lam = relax ? g[3] : g[CF_LAM];
            const double cen = relax ? (isk ? g[1] : g[2]) : (tab == 0 ? g[CF_V] : g[CF_U]);
            const double pref = relax ? (isk ? g[0] : 1.0) : (tab == 0 ? 1.0 : g[CF_C0]);
            const double d = node - cen;
            const double val = pref * exp(-lam * d * d);
            if (isk) T[(TK_G + tab) * Nu + idx] = val; else Tm[tab * CM + idx] = val;
        }
    };

    if (tid == 0) {
        for (int i = 0; i < NSX + 2 + NREC; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    for (int i = tid; i < Nu; i += blockDim.x) un[i] = P.u[i];
    for (int i = tid; i < mc; i += blockDim.x) vn[i] = P.v[m0 + i];
    __syncthreads();
    if (tid == 0) {
        issue_rec(c0);
        issue_rec(c0 + 1);
        if (c0 + 2 <= c1) issue_rec(c0 + 2);
        for (int row = rows_first; row < rows_first + NSX && row <= rows_last; ++row) issue_x(row);
        issue_y(c0);
        if (c0 + 1 < c1) issue_y(c0 + 1);
    }
    make_tables(c0);

    const double uk = active ? P.u[k] : 0.0;
    const bool posx = uk > 0.0;
    const double sgx = posx ? 1.0 : -1.0;
    // Per-thread points p = 0..NPT-1: velocity row m = r + p R.  A point outside the chunk (ragged tail, padding
    // threads) is clamped onto point 0 of the row so that the arithmetic stays branch-free; only its store is masked.
    double vreg[NPT], fm[NPT], fc[NPT], Fprev[NPT];
    bool valid[NPT];
    int qo[NPT], mo[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        valid[p] = active && mm < mc;
        qo[p] = valid[p] ? mm * Nu + k : 0;
        mo[p] = valid[p] ? mm : 0;
        vreg[p] = vn[mo[p]];
        Fprev[p] = 0.0;
    }
    {   // prologue: the two oldest rows of each thread's x-window go to registers
        wait_x(c0 - 2); wait_x(c0 - 1); wait_x(c0);
        const double *ra = ring + (size_t)(posx ? 0 : 1) * Qs, *rb = ring + (size_t)(posx ? 1 : 2) * Qs;
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fm[p] = ra[qo[p]]; fc[p] = rb[qo[p]]; }
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
            const double *rn = ring + (size_t)((a + sh - rows_first) % NSX) * Qs;
            const double *tk = T + TK_X * Nu + k;
            const double p0 = tk[0], p1 = tk[Nu], p2 = tk[2 * Nu], p3 = tk[3 * Nu], c4 = tk[4 * Nu], c5 = tk[5 * Nu];
            auto xpass = [&](auto fl) {
                constexpr bool FL = decltype(fl)::value;
                const bool mm_ = (ms >> sh) & 1, mc_ = (ms >> (sh + 1)) & 1, mp_ = (ms >> (sh + 2)) & 1;
                const double rw = rec[REC_X + CF_RHOW];
                const double *gw = P.wallg + (size_t)(posx ? 0 : 1) * P.Npad + q0;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double fn = rn[qo[p]], t = vreg[p];
                    double f0, hs;
                    recon<FL>(fm[p], fc[p], fn, sgx, mm_, mc_, mp_, (FL && mc_) ? rw * gw[qo[p]] : 0.0, f0, hs);
                    const double X = fma(t, fma(t, fma(t, p3, p2), p1), p0) * Tm[mo[p]];
                    const double F = fma(c4, f0, fma(c5, hs, X));
                    D[p] = Fprev[p] - F;
                    Fprev[p] = F;
                    own[p] = posx ? fc[p] : fm[p];                   // row of cell a-1
                    fm[p] = fc[p]; fc[p] = fn;
                }
            };
            if (ms == 0) xpass(std::false_type{}); else xpass(std::true_type{});
        }
        if (a > c0) {
            const int cell = a - 1, buf = (cell - c0) & 1;
            mbar_wait(&bars[NSX + buf], ((cell - c0) >> 1) & 1);
            const double *y0 = ybuf + (size_t)(buf * 4) * Qs, *y1 = y0 + Qs, *y3 = y1 + Qs, *y4 = y3 + Qs;
            // one y-face: UP = 0 lower face j (rows j-2..j+1), UP = 1 upper face j+1 (rows j-1..j+2); returns its flux
            auto yflux = [&](auto fl, auto up, int p, const double *tk, double c4, double c5, double rw, int ms, const double *gwy) {
                constexpr bool FL = decltype(fl)::value;
                constexpr int UP = decltype(up)::value;
                const double n = vreg[p], o = own[p];
                const int q = qo[p];
                const bool pos = n > 0.0;
                double f0, hs;
                if (pos) {                                           // upwind cell is the lower one of the face
                    const double lo = UP ? y1[q] : y0[q], mid = UP ? o : y1[q], hi = UP ? y3[q] : o;
                    recon<FL>(lo, mid, hi, 1.0, ms & 1, ms & 2, ms & 4, (FL && (ms & 2)) ? rw * gwy[q] : 0.0, f0, hs);
                } else {
                    const double lo = UP ? o : y1[q], mid = UP ? y3[q] : o, hi = UP ? y4[q] : y3[q];
                    recon<FL>(lo, mid, hi, -1.0, ms & 2, ms & 4, ms & 8, (FL && (ms & 4)) ? rw * gwy[q] : 0.0, f0, hs);
                }
                const double q1 = pos ? tk[Nu] : tk[4 * Nu], q2 = pos ? tk[2 * Nu] : tk[5 * Nu], q3 = pos ? tk[3 * Nu] : tk[6 * Nu];
                const double poly = fma(n, fma(n, fma(n, q3, q2), q1), tk[0]);
                return n * fma(c4, f0, fma(c5 * n, hs, poly * Tm[(1 + UP) * CM + mo[p]]));
            };
            auto ypass = [&](auto fl) {
                {
                    const double *tk = T + TK_YL * Nu + k;
                    const double c4 = P.dx * rec[REC_YL + CF_MT4], c5 = -P.dx * rec[REC_YL + CF_MT5] * ihy, rw = rec[REC_YL + CF_RHOW];
#pragma unroll
                    for (int p = 0; p < NPT; ++p) D[p] += yflux(fl, std::integral_constant<int, 0>{}, p, tk, c4, c5, rw, msy0, gwy0);
                }
                const double *tk = T + TK_YU * Nu + k;
                const double c4 = P.dx * rec[REC_YU + CF_MT4], c5 = -P.dx * rec[REC_YU + CF_MT5] * ihy, rw = rec[REC_YU + CF_RHOW];
                const double gnu = T[TK_G * Nu + k], gpu = T[(TK_G + 1) * Nu + k];
                const double KF = rec[REC_CC + CC_KF], KD = rec[REC_CC + CC_KD];
                double *out = fnew + ((size_t)j * P.I + cell) * P.Npad + q0;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double Dq = D[p] - yflux(fl, std::integral_constant<int, 1>{}, p, tk, c4, c5, rw, msy1, gwy1);
                    const double g = fma(Tm[4 * CM + mo[p]], gpu, Tm[3 * CM + mo[p]] * gnu);
                    const double fnw = fma(KF, own[p], fma(KD, Dq, g));       // P:L41 Eq. (3), solved for f^{n+1}
                    if (valid[p]) out[qo[p]] = fnw;
                }
            };
            if (!anyms) ypass(std::false_type{}); else ypass(std::true_type{});
        }
        __syncthreads();
        if (tid == 0) {
            if (a + NSX <= rows_last) issue_x(a + NSX);              // row a is consumed, its slot takes row a+4
            if (a > c0 && a + 1 < c1) issue_y(a + 1);
            if (a + 3 <= c1) issue_rec(a + 3);
        }
    }
}

size_t smem_flux_update(const UgksParams &P)
{
    const size_t Qs = ((size_t)P.chunk_m * P.Nu + 1) & ~(size_t)1;
    const size_t tabsz = ((size_t)NKT * P.Nu + (size_t)NMT * P.chunk_m + 1) & ~(size_t)1;
    return ((NSX + 8) * Qs + 2 * tabsz + NREC * REC_SIZE + (((size_t)P.Nu + 1) & ~(size_t)1) + (((size_t)P.chunk_m + 1) & ~(size_t)1)) * sizeof(double)
           + (NSX + 2 + NREC) * sizeof(uint64_t);
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
