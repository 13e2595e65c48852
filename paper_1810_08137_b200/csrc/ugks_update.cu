// ugks_update.cu -- k_flux_update: S6 + S8 at the four faces of every cell fused with the update U3
// (Eq. (3)); the per-face coefficients (S2..S5), the per-cell relaxation scalars (U1/U2) and every exponential
// come precomputed from k_face_scalars / k_cell_scalars / k_tables.
//
// One CTA marches along a strip of cells of row j for one chunk of velocity rows (all v_m of one sign where the grid
// allows: SGN = +1 / -1; SGN = 0 is the generic per-point path).  Thread (k, r) owns velocity column k and the rows
// m = r + p*R.  Step a evaluates x-face a and then finishes cell a-1.
//   * everything that depends on the face and on u_k only is formed once per face per thread: the four coefficients of the
//     flux polynomial in the other velocity (already multiplied by the separable Maxwellian factor of u_k) and the two
//     coefficients of f0 and h sigma0.  Per point that leaves a cubic (Horner), one table factor and two FMAs per face.
//   * x-stencil: the two older rows of each thread's window live in registers; ONE new row per step comes from a 3-slot
//     shared-memory ring fed by 1-D TMA bulk copies.  The x-face flux is evaluated once per face and carried in registers to
//     the next cell.
//   * y-stencil: three rows ((j-2, j-1, j+1) for v > 0, (j-1, j+1, j+2) for v < 0) are TMA-staged per cell, double-buffered,
//     together with the records of the step (face and cell coefficients, separable factors).
//   * f^{n+1} is written straight from registers: f crosses HBM once each way in this kernel.
#include "ugks_common.cuh"
#include <type_traits>

constexpr int NSX = 3;                                               // x-ring slots: rows a, a+1 live, a+2 in flight

struct StageLayout {                                                 // offsets in doubles inside one step stage
    int yrow, xrec, xm, ylrec, ylm, yurec, yum, crec, cgn, cgp, size;
};
__host__ __device__ inline StageLayout stage_layout(int ny, int Qb, int NuP, int cmp)
{
    StageLayout L;
    int o = 0;
    L.yrow = o; o += ny * Qb;
    L.xrec = o; o += FR_NCOEF + NuP;
    L.xm = o; o += cmp;
    L.ylrec = o; o += FR_NCOEF + NuP;
    L.ylm = o; o += cmp;
    L.yurec = o; o += FR_NCOEF + NuP;
    L.yum = o; o += cmp;
    L.crec = o; o += CR_NCOEF + 2 * NuP;
    L.cgn = o; o += cmp;
    L.cgp = o; o += cmp;
    L.size = o;
    return L;
}

template <int NPT, int SGN, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_flux_update(const UgksParams P, const int cur, const int chunk0)
{
    constexpr int NY = SGN == 0 ? 4 : 3;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    int b = blockIdx.x;
    const int j = b % P.J; b /= P.J;
    const int s = b % nstrip;
    const int chunk = chunk0 + b / nstrip;                           // chunks are sorted by sign: one launch per sign class
    const int4 ch = P.chunks[chunk];
    const int c0 = s * P.strip, c1 = min(c0 + P.strip, P.I);         // cells [c0, c1) of row j
    const int m0 = ch.x, mc = ch.y;
    const int Nu = P.Nu, R = P.R, NuP = P.NuP;
    const int q0 = m0 * Nu, qa = q0 & ~1, qsh = q0 - qa;
    const int ma = m0 & ~1, msh = m0 - ma;
    const int Qb = pad2(P.cmax * Nu + 1), cmp = pad2(P.cmax + 1);
    const uint32_t bytes = (uint32_t)(pad2(mc * Nu + qsh) * sizeof(double));
    const uint32_t mbytes = (uint32_t)(pad2(mc + msh) * sizeof(double));
    const uint32_t kbytes = (uint32_t)((FR_NCOEF + NuP) * sizeof(double));
    const uint32_t cbytes = (uint32_t)((CR_NCOEF + 2 * NuP) * sizeof(double));
    const StageLayout L = stage_layout(NY, Qb, NuP, cmp);

    double *ring = reinterpret_cast<double *>(smem_raw);             // [NSX][Qb]
    double *stages = ring + (size_t)NSX * Qb;                        // [2][L.size]
    uint64_t *bars = reinterpret_cast<uint64_t *>(stages + (size_t)2 * L.size);   // [NSX] x rows, [2] stages

    const int tid = threadIdx.x;
    const bool active = tid < Nu * R;
    const int k = active ? tid % Nu : 0, r = active ? tid / Nu : 0;
    const double *fcur = P.f[cur];
    double *fnew = P.f[cur ^ 1];
    const int rows_first = c0 - 2, rows_last = c1 + 1;

    auto issue_x = [&](int row) {
        const int sl = (row - rows_first) % NSX;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(ring + (size_t)sl * Qb, row_ptr<0>(P, fcur, row, j) + qa, bytes, &bars[sl]);
    };
    auto wait_x = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSX], (idx / NSX) & 1);
    };
    // stage of step st: record of x-face st and, for cell st-1, its y-neighbour rows, y-face records and cell record
    auto issue_stage = [&](int st) {
        const int sl = (st - c0) & 1;
        double *S = stages + (size_t)sl * L.size;
        uint64_t *bar = &bars[NSX + sl];
        const bool have_cell = st > c0;
        const bool have_face = true;
        uint32_t total = (have_face ? kbytes + mbytes : 0) + (have_cell ? NY * bytes + 2 * (kbytes + mbytes) + cbytes + 2 * mbytes : 0);
        mbar_expect_tx(bar, total);
        const double *xr = P.frec[0] + ((size_t)j * (P.I + 1) + st) * P.frs;
        tma_load_1d(S + L.xrec, xr, kbytes, bar);
        tma_load_1d(S + L.xm, xr + FR_NCOEF + NuP + ma, mbytes, bar);
        if (have_cell) {
            const int cell = st - 1;
            const int dj3[3] = { SGN > 0 ? -2 : -1, SGN > 0 ? -1 : 1, SGN > 0 ? 1 : 2 };
            const int dj4[4] = { -2, -1, 1, 2 };
#pragma unroll
            for (int d = 0; d < NY; ++d)
                tma_load_1d(S + L.yrow + (size_t)d * Qb, row_ptr<1>(P, fcur, j + (SGN == 0 ? dj4[d] : dj3[d]), cell) + qa, bytes, bar);
            const double *yl = P.frec[1] + ((size_t)j * P.I + cell) * P.frs, *yu = yl + (size_t)P.I * P.frs;
            tma_load_1d(S + L.ylrec, yl, kbytes, bar);
            tma_load_1d(S + L.ylm, yl + FR_NCOEF + NuP + ma, mbytes, bar);
            tma_load_1d(S + L.yurec, yu, kbytes, bar);
            tma_load_1d(S + L.yum, yu + FR_NCOEF + NuP + ma, mbytes, bar);
            const double *cr = P.crec + ((size_t)j * P.I + cell) * P.crs;
            tma_load_1d(S + L.crec, cr, cbytes, bar);
            tma_load_1d(S + L.cgn, cr + CR_NCOEF + 2 * NuP + ma, mbytes, bar);
            tma_load_1d(S + L.cgp, cr + CR_NCOEF + 2 * NuP + P.NvP + ma, mbytes, bar);
        }
    };

    if (tid == 0) {
        for (int i = 0; i < NSX + 2; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        for (int row = rows_first; row < rows_first + NSX; ++row) issue_x(row);
        issue_stage(c0);
        issue_stage(c0 + 1);
    }

    const double uk = P.u[k];
    const bool posx = uk > 0.0;
    const double sgx = posx ? 1.0 : -1.0;
    // Per-thread points p: velocity row m = r + p R.  A point outside the chunk (ragged tail, padding threads) is clamped
    // onto the first point of the chunk so that the arithmetic stays branch-free; only its store is masked.
    double vn[NPT], fm[NPT], fc[NPT], Fprev[NPT];
    bool valid[NPT];
    int qoff[NPT], moff[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        valid[p] = active && mm < mc;
        qoff[p] = qsh + (valid[p] ? mm * Nu + k : 0);
        moff[p] = msh + (valid[p] ? mm : 0);
        vn[p] = P.v[m0 + (valid[p] ? mm : 0)];
        Fprev[p] = 0.0;
    }
    {   // prologue: the two oldest rows of each thread's x-window go to registers
        wait_x(c0 - 2); wait_x(c0 - 1); wait_x(c0);
        const double *ra = ring + (size_t)(posx ? 0 : 1) * Qb, *rb = ring + (size_t)(posx ? 1 : 2) * Qb;
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fm[p] = ra[qoff[p]]; fc[p] = rb[qoff[p]]; }
    }
    __syncthreads();                                                 // rows c0-2, c0-1 consumed
    if (tid == 0) { issue_x(c0 + 1); issue_x(c0 + 2); }
    // wall flags of the two y-faces (CTA-uniform)
    const bool wl2 = beyond_wall<1>(P, j - 2), wl1 = beyond_wall<1>(P, j - 1), wu1 = beyond_wall<1>(P, j + 1), wu2 = beyond_wall<1>(P, j + 2);
    const bool anyy = wl2 || wl1 || wu1 || wu2;
    const double *gwy0 = P.wallg + (size_t)2 * P.Npad + qa, *gwy1 = P.wallg + (size_t)3 * P.Npad + qa;

    for (int a = c0; a <= c1; ++a) {                                 // x-face a, then cell a-1
        const double *S = stages + (size_t)((a - c0) & 1) * L.size;
        mbar_wait(&bars[NSX + ((a - c0) & 1)], ((a - c0) >> 1) & 1);
        wait_x(a + 1);
        const bool have_cell = a > c0;
        // ---- x-face a: polynomial column of this thread
        const double *xr = S + L.xrec;
        const double *xlr = xr + (posx ? FR_L : FR_R);
        const double Ek = uk * xr[FR_NCOEF + k];
        const double p0 = Ek * fma(uk, fma(uk, fma(uk, xlr[LR_C30], xlr[LR_C20]), xlr[LR_C10]), xr[FR_C00]);
        const double p1 = Ek * fma(uk, fma(uk, xr[FR_C21], xlr[LR_C11]), xr[FR_C01]);
        const double p2 = Ek * fma(uk, xlr[LR_C12], xr[FR_C02]);
        const double p3 = Ek * xr[FR_C03];
        const double c4 = uk * xr[FR_MT4];
        const double c45 = uk * fma(uk, xr[FR_MT5], sgx * xr[FR_MT4]);
        const double *xm = S + L.xm;
        const int sh = posx ? 0 : 1;
        const double *rn = ring + (size_t)((a + sh - rows_first) % NSX) * Qb;
        const bool xw0 = beyond_wall<0>(P, a - 2), xw1 = beyond_wall<0>(P, a - 1), xw2 = beyond_wall<0>(P, a), xw3 = beyond_wall<0>(P, a + 1);
        const bool anyx = xw0 || xw1 || xw2 || xw3;
        // ---- y-faces of cell a-1: polynomial columns (t = u_k), L (n > 0) / R (n < 0) variants
        const double *ylr = S + L.ylrec, *yur = S + L.yurec;
        double ql0 = 0, ql1 = 0, ql2 = 0, ql3 = 0, qu0 = 0, qu1 = 0, qu2 = 0, qu3 = 0;
        double ql1n = 0, ql2n = 0, ql3n = 0, qu1n = 0, qu2n = 0, qu3n = 0;         // R variants (mixed chunks only)
        double gnu = 0, gpu = 0, KF = 0, KD = 0, l4 = 0, l5 = 0, u4 = 0, u5 = 0;
        if (have_cell) {
            auto ycol = [&](const double *yr, const double *lr, double &q0_, double &q1_, double &q2_, double &q3_, bool first) {
                const double E = yr[FR_NCOEF + k];
                if (first) q0_ = E * fma(uk, fma(uk, fma(uk, yr[FR_C03], yr[FR_C02]), yr[FR_C01]), yr[FR_C00]);
                q1_ = E * fma(uk, fma(uk, lr[LR_C12], lr[LR_C11]), lr[LR_C10]);
                q2_ = E * fma(uk, yr[FR_C21], lr[LR_C20]);
                q3_ = E * lr[LR_C30];
            };
            ycol(ylr, ylr + (SGN >= 0 ? FR_L : FR_R), ql0, ql1, ql2, ql3, true);
            ycol(yur, yur + (SGN >= 0 ? FR_L : FR_R), qu0, qu1, qu2, qu3, true);
            if (SGN == 0) {
                double dummy;
                ycol(ylr, ylr + FR_R, dummy, ql1n, ql2n, ql3n, false);
                ycol(yur, yur + FR_R, dummy, qu1n, qu2n, qu3n, false);
            }
            const double *cr = S + L.crec;
            gnu = cr[CR_NCOEF + k]; gpu = cr[CR_NCOEF + NuP + k];
            KF = cr[CR_KF]; KD = cr[CR_KD];
            l4 = ylr[FR_MT4]; l5 = ylr[FR_MT5]; u4 = yur[FR_MT4]; u5 = yur[FR_MT5];
        }
        const double *y0 = S + L.yrow, *y1 = y0 + Qb, *y2 = y1 + Qb, *y3 = y2 + Qb;
        const double *ylm = S + L.ylm, *yum = S + L.yum, *cgn = S + L.cgn, *cgp = S + L.cgp;
        double *out = fnew + ((size_t)j * P.I + max(a - 1, 0)) * P.Npad + qa;

        auto body = [&](auto fl) {                                   // fl: some stencil of this step touches a wall
            constexpr bool FLX = decltype(fl)::value, FLY = decltype(fl)::value;
            // wall flags of this thread's x-window (cells a-2+sh, a-1+sh, a+sh)
            const bool xmm = FLX && (sh ? xw1 : xw0), xmc = FLX && (sh ? xw2 : xw1), xmp = FLX && (sh ? xw3 : xw2);
            const double rwx = FLX ? xr[FR_RHOW] : 0.0;
            const double *gwx = P.wallg + (size_t)(posx ? 0 : 1) * P.Npad + qa;
#pragma unroll
            for (int p = 0; p < NPT; ++p) {
                const double fn = rn[qoff[p]], t = vn[p];
                // x-face a (upwind cell = middle of the window)
                double dmx = fc[p] - fm[p], dpx = fn - fc[p], fup = fc[p];
                if (FLX) { if (xmm) dmx = dpx; if (xmp) dpx = dmx; }
                double hs = vl_half(dmx, dpx);
                if (FLX && xmc) { fup = rwx * gwx[qoff[p]]; hs = 0.0; }
                const double X = fma(t, fma(t, fma(t, p3, p2), p1), p0) * xm[moff[p]];
                const double F = fma(c4, fup, fma(c45, hs, X));
                const double Dx = Fprev[p] - F;
                Fprev[p] = F;
                const double own = posx ? fc[p] : fm[p];             // row of cell a-1
                fm[p] = fc[p]; fc[p] = fn;
                if (!have_cell) continue;
                // y-faces of cell a-1: G = F / n
                const double n = t;
                const bool pos = SGN > 0 || (SGN == 0 && n > 0.0);
                const double sg = pos ? 1.0 : -1.0;
                double r0, r1, r2;                                   // the three neighbour rows of this point's stencil
                if (SGN != 0) { r0 = y0[qoff[p]]; r1 = y1[qoff[p]]; r2 = y2[qoff[p]]; }
                else if (pos) { r0 = y0[qoff[p]]; r1 = y1[qoff[p]]; r2 = y2[qoff[p]]; }
                else { r0 = y1[qoff[p]]; r1 = y2[qoff[p]]; r2 = y3[qoff[p]]; }
                double d1, d2, d3, ful, fuu;
                if (pos) { d1 = r1 - r0; d2 = own - r1; d3 = r2 - own; ful = r1; fuu = own; }     // rows j-2, j-1 | j+1
                else { d1 = own - r0; d2 = r1 - own; d3 = r2 - r1; ful = own; fuu = r1; }         // rows j-1 | j+1, j+2
                double dl1 = d1, dl2 = d2, du2 = d2, du3 = d3;
                if (FLY) {                                           // AMB-13: one-sided slope next to a wall
                    if (pos) { if (wl2) dl1 = dl2; if (wl1) du2 = du3; if (wu1) du3 = du2; }      // lower: (j-2, j-1, j); upper: (j-1, j, j+1)
                    else { if (wl1) dl1 = dl2; if (wu1) dl2 = dl1; if (wu2) du3 = du2; }          // lower: (j-1, j, j+1); upper: (j, j+1, j+2)
                }
                double hl = vl_half(dl1, dl2), hu = vl_half(du2, du3);
                if (FLY) {
                    if (pos && wl1) { ful = ylr[FR_RHOW] * gwy0[qoff[p]]; hl = 0.0; }             // lower face is the ymin wall
                    if (!pos && wu1) { fuu = yur[FR_RHOW] * gwy1[qoff[p]]; hu = 0.0; }            // upper face is the ymax wall
                }
                const bool useR = SGN == 0 && !pos;
                const double a1 = useR ? ql1n : ql1, a2 = useR ? ql2n : ql2, a3 = useR ? ql3n : ql3;
                const double b1 = useR ? qu1n : qu1, b2 = useR ? qu2n : qu2, b3 = useR ? qu3n : qu3;
                const double Xl = fma(n, fma(n, fma(n, a3, a2), a1), ql0) * ylm[moff[p]];
                const double Xu = fma(n, fma(n, fma(n, b3, b2), b1), qu0) * yum[moff[p]];
                const double Gl = fma(l4, ful, fma(fma(l5, n, sg * l4), hl, Xl));
                const double Gu = fma(u4, fuu, fma(fma(u5, n, sg * u4), hu, Xu));
                const double Dq = fma(n, Gl - Gu, Dx);
                const double g = fma(cgp[moff[p]], gpu, cgn[moff[p]] * gnu);
                const double fnw = fma(KF, own, fma(KD, Dq, g));     // P:L41 Eq. (3), solved for f^{n+1}
                if (valid[p]) out[qoff[p]] = fnw;
            }
        };
        if (anyx || (anyy && have_cell)) body(std::true_type{}); else body(std::false_type{});
        __syncthreads();
        if (tid == 0) {
            if (a + 3 <= rows_last) issue_x(a + 3);                  // row a is consumed, its slot takes row a+3
            if (a + 2 <= c1) issue_stage(a + 2);
        }
    }
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32; }

static size_t smem_fu(const UgksParams &P, int ny)
{
    const int Qb = pad2(P.cmax * P.Nu + 1), cmp = pad2(P.cmax + 1);
    const StageLayout L = stage_layout(ny, Qb, P.NuP, cmp);
    return ((size_t)NSX * Qb + 2 * (size_t)L.size) * sizeof(double) + (NSX + 2) * sizeof(uint64_t);
}
size_t smem_flux_update(const UgksParams &P) { return smem_fu(P, 4); }

template <int SGN, int MAXT, int MINB>
static void launch_sgn(const UgksParams &P, int cur, int chunk0, int grid, int threads, size_t smem, cudaStream_t st)
{
    switch (P.npt) {
#define CASE(N) case N: k_flux_update<N, SGN, MAXT, MINB><<<grid, threads, smem, st>>>(P, cur, chunk0); break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7)
#undef CASE
    }
}
template <int SGN>
static void launch_class(const UgksParams &P, int cur, int chunk0, int nch, cudaStream_t st)
{
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    const int threads = block_threads(P);
    const int grid = P.J * nstrip * nch;
    const size_t smem = smem_fu(P, SGN == 0 ? 4 : 3);
    if (threads <= 64) launch_sgn<SGN, 64, 6>(P, cur, chunk0, grid, threads, smem, st);
    else if (threads <= 128) launch_sgn<SGN, 128, 3>(P, cur, chunk0, grid, threads, smem, st);
    else launch_sgn<SGN, 256, 2>(P, cur, chunk0, grid, threads, smem, st);
}

int launch_flux_update(const UgksParams &P, int cur, cudaStream_t st)
{
    // chunk order: [v < 0 ...][v > 0 ...][mixed ...]
    int n = 0;
    if (P.nneg) { launch_class<-1>(P, cur, 0, P.nneg, st); ++n; }
    if (P.npos) { launch_class<1>(P, cur, P.nneg, P.npos, st); ++n; }
    if (P.nmix) { launch_class<0>(P, cur, P.nneg + P.npos, P.nmix, st); ++n; }
    return n;
}

template <int SGN, int MAXT, int MINB>
static cudaError_t set_attr_all(int smem)
{
    cudaError_t e = cudaSuccess;
#define ATTR(N) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_flux_update<N, SGN, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    ATTR(1) ATTR(2) ATTR(3) ATTR(4) ATTR(5) ATTR(6) ATTR(7)
#undef ATTR
    return e;
}
template <int SGN>
static cudaError_t set_attr_sgn(int smem)
{
    cudaError_t e = set_attr_all<SGN, 64, 6>(smem);
    if (e == cudaSuccess) e = set_attr_all<SGN, 128, 3>(smem);
    if (e == cudaSuccess) e = set_attr_all<SGN, 256, 2>(smem);
    return e;
}

int setup_update_attributes(const UgksParams &P)
{
    const int s3 = (int)smem_fu(P, 3), s4 = (int)smem_fu(P, 4);
    if (s4 > 227 * 1024) return 1;
    cudaError_t e = set_attr_sgn<1>(s3);
    if (e == cudaSuccess) e = set_attr_sgn<-1>(s3);
    if (e == cudaSuccess) e = set_attr_sgn<0>(s4);
    return e == cudaSuccess ? 0 : 1;
}
