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

template <int NPT, int SGN>
__device__ __forceinline__ void flux_update_body(const UgksParams &P, const int cur, const int4 ch, const int j, const int s)
{
    constexpr int NY = SGN == 0 ? 4 : 3;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int c0 = s * P.strip, c1 = min(c0 + P.strip, P.I);         // cells [c0, c1) of row j
    const int m0 = ch.x, mc = ch.y;
    const int Nu = P.Nu, R = P.R, NuP = P.NuP;
    const int q0 = m0 * Nu, qa = q0 & ~1, qsh = q0 - qa;
    const int ma = m0 & ~1, msh = m0 - ma;
    const int Qb = pad2(P.cmax * Nu + 1), QbB = Qb * 8, cmp = pad2(P.cmax + 1);
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
    const int ncomp = blockDim.x - 32;                               // compute threads; the last warp is the TMA producer
    if (tid >= ncomp) {                                              // ---- producer warp: one lane issues every bulk copy
        const bool lead = tid == ncomp;
    // global sources of a step, linear in the cell index: y-neighbour rows, face records, cell records
        const int djs[4] = { SGN == 0 ? -2 : (SGN > 0 ? -2 : -1), SGN == 0 ? -1 : (SGN > 0 ? -1 : 1), SGN == 0 ? 1 : (SGN > 0 ? 1 : 2), 2 };
        const double *yb[NY];
        int yst[NY];
#pragma unroll
        for (int d = 0; d < NY; ++d) yb[d] = yrow_base(P, fcur, j + djs[d], &yst[d]) + qa;
        const double *xrp = P.frec[0] + (size_t)j * (P.I + 1) * P.frs;
        const double *ylp = P.frec[1] + (size_t)j * P.I * P.frs, *yup = ylp + (size_t)P.I * P.frs;
        const double *crp = P.crec + (size_t)j * P.I * P.crs;
        const int moffK = FR_NCOEF + NuP + ma, moffC = CR_NCOEF + 2 * NuP + ma;

        auto issue_x = [&](int row) {
            const int sl = (row - rows_first) % NSX;
            mbar_expect_tx(&bars[sl], bytes);
            tma_load_1d(ring + (size_t)sl * Qb, row_ptr<0>(P, fcur, row, j) + qa, bytes, &bars[sl]);
        };
        // stage of step st: record of x-face st and, for cell st-1, its y-neighbour rows, y-face records and cell record
        auto issue_stage = [&](int st) {
            const int sl = (st - c0) & 1;
            double *S = stages + (size_t)sl * L.size;
            uint64_t *bar = &bars[NSX + sl];
            const bool have_cell = st > c0;
            mbar_expect_tx(bar, kbytes + mbytes + (have_cell ? NY * bytes + 2 * (kbytes + mbytes) + cbytes + 2 * mbytes : 0));
            const double *xr = xrp + (size_t)st * P.frs;
            tma_load_1d(S + L.xrec, xr, kbytes, bar);
            tma_load_1d(S + L.xm, xr + moffK, mbytes, bar);
            if (have_cell) {
                const size_t cell = st - 1;
#pragma unroll
                for (int d = 0; d < NY; ++d) tma_load_1d(S + L.yrow + (size_t)d * Qb, yb[d] + cell * yst[d], bytes, bar);
                const double *yl = ylp + cell * P.frs, *yu = yup + cell * P.frs, *cr = crp + cell * P.crs;
                tma_load_1d(S + L.ylrec, yl, kbytes, bar);
                tma_load_1d(S + L.ylm, yl + moffK, mbytes, bar);
                tma_load_1d(S + L.yurec, yu, kbytes, bar);
                tma_load_1d(S + L.yum, yu + moffK, mbytes, bar);
                tma_load_1d(S + L.crec, cr, cbytes, bar);
                tma_load_1d(S + L.cgn, cr + moffC, mbytes, bar);
                tma_load_1d(S + L.cgp, cr + moffC + P.NvP, mbytes, bar);
            }
        };

        if (lead) {
            for (int i = 0; i < NSX + 2; ++i) mbar_init(&bars[i], 1);
            mbar_fence_init();
        }
        __syncthreads();
        if (lead) {
            for (int row = rows_first; row < rows_first + NSX; ++row) issue_x(row);
            issue_stage(c0);
            issue_stage(c0 + 1);
        }
        __syncthreads();                                             // rows c0-2, c0-1 consumed
        if (lead) { issue_x(c0 + 1); issue_x(c0 + 2); }
        for (int a = c0; a <= c1; ++a) {
            __syncthreads();                                         // step a done: row a and stage a are free
            if (lead) {
                if (a + 3 <= rows_last) issue_x(a + 3);
                if (a + 2 <= c1) issue_stage(a + 2);
            }
        }
        return;
    }
    auto wait_x = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSX], (idx / NSX) & 1);
    };
    __syncthreads();                                                 // barriers initialised

    const double uk = P.u[k];
    const bool posx = uk > 0.0;
    const double sgx = posx ? 1.0 : -1.0;
    // Per-thread points p: velocity row m = r + p R (byte offsets).  A point outside the chunk (ragged tail, padding
    // threads) is clamped onto the first point of the chunk so that the arithmetic stays branch-free; only its store is masked.
    double vn[NPT], fm[NPT], fc[NPT], Fprev[NPT];
    bool valid[NPT];
    int qb[NPT], mb[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        valid[p] = active && mm < mc;
        qb[p] = (qsh + (valid[p] ? mm * Nu + k : 0)) * 8;
        mb[p] = (msh + (valid[p] ? mm : 0)) * 8;
        vn[p] = P.v[m0 + (valid[p] ? mm : 0)];
        Fprev[p] = 0.0;
    }
    const unsigned char *ring_b = reinterpret_cast<const unsigned char *>(ring);
    const unsigned char *stages_b = reinterpret_cast<const unsigned char *>(stages);
    const int kb = k * 8;
    {   // prologue: the two oldest rows of each thread's x-window go to registers
        wait_x(c0 - 2); wait_x(c0 - 1); wait_x(c0);
        const unsigned char *ra = ring_b + (posx ? 0 : 1) * QbB, *rb = ra + QbB;
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fm[p] = ldsd(ra, qb[p]); fc[p] = ldsd(rb, qb[p]); }
    }
    __syncthreads();                                                 // rows c0-2, c0-1 consumed
    // wall flags of the two y-faces (CTA-uniform)
    const bool wl2 = beyond_wall<1>(P, j - 2), wl1 = beyond_wall<1>(P, j - 1), wu1 = beyond_wall<1>(P, j + 1), wu2 = beyond_wall<1>(P, j + 2);
    const bool anyy = wl2 || wl1 || wu1 || wu2;
    const unsigned char *gwy0 = reinterpret_cast<const unsigned char *>(P.wallg + (size_t)2 * P.Npad + qa);
    const unsigned char *gwy1 = reinterpret_cast<const unsigned char *>(P.wallg + (size_t)3 * P.Npad + qa);
    const unsigned char *gwx = reinterpret_cast<const unsigned char *>(P.wallg + (size_t)(posx ? 0 : 1) * P.Npad + qa);
    const int sh = posx ? 0 : 1;

    for (int a = c0; a <= c1; ++a) {                                 // x-face a, then cell a-1
        const unsigned char *S = stages_b + (size_t)((a - c0) & 1) * L.size * 8;
        mbar_wait(&bars[NSX + ((a - c0) & 1)], ((a - c0) >> 1) & 1);
        wait_x(a + 1);
        const bool have_cell = a > c0;
        // ---- x-face a: polynomial column of this thread (n = u_k; cubic in t = v_m)
        const double *xr = reinterpret_cast<const double *>(S + L.xrec * 8);
        const double *xlr = xr + (posx ? FR_L : FR_R);
        const double Ek = uk * ldsd(S + (L.xrec + FR_NCOEF) * 8, kb);
        const double p0 = Ek * fma(uk, fma(uk, fma(uk, xlr[LR_C30], xlr[LR_C20]), xlr[LR_C10]), xr[FR_C00]);
        const double p1 = Ek * fma(uk, fma(uk, xr[FR_C21], xlr[LR_C11]), xr[FR_C01]);
        const double p2 = Ek * fma(uk, xlr[LR_C12], xr[FR_C02]);
        const double p3 = Ek * xr[FR_C03];
        const double c4 = uk * xr[FR_MT4];
        const double c45 = uk * fma(uk, xr[FR_MT5], sgx * xr[FR_MT4]);
        const unsigned char *xm = S + L.xm * 8;
        const unsigned char *rn = ring_b + ((a + sh - rows_first) % NSX) * QbB;
        bool xw0 = false, xw1 = false, xw2 = false, xw3 = false;
        if (a < 2 || a + 2 > P.I) { xw0 = beyond_wall<0>(P, a - 2); xw1 = beyond_wall<0>(P, a - 1); xw2 = beyond_wall<0>(P, a); xw3 = beyond_wall<0>(P, a + 1); }
        const bool anyx = xw0 || xw1 || xw2 || xw3;
        // ---- y-faces of cell a-1: polynomial columns (t = u_k; cubic in n = v_m), L (n > 0) / R (n < 0) variants
        const double *ylr = reinterpret_cast<const double *>(S + L.ylrec * 8), *yur = reinterpret_cast<const double *>(S + L.yurec * 8);
        double ql0 = 0, ql1 = 0, ql2 = 0, ql3 = 0, qu0 = 0, qu1 = 0, qu2 = 0, qu3 = 0;
        double ql1n = 0, ql2n = 0, ql3n = 0, qu1n = 0, qu2n = 0, qu3n = 0;         // R variants (mixed chunks only)
        double gnu = 0, gpu = 0, KF = 0, KD = 0, l4 = 0, l5 = 0, u4 = 0, u5 = 0;
        if (have_cell) {
            auto ycol = [&](const double *yr, const double *lr, double E, double &q0_, double &q1_, double &q2_, double &q3_, bool first) {
                if (first) q0_ = E * fma(uk, fma(uk, fma(uk, yr[FR_C03], yr[FR_C02]), yr[FR_C01]), yr[FR_C00]);
                q1_ = E * fma(uk, fma(uk, lr[LR_C12], lr[LR_C11]), lr[LR_C10]);
                q2_ = E * fma(uk, yr[FR_C21], lr[LR_C20]);
                q3_ = E * lr[LR_C30];
            };
            const double El = ldsd(S + (L.ylrec + FR_NCOEF) * 8, kb), Eu = ldsd(S + (L.yurec + FR_NCOEF) * 8, kb);
            ycol(ylr, ylr + (SGN >= 0 ? FR_L : FR_R), El, ql0, ql1, ql2, ql3, true);
            ycol(yur, yur + (SGN >= 0 ? FR_L : FR_R), Eu, qu0, qu1, qu2, qu3, true);
            if (SGN == 0) {
                double dummy;
                ycol(ylr, ylr + FR_R, El, dummy, ql1n, ql2n, ql3n, false);
                ycol(yur, yur + FR_R, Eu, dummy, qu1n, qu2n, qu3n, false);
            }
            const double *cr = reinterpret_cast<const double *>(S + L.crec * 8);
            gnu = ldsd(S + (L.crec + CR_NCOEF) * 8, kb); gpu = ldsd(S + (L.crec + CR_NCOEF + NuP) * 8, kb);
            KF = cr[CR_KF]; KD = cr[CR_KD];
            l4 = ylr[FR_MT4]; l5 = ylr[FR_MT5]; u4 = yur[FR_MT4]; u5 = yur[FR_MT5];
        }
        const unsigned char *y0 = S + L.yrow * 8, *y1 = y0 + QbB, *y2 = y1 + QbB, *y3 = y2 + QbB;
        const unsigned char *ylm = S + L.ylm * 8, *yum = S + L.yum * 8, *cgn = S + L.cgn * 8, *cgp = S + L.cgp * 8;
        unsigned char *out = reinterpret_cast<unsigned char *>(fnew + ((size_t)j * P.I + max(a - 1, 0)) * P.Npad + qa);

        auto body = [&](auto fl) {                                   // fl: some stencil of this step touches a wall
            constexpr bool FL = decltype(fl)::value;
            // wall flags of this thread's x-window (cells a-2+sh, a-1+sh, a+sh)
            const bool xmm = FL && (sh ? xw1 : xw0), xmc = FL && (sh ? xw2 : xw1), xmp = FL && (sh ? xw3 : xw2);
            const double rwx = FL ? xr[FR_RHOW] : 0.0;
#pragma unroll
            for (int p = 0; p < NPT; ++p) {
                const double fn = ldsd(rn, qb[p]), t = vn[p];
                // x-face a (upwind cell = middle of the window)
                double dmx = fc[p] - fm[p], dpx = fn - fc[p], fup = fc[p];
                if (FL) { if (xmm) dmx = dpx; if (xmp) dpx = dmx; }
                double hs = vl_half(dmx, dpx);
                if (FL && xmc) { fup = rwx * ldsd(gwx, qb[p]); hs = 0.0; }
                const double X = fma(t, fma(t, fma(t, p3, p2), p1), p0) * ldsd(xm, mb[p]);
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
                if (SGN != 0 || pos) { r0 = ldsd(y0, qb[p]); r1 = ldsd(y1, qb[p]); r2 = ldsd(y2, qb[p]); }
                else { r0 = ldsd(y1, qb[p]); r1 = ldsd(y2, qb[p]); r2 = ldsd(y3, qb[p]); }
                double d1, d2, d3, ful, fuu;
                if (pos) { d1 = r1 - r0; d2 = own - r1; d3 = r2 - own; ful = r1; fuu = own; }     // rows j-2, j-1 | j+1
                else { d1 = own - r0; d2 = r1 - own; d3 = r2 - r1; ful = own; fuu = r1; }         // rows j-1 | j+1, j+2
                double dl1 = d1, dl2 = d2, du2 = d2, du3 = d3;
                if (FL) {                                            // AMB-13: one-sided slope next to a wall
                    if (pos) { if (wl2) dl1 = dl2; if (wl1) du2 = du3; if (wu1) du3 = du2; }      // lower: (j-2, j-1, j); upper: (j-1, j, j+1)
                    else { if (wl1) dl1 = dl2; if (wu1) dl2 = dl1; if (wu2) du3 = du2; }          // lower: (j-1, j, j+1); upper: (j, j+1, j+2)
                }
                double hl = vl_half(dl1, dl2), hu = vl_half(du2, du3);
                if (FL) {
                    if (pos && wl1) { ful = ylr[FR_RHOW] * ldsd(gwy0, qb[p]); hl = 0.0; }         // lower face is the ymin wall
                    if (!pos && wu1) { fuu = yur[FR_RHOW] * ldsd(gwy1, qb[p]); hu = 0.0; }        // upper face is the ymax wall
                }
                const bool useR = SGN == 0 && !pos;
                const double a1 = useR ? ql1n : ql1, a2 = useR ? ql2n : ql2, a3 = useR ? ql3n : ql3;
                const double b1 = useR ? qu1n : qu1, b2 = useR ? qu2n : qu2, b3 = useR ? qu3n : qu3;
                const double Xl = fma(n, fma(n, fma(n, a3, a2), a1), ql0) * ldsd(ylm, mb[p]);
                const double Xu = fma(n, fma(n, fma(n, b3, b2), b1), qu0) * ldsd(yum, mb[p]);
                const double Gl = fma(l4, ful, fma(fma(l5, n, sg * l4), hl, Xl));
                const double Gu = fma(u4, fuu, fma(fma(u5, n, sg * u4), hu, Xu));
                const double Dq = fma(n, Gl - Gu, Dx);
                const double g = fma(ldsd(cgp, mb[p]), gpu, ldsd(cgn, mb[p]) * gnu);
                const double fnw = fma(KF, own, fma(KD, Dq, g));     // P:L41 Eq. (3), solved for f^{n+1}
                if (valid[p]) *reinterpret_cast<double *>(out + qb[p]) = fnw;
            }
        };
        if (anyx || (anyy && have_cell)) body(std::true_type{}); else body(std::false_type{});
        __syncthreads();                                             // row a and stage a are consumed
    }
}

// SGN = +1 / -1 / 0: one sign class per launch; SGN = 2: both uniform classes in one launch, the CTA dispatches on its chunk's sign
// (twice the CTAs per launch on small meshes, and the two classes of a cell read its records while they are in the L2)
template <int NPT, int SGN, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_flux_update(const UgksParams P, const int cur, const int chunk0, const int nch)
{
    int b = blockIdx.x;
    const int j = b % P.J; b /= P.J;
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    const int s = b % nstrip, c = b / nstrip;                        // launch order: rows fastest, then strips, then chunks
    const int4 ch = P.chunks[chunk0 + c];
    if (SGN == 2) {
        if (ch.z > 0) flux_update_body<NPT, 1>(P, cur, ch, j, s);
        else flux_update_body<NPT, -1>(P, cur, ch, j, s);
    } else flux_update_body<NPT, SGN == 2 ? 1 : SGN>(P, cur, ch, j, s);
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32 + 32; }   // + producer warp

static size_t smem_fu(const UgksParams &P, int ny)
{
    const int Qb = pad2(P.cmax * P.Nu + 1), cmp = pad2(P.cmax + 1);
    const StageLayout L = stage_layout(ny, Qb, P.NuP, cmp);
    return ((size_t)NSX * Qb + 2 * (size_t)L.size) * sizeof(double) + (NSX + 2) * sizeof(uint64_t);
}
size_t smem_flux_update(const UgksParams &P) { return smem_fu(P, 4); }

template <int SGN, int MAXT, int MINB>
static void launch_sgn(const UgksParams &P, int cur, int chunk0, int nch, int grid, int threads, size_t smem, cudaStream_t st)
{
    switch (P.npt) {
#define CASE(N) case N: k_flux_update<N, SGN, MAXT, MINB><<<grid, threads, smem, st>>>(P, cur, chunk0, nch); break;
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
    if (threads <= 96) launch_sgn<SGN, 96, 4>(P, cur, chunk0, nch, grid, threads, smem, st);
    else if (threads <= 160) launch_sgn<SGN, 160, 3>(P, cur, chunk0, nch, grid, threads, smem, st);
    else launch_sgn<SGN, 288, 1>(P, cur, chunk0, nch, grid, threads, smem, st);
}

int launch_flux_update(const UgksParams &P, int cur, cudaStream_t st)
{
    // chunk order: [v < 0 ...][v > 0 ...][mixed ...]
    int n = 0;
    // small meshes: both uniform classes in one launch (fills the GPU); large meshes: one launch per class (measured 1-3 % faster)
    const long per_class = (long)P.J * ((P.I + P.strip - 1) / P.strip) * (P.nneg > P.npos ? P.nneg : P.npos);
    if (P.nneg && P.npos && per_class < 148L * 8) { launch_class<2>(P, cur, 0, P.nneg + P.npos, st); ++n; }
    else {
        if (P.nneg) { launch_class<-1>(P, cur, 0, P.nneg, st); ++n; }
        if (P.npos) { launch_class<1>(P, cur, P.nneg, P.npos, st); ++n; }
    }
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
    cudaError_t e = set_attr_all<SGN, 96, 4>(smem);
    if (e == cudaSuccess) e = set_attr_all<SGN, 160, 3>(smem);
    if (e == cudaSuccess) e = set_attr_all<SGN, 288, 1>(smem);
    return e;
}

int setup_update_attributes(const UgksParams &P)
{
    const int s3 = (int)smem_fu(P, 3), s4 = (int)smem_fu(P, 4);
    if (s4 > 227 * 1024) return 1;
    (void)s3;
    static bool done = false;                                        // per kernel, not per context: opt in to the device maximum once
    if (done) return 0;
    cudaError_t e = set_attr_sgn<2>(227 * 1024);
    if (e == cudaSuccess) e = set_attr_sgn<1>(227 * 1024);
    if (e == cudaSuccess) e = set_attr_sgn<-1>(227 * 1024);
    if (e == cudaSuccess) e = set_attr_sgn<0>(227 * 1024);
    done = e == cudaSuccess;
    return e == cudaSuccess ? 0 : 1;
}
