// ugks_jit_update.cuh -- k_flux_update: S6 + S8 at the four faces of every cell fused with the update U3
// (Eq. (3)); the per-face coefficients (S2..S5), the per-cell relaxation scalars (U1/U2) and every exponential
// come precomputed from k_face_scalars / k_cell_scalars / k_tables.  Compiled by NVRTC per context (ugks_jit_common.cuh).
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
//     together with the records of the step (face and cell coefficients, separable factors; whole records, one copy each).
//   * f^{n+1} is written straight from registers: f crosses HBM once each way in this kernel.
//   * option "tangential" (TG; NEXT-1, O3t/O8t): every face flux gets -ell Mt5 n t theta0, theta0 = the limited slope of the upwind
//     cell in the face's tangential direction.  Three more rows are staged per step -- the x-neighbours (c-1, jn), (c+1, jn) of
//     the upwind y-neighbour row jn and (c+1, jo) on the other side -- so that every slope is formed from explicitly staged rows;
//     the x-slope of the own cell is the x-face limiter result of this step (u > 0) or of the previous one (u < 0).
//   * there is no producer warp: after the barrier that ends step a, one lane of warp (a mod W) issues the 8 bulk copies of
//     step a+2 / row a+3 (with compile-time geometry that is a few dozen instructions), so every resident warp computes and
//     no warp's registers idle.
#pragma once
#include "ugks_jit_common.cuh"

constexpr int NSX = 3;                                               // x-ring slots: rows a, a+1 live, a+2 in flight
// Record slices: a chunk needs, of the separable factors over v (E_m[Nv] of a face record, g_v^n[Nv], g_v^{n+1}[Nv] of a cell record),
// only its own rows.  With SLICE the stage holds [coefficients | factors over u | rows m0a .. m0a + MSL) of the factors over v]
// (m0a = m0 rounded down to even: bulk copies start 16-byte aligned), two / three bulk copies per record instead of one: on wide
// velocity grids (C5: 5 of 200 rows per chunk) the whole records are twice the bytes of the chunk's f rows.
constexpr bool SLICE = G_SLICE != 0;
constexpr int MSL = pad2c(MC + 1);                                   // staged rows of a factor table over v
constexpr int FRSS = SLICE ? FR_NCOEF + NUP + MSL : FRS, CRSS = SLICE ? CR_NCOEF + 2 * NUP + 2 * MSL : CRS;
constexpr int VTS = SLICE ? MSL : NVP;                               // stride between the two v-tables of a staged cell record

template <int NY>
struct StageL {                                                      // offsets in doubles inside one step stage
    static constexpr int yrow = 0;
    static constexpr int xrec = yrow + NY * QB;
    static constexpr int ylrec = xrec + FRSS;
    static constexpr int yurec = ylrec + FRSS;
    static constexpr int crec = yurec + FRSS;
    static constexpr int size = crec + CRSS;
    static constexpr int BYTES = (NSX * QB + 2 * size) * 8 + (NSX + 2) * 8;
};

template <int SGN>
__device__ __forceinline__ void flux_update_body(const KArgs &A, const int4 ch, const int j, const int s)
{
    constexpr int NY = SGN == 0 ? 4 : (TG ? 6 : 3);
    using L = StageL<NY>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // every CTA marches exactly STRIP cells (a compile-time trip count): the last strip of a row that STRIP does not divide
    // starts at GI - STRIP and re-computes a few cells of its neighbour (same inputs, same arithmetic, same bits)
    const int c0 = min(s * STRIP, GI - STRIP), c1 = c0 + STRIP;      // cells [c0, c1) of row j
    const int m0 = ch.x, mc = ch.y;
    const int q0 = m0 * NU, qa = q0 & ~1, qsh = q0 - qa;
    const uint32_t bytes = (uint32_t)(pad2c(mc * NU + qsh) * 8);
    const int m0a = m0 & ~1, msh = m0 - m0a;                         // SLICE: first staged row of the v-tables, shift of the chunk inside
    const uint32_t sbytes = (uint32_t)(pad2c(mc + msh) * 8);
    const uint32_t fbytes = SLICE ? (FR_NCOEF + NUP) * 8 + sbytes : FRS * 8, cbytes = SLICE ? (CR_NCOEF + 2 * NUP) * 8 + 2 * sbytes : CRS * 8;
    // whole record, or its head and the chunk's rows of its v-tables
    auto copy_frec = [&](double *dst, const double *src, uint64_t *bar) {
        if constexpr (!SLICE) tma_load_1d(dst, src, FRS * 8, bar);
        else {
            tma_load_1d(dst, src, (FR_NCOEF + NUP) * 8, bar);
            tma_load_1d(dst + FR_NCOEF + NUP, src + FR_NCOEF + NUP + m0a, sbytes, bar);
        }
    };
    auto copy_crec = [&](double *dst, const double *src, uint64_t *bar) {
        if constexpr (!SLICE) tma_load_1d(dst, src, CRS * 8, bar);
        else {
            tma_load_1d(dst, src, (CR_NCOEF + 2 * NUP) * 8, bar);
            tma_load_1d(dst + CR_NCOEF + 2 * NUP, src + CR_NCOEF + 2 * NUP + m0a, sbytes, bar);
            tma_load_1d(dst + CR_NCOEF + 2 * NUP + MSL, src + CR_NCOEF + 2 * NUP + NVP + m0a, sbytes, bar);
        }
    };

    double *ring = reinterpret_cast<double *>(smem_raw);             // [NSX][QB]
    double *stages = ring + NSX * QB;                                // [2][L::size]
    uint64_t *bars = reinterpret_cast<uint64_t *>(stages + 2 * L::size);   // [NSX] x rows, [2] stages

    const int tid = threadIdx.x;
    const bool active = tid < NU * R;
    const int k = active ? tid % NU : 0, r = active ? tid / NU : 0;
    const double *fcur = A.fcur;
    const int rows_first = c0 - 2, rows_last = c1 + 1;
    // ---- bulk copies (issued by one elected lane): global sources of a step are linear in the cell index
    constexpr int DJ0 = SGN == 0 ? -2 : (SGN > 0 ? -2 : -1), DJ1 = SGN == 0 ? -1 : (SGN > 0 ? -1 : 1), DJ2 = SGN == 0 ? 1 : (SGN > 0 ? 1 : 2);
    auto issue_x = [&](int row) {
        const int sl = (row - rows_first) % NSX;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(ring + sl * QB, xrow_ptr(fcur, A.ghost, row, j) + qa, bytes, &bars[sl]);
    };
    // stage of step st: record of x-face st and, for cell st-1, its y-neighbour rows, y-face records and cell record
    auto issue_stage = [&](int st) {
        const int sl = (st - c0) & 1;
        double *S = stages + sl * L::size;
        uint64_t *bar = &bars[NSX + sl];
        const bool have_cell = st > c0;
        if constexpr (TG) {
            // rows relative to c = st - 1 (also for st = c0: x-face c0 needs the y-slope of its upwind cell c0-1 or c0):
            // 0..2 as without TG; 3 = (c-1, jn), 4 = (c+1, jn), 5 = (c+1, jo) with jn the upwind y-neighbour row of the chunk's sign
            constexpr int JN = SGN > 0 ? -1 : 1, JO = -JN;
            const int c = st - 1;
            mbar_expect_tx(bar, fbytes + 6 * bytes + (have_cell ? 2 * fbytes + cbytes : 0));
            copy_frec(S + L::xrec, A.frec0 + ((size_t)j * (GI + 1) + st) * FRS, bar);
            tma_load_1d(S + L::yrow, cell_row_ptr(fcur, A.ghost, c, j + DJ0) + qa, bytes, bar);
            tma_load_1d(S + L::yrow + QB, cell_row_ptr(fcur, A.ghost, c, j + DJ1) + qa, bytes, bar);
            tma_load_1d(S + L::yrow + 2 * QB, cell_row_ptr(fcur, A.ghost, c, j + DJ2) + qa, bytes, bar);
            tma_load_1d(S + L::yrow + 3 * QB, cell_row_ptr(fcur, A.ghost, c - 1, j + JN) + qa, bytes, bar);
            tma_load_1d(S + L::yrow + 4 * QB, cell_row_ptr(fcur, A.ghost, c + 1, j + JN) + qa, bytes, bar);
            tma_load_1d(S + L::yrow + 5 * QB, cell_row_ptr(fcur, A.ghost, c + 1, j + JO) + qa, bytes, bar);
            if (have_cell) {
                const double *yl = A.frec1 + ((size_t)j * GI + c) * FRS;
                copy_frec(S + L::ylrec, yl, bar);
                copy_frec(S + L::yurec, yl + (size_t)GI * FRS, bar);
                copy_crec(S + L::crec, A.crec + ((size_t)j * GI + c) * CRS, bar);
            }
            return;
        }
        mbar_expect_tx(bar, fbytes + (have_cell ? NY * bytes + 2 * fbytes + cbytes : 0));
        copy_frec(S + L::xrec, A.frec0 + ((size_t)j * (GI + 1) + st) * FRS, bar);
        if (have_cell) {
            const size_t cell = st - 1;
            int yst;
            const double *y0p = yrow_base(fcur, A.ghost, j + DJ0, &yst) + qa;
            tma_load_1d(S + L::yrow, y0p + cell * yst, bytes, bar);
            const double *y1p = yrow_base(fcur, A.ghost, j + DJ1, &yst) + qa;
            tma_load_1d(S + L::yrow + QB, y1p + cell * yst, bytes, bar);
            const double *y2p = yrow_base(fcur, A.ghost, j + DJ2, &yst) + qa;
            tma_load_1d(S + L::yrow + 2 * QB, y2p + cell * yst, bytes, bar);
            if (NY == 4) {
                const double *y3p = yrow_base(fcur, A.ghost, j + 2, &yst) + qa;
                tma_load_1d(S + L::yrow + 3 * QB, y3p + cell * yst, bytes, bar);
            }
            const double *yl = A.frec1 + ((size_t)j * GI + cell) * FRS;
            copy_frec(S + L::ylrec, yl, bar);
            copy_frec(S + L::yurec, yl + (size_t)GI * FRS, bar);
            copy_crec(S + L::crec, A.crec + ((size_t)j * GI + cell) * CRS, bar);
        }
    };
    if (tid == 0) {
        for (int i = 0; i < NSX + 2; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
        for (int row = rows_first; row < rows_first + NSX; ++row) issue_x(row);
        issue_stage(c0);
        issue_stage(c0 + 1);
    }
    __syncthreads();                                                 // barriers initialised

    const double uk = c_u[k];
    const bool posx = uk > 0.0;
    const double sgx = posx ? 1.0 : -1.0;
    // Per-thread points p: velocity row m = r + p R; byte offsets are thread base + immediates.  A point outside the chunk
    // (the last point when R*NPT > MC, the tail of a ragged chunk) re-reads the chunk's first element; only its store is masked.
    constexpr int QSTEP = R * NU * 8, MSTEP = R * 8;
    const int mfirst = (SLICE ? msh : m0) * 8;                       // byte offset of the chunk's first row in a staged v-table
    const int qb0 = (qsh + r * NU + k) * 8, mb0 = mfirst + r * 8;
    int qo[NPT], mo[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) { qo[p] = r + p * R < mc ? p * QSTEP : qsh * 8 - qb0; mo[p] = r + p * R < mc ? p * MSTEP : mfirst - mb0; }
#define QOFF(p) ((G_RAGGED == 0 && ((p) + 1) * R <= MC) ? (p) * QSTEP : qo[p])
#define MOFF(p) ((G_RAGGED == 0 && ((p) + 1) * R <= MC) ? (p) * MSTEP : mo[p])
    double vn[NPT], fm[NPT], fc[NPT], Fprev[NPT];
    double hsp[TG ? NPT : 1];                                        // TG: x-face limiter result of the previous step (x-slope of the own cell for u < 0)
    bool valid[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        valid[p] = active && mm < mc;
        vn[p] = c_v[m0 + (mm < mc ? mm : 0)];
        Fprev[p] = 0.0;
        if (TG) hsp[TG ? p : 0] = 0.0;
    }
    const unsigned char *ring_b = reinterpret_cast<const unsigned char *>(ring) + qb0;
    const unsigned char *stages_b = reinterpret_cast<const unsigned char *>(stages);
    const int kb = k * 8;
    {   // prologue: the two oldest rows of each thread's x-window go to registers
        mbar_wait(&bars[0], 0); mbar_wait(&bars[1], 0); mbar_wait(&bars[2], 0);
        const unsigned char *ra = ring_b + (posx ? 0 : 1) * QBB, *rb = ra + QBB;
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fm[p] = ldsd(ra, QOFF(p)); fc[p] = ldsd(rb, QOFF(p)); }
    }
    __syncthreads();                                                 // rows c0-2, c0-1 consumed
    if (tid == 0) { issue_x(c0 + 1); issue_x(c0 + 2); }
    // wall flags of the two y-faces (CTA-uniform)
    const bool wl2 = beyond_wall_y(j - 2), wl1 = beyond_wall_y(j - 1), wu1 = beyond_wall_y(j + 1), wu2 = beyond_wall_y(j + 2);
    const bool anyy = wl2 || wl1 || wu1 || wu2;
    const unsigned char *gwy0 = reinterpret_cast<const unsigned char *>(A.wallg + 2 * NPAD + qa) + qb0;
    const unsigned char *gwy1 = reinterpret_cast<const unsigned char *>(A.wallg + 3 * NPAD + qa) + qb0;
    const unsigned char *gwx = reinterpret_cast<const unsigned char *>(A.wallg + (posx ? 0 : 1) * NPAD + qa) + qb0;
    const int sh = posx ? 0 : 1;
    unsigned char *out_row = reinterpret_cast<unsigned char *>(A.fnew + (size_t)j * GI * NPAD + qa) + qb0;

    int xslot_new = sh;                                              // ring slot of row a + sh  (a = c0: index c0 + sh - rows_first = 2 + sh)
    xslot_new = (2 + sh) % NSX;
    int xw_slot = 0, xw_phase = 1;                                   // barrier slot / phase of row a+1 (index a+1-rows_first = 3 at a = c0)
    int stage_i = 0, stage_phase = 0;
    int issuer = 0;                                                  // thread that issues the bulk copies after this step (lane 0 of a rotating warp)
    // measured: C4 (160 threads) -10 % (the ring / stage parities and half of the register rotation fold away), C5 0; CTAs of
    // 64-96 threads (C3, M4-69) +3 %, short strips +10 %
    constexpr int UNROLL_U = (STRIP >= 16 && NU * R >= 128) ? 2 : 1;
    // one step: x-face a, then cell a-1.  The first step of a march (a = c0) has no cell to finish: it is peeled off (HC = false) so
    // that the steady-state body carries no "have a cell" branch between its points and the points of a thread form one basic block
    // (the independent FP64 chains of the NPT points can then be interleaved by the scheduler)
    auto step = [&](const int a, auto hc) {
        constexpr bool have_cell = decltype(hc)::value;
        const unsigned char *S = stages_b + stage_i * (L::size * 8);
        mbar_wait(&bars[NSX + stage_i], stage_phase);
        if (stage_i) stage_phase ^= 1;
        stage_i ^= 1;
        mbar_wait(&bars[xw_slot], xw_phase);                         // row a+1
        if (++xw_slot == NSX) { xw_slot = 0; xw_phase ^= 1; }
        // ---- x-face a: polynomial column of this thread (n = u_k; cubic in t = v_m)
        const double *xr = reinterpret_cast<const double *>(S + L::xrec * 8);
        const double *xlr = xr + (posx ? FR_L : FR_R);
        const double Ek = uk * ldsd(S + (L::xrec + FR_NCOEF) * 8, kb);
        const double p0 = Ek * fma(uk, fma(uk, fma(uk, xlr[LR_C30], xlr[LR_C20]), xlr[LR_C10]), xr[FR_C00]);
        const double p1 = Ek * fma(uk, fma(uk, xr[FR_C21], xlr[LR_C11]), xr[FR_C01]);
        const double p2 = Ek * fma(uk, xlr[LR_C12], xr[FR_C02]);
        const double p3 = Ek * xr[FR_C03];
        const double c4 = uk * xr[FR_MT4];
        const double c45 = uk * fma(uk, xr[FR_MT5], sgx * xr[FR_MT4]);
        const double cx6 = TG ? uk * xr[FR_MT5T] : 0.0;              // O8t: -ell Mt5 n t theta0 on the x-face, per unit of t (h_y theta0)
        const unsigned char *xm = S + (L::xrec + FR_NCOEF + NUP) * 8 + mb0;
        const unsigned char *rn = ring_b + xslot_new * QBB;
        if (++xslot_new == NSX) xslot_new = 0;
        bool xw0 = false, xw1 = false, xw2 = false, xw3 = false;
        if (a < 2 || a + 2 > GI) { xw0 = beyond_wall_x(a - 2); xw1 = beyond_wall_x(a - 1); xw2 = beyond_wall_x(a); xw3 = beyond_wall_x(a + 1); }
        const bool anyx = xw0 || xw1 || xw2 || xw3;
        // ---- y-faces of cell a-1: polynomial columns (t = u_k; cubic in n = v_m), L (n > 0) / R (n < 0) variants
        const double *ylr = reinterpret_cast<const double *>(S + L::ylrec * 8), *yur = reinterpret_cast<const double *>(S + L::yurec * 8);
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
            const double El = ldsd(S + (L::ylrec + FR_NCOEF) * 8, kb), Eu = ldsd(S + (L::yurec + FR_NCOEF) * 8, kb);
            ycol(ylr, ylr + (SGN >= 0 ? FR_L : FR_R), El, ql0, ql1, ql2, ql3, true);
            ycol(yur, yur + (SGN >= 0 ? FR_L : FR_R), Eu, qu0, qu1, qu2, qu3, true);
            if (SGN == 0) {
                double dummy;
                ycol(ylr, ylr + FR_R, El, dummy, ql1n, ql2n, ql3n, false);
                ycol(yur, yur + FR_R, Eu, dummy, qu1n, qu2n, qu3n, false);
            }
            const double *cr = reinterpret_cast<const double *>(S + L::crec * 8);
            gnu = ldsd(S + (L::crec + CR_NCOEF) * 8, kb); gpu = ldsd(S + (L::crec + CR_NCOEF + NUP) * 8, kb);
            KF = cr[CR_KF]; KD = cr[CR_KD];
            l4 = ylr[FR_MT4]; l5 = ylr[FR_MT5]; u4 = yur[FR_MT4]; u5 = yur[FR_MT5];
        }
        // O8t on the y-faces of the own cell: t = u_k, so the coefficient of (h_x theta0) is per thread and face
        const double cl6 = (TG && have_cell) ? uk * ylr[FR_MT5T] : 0.0, cu6 = (TG && have_cell) ? uk * yur[FR_MT5T] : 0.0;
        const unsigned char *y0 = S + L::yrow * 8 + qb0, *y1 = y0 + QBB, *y2 = y1 + QBB, *y3 = y2 + QBB;
        // TG rows: y3 = (c-1, jn), y4 = (c+1, jn), y5 = (c+1, jo); the y-neighbours (j-1, j+1) of the x-face's upwind cell are
        // (y1, y2) / (y0, y1) of the own column for u > 0 and (y4, y5) / (y5, y4) of column c+1 for u < 0 (v > 0 / v < 0 chunks)
        const unsigned char *y4 = y3 + QBB, *y5 = y4 + QBB;
        const unsigned char *tlo = posx ? (SGN > 0 ? y1 : y0) : (SGN > 0 ? y4 : y5), *thi = posx ? (SGN > 0 ? y2 : y1) : (SGN > 0 ? y5 : y4);
        const int cown = a - 1;
        const bool cm_miss = TG && cown == 0 && BCX0 == BC_WALL, cp_miss = TG && cown == GI - 1 && BCX1 == BC_WALL;
        const bool nb_ghost = TG && (SGN > 0 ? (j - 1 < 0 && BCY0 == BC_FIXED) : (j + 1 >= GJ && BCY1 == BC_FIXED));
        const bool tgb = TG && (a < 2 || a + 2 > GI || j < 1 || j > GJ - 2);      // near a boundary: take the flagged body
        const unsigned char *ylm = S + (L::ylrec + FR_NCOEF + NUP) * 8 + mb0, *yum = S + (L::yurec + FR_NCOEF + NUP) * 8 + mb0;
        const unsigned char *cgn = S + (L::crec + CR_NCOEF + 2 * NUP) * 8 + mb0, *cgp = cgn + VTS * 8;
        unsigned char *out = out_row + (size_t)max(a - 1, 0) * (NPAD * 8);

        auto body = [&](auto fl) {                                   // fl: some stencil of this step touches a wall
            constexpr bool FL = decltype(fl)::value;
            // wall flags of this thread's x-window (cells a-2+sh, a-1+sh, a+sh)
            const bool xmm = FL && (sh ? xw1 : xw0), xmc = FL && (sh ? xw2 : xw1), xmp = FL && (sh ? xw3 : xw2);
            const double rwx = FL ? xr[FR_RHOW] : 0.0;
#pragma unroll
            for (int p = 0; p < NPT; ++p) {
                const double fn = ldsd(rn, QOFF(p)), t = vn[p];
                // x-face a (upwind cell = middle of the window)
                double dmx = fc[p] - fm[p], dpx = fn - fc[p], fup = fc[p];
                if (FL) { if (xmm) dmx = dpx; if (xmp) dpx = dmx; }
                double hs = vl_half(dmx, dpx);
                if (FL && xmc) { fup = rwx * ldsd(gwx, QOFF(p)); hs = 0.0; }
                const double X = fma(t, fma(t, fma(t, p3, p2), p1), p0) * ldsd(xm, MOFF(p));
                double F = fma(c4, fup, fma(c45, hs, X));
                double hown = 0.0;                                   // TG: h_x sigma_x of the own cell a-1
                if constexpr (TG) {
                    // tangential slope on the x-face: limited y-slope of its upwind cell (value fc, y-neighbours tlo / thi)
                    double dlo = fc[p] - ldsd(tlo, QOFF(p)), dhi = ldsd(thi, QOFF(p)) - fc[p];
                    if (FL) { if (wl1) dlo = dhi; if (wu1) dhi = dlo; }
                    const double hty = vl_half(dlo, dhi);
                    F = fma(cx6 * t, hty, F);
                    hown = posx ? hs : hsp[p];
                    hsp[p] = hs;
                }
                const double Dx = Fprev[p] - F;
                Fprev[p] = F;
                const double own = posx ? fc[p] : fm[p];             // row of cell a-1
                fm[p] = fc[p]; fc[p] = fn;
                if constexpr (!have_cell) continue;
                // y-faces of cell a-1: G = F / n
                const double n = t;
                const bool pos = SGN > 0 || (SGN == 0 && n > 0.0);
                const double sg = pos ? 1.0 : -1.0;
                double r0, r1, r2;                                   // the three neighbour rows of this point's stencil
                if (SGN != 0 || pos) { r0 = ldsd(y0, QOFF(p)); r1 = ldsd(y1, QOFF(p)); r2 = ldsd(y2, QOFF(p)); }
                else { r0 = ldsd(y1, QOFF(p)); r1 = ldsd(y2, QOFF(p)); r2 = ldsd(y3, QOFF(p)); }
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
                    if (pos && wl1) { ful = ylr[FR_RHOW] * ldsd(gwy0, QOFF(p)); hl = 0.0; }     // lower face is the ymin wall
                    if (!pos && wu1) { fuu = yur[FR_RHOW] * ldsd(gwy1, QOFF(p)); hu = 0.0; }    // upper face is the ymax wall
                }
                const bool useR = SGN == 0 && !pos;
                const double a1 = useR ? ql1n : ql1, a2 = useR ? ql2n : ql2, a3 = useR ? ql3n : ql3;
                const double b1 = useR ? qu1n : qu1, b2 = useR ? qu2n : qu2, b3 = useR ? qu3n : qu3;
                const double Xl = fma(n, fma(n, fma(n, a3, a2), a1), ql0) * ldsd(ylm, MOFF(p));
                const double Xu = fma(n, fma(n, fma(n, b3, b2), b1), qu0) * ldsd(yum, MOFF(p));
                double Gl = fma(l4, ful, fma(fma(l5, n, sg * l4), hl, Xl));
                double Gu = fma(u4, fuu, fma(fma(u5, n, sg * u4), hu, Xu));
                if constexpr (TG) {
                    // tangential slopes on the y-faces: x-slope of the upwind neighbour cell (c, jn) from its staged x-neighbours,
                    // and the own cell's x-slope
                    double dlo = r1 - ldsd(y3, QOFF(p)), dhi = ldsd(y4, QOFF(p)) - r1;
                    if (FL) { if (cm_miss) dlo = dhi; if (cp_miss) dhi = dlo; }
                    double hnb = vl_half(dlo, dhi);
                    if (FL && nb_ghost) hnb = 0.0;                   // a ghost cell has no slope (O1)
                    Gl = fma(cl6, SGN > 0 ? hnb : hown, Gl);
                    Gu = fma(cu6, SGN > 0 ? hown : hnb, Gu);
                }
                const double Dq = fma(n, Gl - Gu, Dx);
                const double g = fma(ldsd(cgp, MOFF(p)), gpu, ldsd(cgn, MOFF(p)) * gnu);
                const double fnw = fma(KF, own, fma(KD, Dq, g));     // P:L41 Eq. (3), solved for f^{n+1}
                if (valid[p]) *reinterpret_cast<double *>(out + p * QSTEP) = fnw;
            }
        };
        if (anyx || (anyy && have_cell) || tgb) body(true_c{}); else body(false_c{});
        __syncthreads();                                             // row a and stage a are consumed
        if (tid == issuer) {                                         // one lane of warp (a - c0) mod W issues the copies of two steps ahead
            if (a + 3 <= rows_last) issue_x(a + 3);
            if (a + 2 <= c1) issue_stage(a + 2);
        }
        issuer += 32;
        if (issuer >= BT) issuer = 0;
    };
    step(c0, false_c{});
#pragma unroll UNROLL_U
    for (int a = c0 + 1; a <= c1; ++a) step(a, true_c{});
}

static_assert(StageL<TG ? 6 : 3>::BYTES == G_SMEM_UPD3 && StageL<4>::BYTES == G_SMEM_UPD4, "host mirror of the shared-memory layout (ugks_jit.cu) disagrees");
#if G_NMIX > 0
static_assert(!TG, "the tangential reconstruction needs sorted velocity nodes (no mixed-sign chunks)");
#endif

// one launch covers the chunk range [chunk0, chunk0 + nch): the CTA dispatches on the sign class of its chunk (the two uniform
// classes of a cell read its records while they are in the L2)
extern "C" __global__ void __launch_bounds__(BT, G_MINB_UPD) k_flux_update(const KArgs A, const int chunk0)
{
    int b = blockIdx.x;
    const int j = b % GJ; b /= GJ;
    const int s = b % NSTRIP, c = b / NSTRIP;                        // rows fastest, then strips, then chunks
    const int4 ch = c_chunks[chunk0 + c];
    if (ch.z > 0) flux_update_body<1>(A, ch, j, s);
    else if (ch.z < 0) flux_update_body<-1>(A, ch, j, s);
#if G_NMIX > 0
    else flux_update_body<0>(A, ch, j, s);
#endif
}
