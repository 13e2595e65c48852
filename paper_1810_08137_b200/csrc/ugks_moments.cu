// ugks_moments.cu -- k_cell_moments: reconstruction (R) and the velocity-space reductions of S1 and S7
// ("12 times parallel reduction"), written cell by cell.
//
// The upwind face state of O3 is f0 = f_c + h sigma_c on the plus-side face of cell c where n > 0 and f_c - h sigma_c on
// its minus-side face where n < 0, so every face sum splits into a part owned by the left cell and a part owned by the
// right cell.  One pass over the cells therefore serves the x- and the y-faces: per cell and direction ONE limiter
// evaluation per velocity point, from the centred stencil (c-1, c, c+1), and f is read from HBM once.
//
// One CTA marches along a strip of cells of row j for one chunk of velocity rows (all v_m of one sign where the grid
// allows, so that the y-side of a point is CTA-uniform).  Thread (k, r) owns velocity column k and the rows m = r + p*R.
//   * x-stencil: (f_c, f_c - f_{c-1}) live in registers; ONE new row per cell comes from a 3-slot shared-memory ring fed by
//     1-D TMA bulk copies (cp.async.bulk + mbarrier).  y-neighbours (i, j-1), (i, j+1): TMA-staged, double-buffered.
//   * sums are tensor products: a thread accumulates sum_m wv v^p (.) for its column (13 sums; the weights wv v^p come as
//     broadcast shared-memory loads).  Four pipelined stages, one per cell step and one barrier per step, finish the
//     reduction: (1) partial sums to shared memory; (2) sum over the R threads of a column, forming C_b +- B_b for the two
//     x-sides; (3) balanced work items (output, k-range): dot product over k with the factors wu u^a H(+-u);
//     (4) one thread per output adds its items and stores.
#include "ugks_common.cuh"
#include <type_traits>

constexpr int NSXM = 3;                                              // x-ring slots
constexpr int NFAC = 13;                                             // factor tables: 5 (x+), 5 (x-), 3 (y)
// raw sum idx -> (power of the per-column velocity, column sum) ; x sets: columns 0..2 = C_b +- B_b, 3..5 = B_b
__constant__ int c_xa[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 2, 3, 4, 2, 2 };
__constant__ int c_xc[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 3, 3, 3, 4, 5 };
__constant__ int c_yt[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 0, 0, 0, 1, 2 };   // y sets: columns A_0..A_3, B_2..B_4
__constant__ int c_yc[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 4, 5, 6, 4, 4 };

struct MomLayout {                                                   // shared-memory carve-up (offsets in doubles)
    int ybuf, part, col, fac, mtab, ires, desc, odesc, bars, NuS, nitem, bytes;
};
__host__ __device__ inline MomLayout mom_layout(bool mixed, int Nu, int cmax, int R, int npt, int B, int nsx, int nsy)
{
    const int NA = mixed ? 20 : 13, NC = mixed ? 23 : 16, NOUT = mixed ? 4 * NRAW : 3 * NRAW;
    const int Qb = pad2(cmax * Nu + 1), nrow = R * npt + 1;
    MomLayout L;
    L.NuS = Nu | 1;                                                  // odd column stride: conflict-free across columns
    L.nitem = 2 * NRAW * nsx + (mixed ? 2 : 1) * NRAW * nsy;
    int o = NSXM * Qb;
    L.ybuf = o; o += 4 * Qb;
    L.part = o; o += R == 1 ? 0 : 2 * NA * B;                        // R = 1: a thread owns its column, stage 1 writes the columns
    L.col = o; o += pad2(2 * NC * L.NuS);
    L.fac = o; o += pad2(NFAC * L.NuS);
    L.mtab = o; o += pad2(nrow * 6);
    L.ires = o; o += pad2(2 * L.nitem);
    L.desc = o; o += 2 * L.nitem;                                    // int4 per item
    L.odesc = o; o += 2 * NOUT;                                      // int4 per output
    L.bars = o; o += NSXM + 2;
    L.bytes = o * 8;
    return L;
}

template <int NPT, bool MIXED, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_cell_moments(const UgksParams P, const int cur, const int chunk0)
{
    constexpr int NA = MIXED ? 20 : 13;                              // per-thread sums: 6 (x) + 7 (y) [+ 7 (y-)]
    constexpr int NC = MIXED ? 23 : 16;                              // columns after stage 2: 9 (x) + 7 (y) [+ 7]
    constexpr int NOUT = MIXED ? 4 * NRAW : 3 * NRAW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    int b = blockIdx.x;
    const int j = b % P.J; b /= P.J;
    const int s = b % nstrip;
    const int chunk = chunk0 + b / nstrip;                           // chunks are sorted: [v < 0][v > 0][mixed]
    const int4 ch = P.chunks[chunk];
    const int c0 = s * P.strip, c1 = min(c0 + P.strip, P.I);         // cells [c0, c1)
    const int m0 = ch.x, mc = ch.y;
    const int Nu = P.Nu, R = P.R;
    const int q0 = m0 * Nu, qa = q0 & ~1, qsh = q0 - qa;             // 16-byte aligned copy start; shift of the chunk inside
    const int Qb = pad2(P.cmax * Nu + 1), QbB = Qb * 8;
    const uint32_t bytes = (uint32_t)(pad2(mc * Nu + qsh) * sizeof(double));
    const int B = blockDim.x - 32;                                   // compute threads; the last warp is the TMA producer
    const int nrow = R * NPT + 1;                                    // weight rows incl. a zero row
    const MomLayout L = mom_layout(MIXED, Nu, P.cmax, R, NPT, B, P.s3_nsx, P.s3_nsy);
    const int NuS = L.NuS, nitem = L.nitem;

    double *sm = reinterpret_cast<double *>(smem_raw);
    double *xring = sm;                                              // [NSXM][Qb]
    double *ybuf = sm + L.ybuf;                                      // [2][2][Qb]
    double *part = sm + L.part;                                      // [2][NA][B]
    double *col = sm + L.col;                                        // [2][NC][NuS]
    double *fac = sm + L.fac;                                        // [NFAC][NuS]
    double *mtab = sm + L.mtab;                                      // [nrow][6]: w, w v, w v^2, w v^3, w v^4, H(v)
    double *ires = sm + L.ires;                                      // [2][nitem] stage-3 item results
    int4 *desc = reinterpret_cast<int4 *>(sm + L.desc);              // [nitem]  (fac offset, col offset, k begin, k end)
    int4 *odesc = reinterpret_cast<int4 *>(sm + L.odesc);            // [NOUT]   (first item, items, set*NRAW+idx, 0)
    uint64_t *bars = reinterpret_cast<uint64_t *>(sm + L.bars);      // [NSXM] x rows, [2] y stages

    const int tid = threadIdx.x;
    const bool active = tid < Nu * R;
    const int k = active ? tid % Nu : 0, r = active ? tid / Nu : 0;
    const double *fcur = P.f[cur];
    const int rows_first = c0 - 1, rows_last = c1;                   // cells c0-1 .. c1 are staged
    int ystm, ystp;
    const double *ybm = yrow_base(P, fcur, j - 1, &ystm) + qa, *ybp = yrow_base(P, fcur, j + 1, &ystp) + qa;

    auto issue_x = [&](int row) {
        const int sl = (row - rows_first) % NSXM;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(xring + (size_t)sl * Qb, row_ptr<0>(P, fcur, row, j) + qa, bytes, &bars[sl]);
    };
    auto wait_x = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSXM], (idx / NSXM) & 1);
    };
    auto issue_y = [&](int cell) {
        const int buf = (cell - c0) & 1;
        mbar_expect_tx(&bars[NSXM + buf], 2 * bytes);
        tma_load_1d(ybuf + (size_t)(buf * 2) * Qb, ybm + (size_t)cell * ystm, bytes, &bars[NSXM + buf]);
        tma_load_1d(ybuf + (size_t)(buf * 2 + 1) * Qb, ybp + (size_t)cell * ystp, bytes, &bars[NSXM + buf]);
    };

    if (tid == 0) {
        for (int i = 0; i < NSXM + 2; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    if (tid >= B) {                                                  // ---- producer warp: one lane issues every bulk copy
        const bool lead = tid == B;
        __syncthreads();                                             // barriers initialised, tables written
        if (lead) {
            for (int row = rows_first; row < rows_first + NSXM && row <= rows_last; ++row) issue_x(row);
            issue_y(c0);
            if (c0 + 1 < c1) issue_y(c0 + 1);
        }
        __syncthreads();                                             // rows c0-1, c0 consumed
        if (lead) {
            if (c0 + 2 <= rows_last) issue_x(c0 + 2);
            if (c0 + 3 <= rows_last) issue_x(c0 + 3);
        }
        for (int a = c0; a < c1 + 3; ++a) {
            __syncthreads();                                         // step a done: row a+1 and y stage a are free
            if (lead && a < c1) {
                if (a + 4 <= rows_last) issue_x(a + 4);
                if (a + 2 < c1) issue_y(a + 2);
            }
        }
        return;
    }
    for (int i = tid; i < Nu; i += B) {
        const double u = P.u[i], w = P.wu[i];
        const double hp = u > 0.0 ? 1.0 : (u < 0.0 ? 0.0 : 0.5);
        double pw = 1.0;
        for (int a = 0; a < 5; ++a) {
            fac[a * NuS + i] = w * hp * pw;
            fac[(5 + a) * NuS + i] = w * (1.0 - hp) * pw;
            if (a < 3) fac[(10 + a) * NuS + i] = w * pw;
            pw *= u;
        }
    }
    for (int i = tid; i < nrow; i += B) {
        const bool in = i < mc;
        const double v = in ? P.v[m0 + i] : 0.0, w = in ? P.wv[m0 + i] : 0.0;
        double *o = mtab + i * 6;
        o[0] = w; o[1] = w * v; o[2] = w * v * v; o[3] = w * v * v * v; o[4] = w * v * v * v * v;
        o[5] = v > 0.0 ? 1.0 : (v < 0.0 ? 0.0 : 0.5);
    }
    // stage-3 work items: output v = (set, idx) split into ns parts of its k-range; x+ sums u_k >= 0, x- sums u_k <= 0
    for (int v = tid; v < NOUT; v += B) {
        int set = v / NRAW;
        const int idx = v % NRAW;
        int fi, ci, kb, ke, ns, first;
        if (set < 2) {
            const int c = c_xc[idx];
            fi = (set == 0 ? 0 : 5) + c_xa[idx];
            ci = c < 3 ? (set == 0 ? c : 3 + c) : 3 + c;             // columns: 0..2 C+B, 3..5 C-B, 6..8 B
            kb = set == 0 ? P.kxp_begin : 0; ke = set == 0 ? Nu : P.kxm_end;
            ns = P.s3_nsx; first = v * ns;
        } else {
            fi = 10 + c_yt[idx];
            ci = 9 + (set - 2) * 7 + c_yc[idx];
            kb = 0; ke = Nu;
            ns = P.s3_nsy; first = 2 * NRAW * P.s3_nsx + (v - 2 * NRAW) * ns;
            if (!MIXED) set = ch.z > 0 ? 2 : 3;
        }
        const int len = ke - kb, per = (len + ns - 1) / ns;
        for (int h = 0; h < ns; ++h)
            desc[first + h] = make_int4(fi * NuS * 8, ci * NuS * 8, min(kb + h * per, ke), min(kb + (h + 1) * per, ke));
        odesc[v] = make_int4(first, ns, set * NRAW + idx, 0);
    }
    __syncthreads();

    // per-thread points (byte offsets); a point outside the chunk (ragged tail, padding threads) reads a valid value and
    // the zero weight row
    int qb[NPT], wb[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        const bool valid = active && mm < mc;
        qb[p] = (valid ? qsh + mm * Nu + k : qsh) * 8;
        wb[p] = (valid ? mm : nrow - 1) * 48;
    }
    const unsigned char *xring_b = reinterpret_cast<const unsigned char *>(xring);
    const unsigned char *ybuf_b = reinterpret_cast<const unsigned char *>(ybuf);
    const unsigned char *mtab_b = reinterpret_cast<const unsigned char *>(mtab);
    double fc[NPT], dm[NPT];
    {
        wait_x(c0 - 1); wait_x(c0);
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fc[p] = ldsd(xring_b + QbB, qb[p]); dm[p] = fc[p] - ldsd(xring_b, qb[p]); }
    }
    __syncthreads();                                                 // rows c0-1, c0 consumed
    const bool ym_miss = beyond_wall<1>(P, j - 1), yp_miss = beyond_wall<1>(P, j + 1);
    const double sy = ch.z > 0 ? 1.0 : -1.0;                         // side of the y-contribution (uniform chunks)
    const int s3lag = R == 1 ? 1 : 2;                                // pipeline lag of stage 3 behind stage 1
    constexpr int NJ = NC - 6;                                       // stage-2 jobs per column: 3 (x, b = 0..2) + 7 (y) [+ 7]

    int xslot = 2, xphase = 0, ybuf_i = 0, yphase = 0;               // ring slot / phase of row a+1 and of y stage a (a = c0: row c0+1 is the 3rd row)
    for (int a = c0; a < c1 + 3; ++a) {
        if (a < c1) {                                                // stage 1: point sums of cell a
            mbar_wait(&bars[xslot], xphase);                         // row a+1
            mbar_wait(&bars[NSXM + ybuf_i], yphase);
            const unsigned char *xn = xring_b + xslot * QbB;
            const unsigned char *ym = ybuf_b + ybuf_i * 2 * QbB, *yp = ym + QbB;
            if (++xslot == NSXM) { xslot = 0; xphase ^= 1; }
            if (ybuf_i) yphase ^= 1;
            ybuf_i ^= 1;
            const bool xm_miss = a == 0 && P.bc[0] == BC_WALL, xp_miss = a == P.I - 1 && P.bc[1] == BC_WALL;
            double acc[NA];
#pragma unroll
            for (int i = 0; i < NA; ++i) acc[i] = 0.0;
            auto pass = [&](auto fl) {
                constexpr bool FL = decltype(fl)::value;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double fn = ldsd(xn, qb[p]), c = fc[p];
                    const double dp = fn - c;
                    double dxm = dm[p], dxp = dp, dym = c - ldsd(ym, qb[p]), dyp = ldsd(yp, qb[p]) - c;
                    if (FL) {                                        // AMB-13: one-sided slope next to a wall
                        if (xm_miss) dxm = dp; if (xp_miss) dxp = dm[p];
                        if (ym_miss) dym = dyp; if (yp_miss) dyp = dym;
                    }
                    const double hx = vl_half(dxm, dxp), hy = vl_half(dym, dyp);
                    dm[p] = dp; fc[p] = fn;
                    const double2 w01 = ldsd2(mtab_b, wb[p]), w23 = ldsd2(mtab_b + 16, wb[p]), w4h = ldsd2(mtab_b + 32, wb[p]);
                    // x-faces: t = v_m;  C_b = sum wv t^b f_c,  B_b = sum wv t^b h sigma
                    acc[0] = fma(w01.x, c, acc[0]); acc[1] = fma(w01.y, c, acc[1]); acc[2] = fma(w23.x, c, acc[2]);
                    acc[3] = fma(w01.x, hx, acc[3]); acc[4] = fma(w01.y, hx, acc[4]); acc[5] = fma(w23.x, hx, acc[5]);
                    // y-faces: n = v_m;  A_a = sum wv n^a f0 (a = 0..3),  B_a = sum wv n^a h sigma (a = 2..4)
                    if (!MIXED) {
                        const double f0 = fma(sy, hy, c);
                        acc[6] = fma(w01.x, f0, acc[6]); acc[7] = fma(w01.y, f0, acc[7]); acc[8] = fma(w23.x, f0, acc[8]);
                        acc[9] = fma(w23.y, f0, acc[9]);
                        acc[10] = fma(w23.x, hy, acc[10]); acc[11] = fma(w23.y, hy, acc[11]); acc[12] = fma(w4h.x, hy, acc[12]);
                    } else {                                         // AMB-5: H(0) = 1/2 sends half of the point to either side
                        const double hp = w4h.y, hm = 1.0 - hp, fp = (c + hy) * hp, fm = (c - hy) * hm, gp = hy * hp, gm = hy * hm;
                        acc[6] = fma(w01.x, fp, acc[6]); acc[7] = fma(w01.y, fp, acc[7]); acc[8] = fma(w23.x, fp, acc[8]);
                        acc[9] = fma(w23.y, fp, acc[9]);
                        acc[10] = fma(w23.x, gp, acc[10]); acc[11] = fma(w23.y, gp, acc[11]); acc[12] = fma(w4h.x, gp, acc[12]);
                        acc[13] = fma(w01.x, fm, acc[13]); acc[14] = fma(w01.y, fm, acc[14]); acc[15] = fma(w23.x, fm, acc[15]);
                        acc[16] = fma(w23.y, fm, acc[16]);
                        acc[17] = fma(w23.x, gm, acc[17]); acc[18] = fma(w23.y, gm, acc[18]); acc[19] = fma(w4h.x, gm, acc[19]);
                    }
                }
            };
            if (xm_miss || xp_miss || ym_miss || yp_miss) pass(std::true_type{}); else pass(std::false_type{});
            if (R == 1) {                                            // the thread's sums are the column sums: stage 2 folded in
                if (active) {
                    double *cc = col + (size_t)(a & 1) * NC * NuS + k;
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) {
                        cc[bb * NuS] = acc[bb] + acc[3 + bb]; cc[(3 + bb) * NuS] = acc[bb] - acc[3 + bb]; cc[(6 + bb) * NuS] = acc[3 + bb];
                    }
#pragma unroll
                    for (int i = 6; i < NA; ++i) cc[(3 + i) * NuS] = acc[i];
                }
            } else {
                double *pp = part + (size_t)(a & 1) * NA * B + tid;
#pragma unroll
                for (int i = 0; i < NA; ++i) pp[i * B] = acc[i];
            }
        }
        if (R > 1 && a - 1 >= c0 && a - 1 < c1 && active) {         // stage 2: column sums of cell a-1
            const double *pp = part + (size_t)((a - 1) & 1) * NA * B + k;
            double *cc = col + (size_t)((a - 1) & 1) * NC * NuS + k;
            for (int jb = r; jb < NJ; jb += R) {
                if (jb < 3) {                                        // x, power b = jb of t: C_b +- B_b for the two sides, B_b
                    double C = pp[jb * B], Bs = pp[(3 + jb) * B];
                    for (int rr = 1; rr < R; ++rr) { C += pp[jb * B + rr * Nu]; Bs += pp[(3 + jb) * B + rr * Nu]; }
                    cc[jb * NuS] = C + Bs; cc[(3 + jb) * NuS] = C - Bs; cc[(6 + jb) * NuS] = Bs;
                } else {                                             // y sums
                    double A = pp[(3 + jb) * B];
                    for (int rr = 1; rr < R; ++rr) A += pp[(3 + jb) * B + rr * Nu];
                    cc[(6 + jb) * NuS] = A;
                }
            }
        }
        const int c3 = a - s3lag, c4 = c3 - 1;
        if (c3 >= c0 && c3 < c1) {                                   // stage 3: items (output, k-range) of cell c3
            const unsigned char *cc = reinterpret_cast<const unsigned char *>(col + (size_t)(c3 & 1) * NC * NuS);
            const unsigned char *fb = reinterpret_cast<const unsigned char *>(fac);
            for (int it = tid; it < nitem; it += B) {
                const int4 d = desc[it];
                const double *pf = reinterpret_cast<const double *>(fb + d.x) + d.z, *pc = reinterpret_cast<const double *>(cc + d.y) + d.z;
                double sum = 0.0;
#pragma unroll 4
                for (int n = d.w - d.z; n > 0; --n) sum = fma(*pf++, *pc++, sum);
                ires[(c3 & 1) * nitem + it] = sum;
            }
        }
        if (c4 >= c0 && c4 < c1) {                                   // stage 4: add the items of each output of cell c4, store
            const double *ir = ires + (c4 & 1) * nitem;
            double *dst = P.cmom + (((size_t)j * P.I + c4) * P.nchunk + chunk) * CMS;
            for (int v = tid; v < NOUT; v += B) {
                const int4 od = odesc[v];
                double sum = ir[od.x];
                for (int h = 1; h < od.y; ++h) sum += ir[od.x + h];
                dst[od.z] = sum;
            }
        }
        __syncthreads();                                             // row a+1 is consumed by every thread
    }
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32; }

template <bool MIXED>
static size_t smem_cm(const UgksParams &P)
{
    return (size_t)mom_layout(MIXED, P.Nu, P.cmax, P.R, P.npt, block_threads(P), P.s3_nsx, P.s3_nsy).bytes;
}
size_t smem_cell_moments(const UgksParams &P) { return smem_cm<true>(P); }

// stage-3 split: the fewest parts per output (nsx for the 26 x-outputs over ~Nu/2 columns, nsy for the y-outputs over Nu
// columns) such that items have about equal length and fit one pass of the CTA's threads
void choose_stage3_split(int Nu, int lenx, int B, bool any_mixed, int *nsx, int *nsy)
{
    const int ny = any_mixed ? 2 * NRAW : NRAW;
    int best_x = 1, best_y = 1;
    for (int per = 1; per <= Nu; ++per) {                            // columns per item
        const int sx = (lenx + per - 1) / per, sy = (Nu + per - 1) / per;
        if (2 * NRAW * sx + ny * sy <= B) { best_x = sx; best_y = sy; break; }
    }
    *nsx = best_x; *nsy = best_y;
}

template <bool MIXED, int MAXT, int MINB>
static void launch_cm(const UgksParams &P, int cur, int chunk0, int grid, int T, size_t smem, cudaStream_t st)
{
    switch (P.npt) {
#define CASE(N) case N: k_cell_moments<N, MIXED, MAXT, MINB><<<grid, T, smem, st>>>(P, cur, chunk0); break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7)
#undef CASE
    }
}
template <bool MIXED>
static void launch_cm_class(const UgksParams &P, int cur, int chunk0, int nch, cudaStream_t st)
{
    const int nstrip = (P.I + P.strip - 1) / P.strip;
    const int T = block_threads(P) + 32;                             // + producer warp
    const int grid = P.J * nstrip * nch;
    const size_t smem = smem_cm<MIXED>(P);
    if (T <= 96) launch_cm<MIXED, 96, 4>(P, cur, chunk0, grid, T, smem, st);
    else if (T <= 160) launch_cm<MIXED, 160, 3>(P, cur, chunk0, grid, T, smem, st);
    else launch_cm<MIXED, 288, 1>(P, cur, chunk0, grid, T, smem, st);
}

int launch_cell_moments(const UgksParams &P, int cur, cudaStream_t st)
{
    int n = 0;
    if (P.nneg + P.npos) { launch_cm_class<false>(P, cur, 0, P.nneg + P.npos, st); ++n; }
    if (P.nmix) { launch_cm_class<true>(P, cur, P.nneg + P.npos, P.nmix, st); ++n; }
    return n;
}

template <bool MIXED, int MAXT, int MINB>
static cudaError_t set_attr_cm(int smem)
{
    cudaError_t e = cudaSuccess;
#define ATTR(N) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cell_moments<N, MIXED, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    ATTR(1) ATTR(2) ATTR(3) ATTR(4) ATTR(5) ATTR(6) ATTR(7)
#undef ATTR
    return e;
}
template <bool MIXED>
static cudaError_t set_attr_cm_all(int smem)
{
    cudaError_t e = set_attr_cm<MIXED, 96, 4>(smem);
    if (e == cudaSuccess) e = set_attr_cm<MIXED, 160, 3>(smem);
    if (e == cudaSuccess) e = set_attr_cm<MIXED, 288, 1>(smem);
    return e;
}
int setup_moments_attributes(const UgksParams &P)
{
    if (smem_cm<true>(P) > 227 * 1024) return 1;
    // the attribute is per kernel, not per context: opt every instantiation in to the device maximum once, so that contexts of
    // different geometries can live side by side
    static bool done = false;
    if (done) return 0;
    cudaError_t e = set_attr_cm_all<false>(227 * 1024);
    if (e == cudaSuccess) e = set_attr_cm_all<true>(227 * 1024);
    done = e == cudaSuccess;
    return e == cudaSuccess ? 0 : 1;
}
