// ugks_jit_moments.cuh -- k_cell_moments: reconstruction (R) and the velocity-space reductions of S1 and S7
// ("12 times parallel reduction"), written cell by cell.  Compiled by NVRTC per context (ugks_jit_common.cuh).
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
//     (4) one thread per output adds its items and stores.  All job tables of stages 2..4 are compile-time.
//   * there is no producer warp: after the barrier of step a one lane of a rotating warp issues the bulk copies of the rows
//     that barrier freed.  The partial sums are single-buffered: an mbarrier ("part free", one arrival per warp after its
//     stage-2 reads) orders the next cell's stores behind them without a second CTA-wide barrier.
#pragma once
#include "ugks_jit_common.cuh"

constexpr int NSXM = G_NSXM;                                         // x-ring slots (>= 2)
constexpr int NW = BT / 32;                                          // warps of a CTA
constexpr int NFAC = 14;                                             // factor tables: 5 (x+), 5 (x-), 4 (y)
// raw sum idx -> (power of the per-column velocity, column sum) ; x sets: columns 0..2 = C_b +- B_b, 3..5 = B_b, and with TG
// 6..8 = D_1..D_3 = sum wv v^b (h_y sigma_y) (the tangential slope on an x-face is the cell's y-slope)
__constant__ int c_xa[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 2, 3, 4, 2, 2,   1, 2, 1, 3, 1 };
__constant__ int c_xc[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 3, 3, 3, 4, 5,   6, 6, 7, 6, 8 };
// y sets: columns A_0..A_3, B_2..B_4, and with TG E_1..E_3 = sum wv v^a (h_x sigma_x) (columns 10..12)
__constant__ int c_yt[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 0, 0, 0, 1, 2,   1, 1, 2, 1, 3 };
__constant__ int c_yc[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 4, 5, 6, 4, 4,   10, 11, 10, 12, 10 };

constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }
constexpr int cmaxi(int a, int b) { return a > b ? a : b; }
// stage-3 split: the fewest columns per item such that all items (26 x-outputs over ~Nu/2 columns, the y-outputs over Nu
// columns) fit one pass of the CTA's compute threads; one item per output if even that does not fit
// A sorted grid with a node v = 0 (odd grids, AMB-5: H(0) = 1/2) keeps that row as the FIRST row of the first v > 0 chunk
// (chunk flag .w): all its y-sums with a power of n vanish, so besides the half weight in A_0 of the y+ set it only adds
// sum w/2 (f_c - h sigma) to M00, M01, M02 of the y- set: one more per-thread sum, column and three outputs (ZROW).
constexpr bool ZROW = G_HAS_ZROW != 0;
constexpr int NYX = ZROW ? 3 : 0;                                    // extra y- outputs of the chunk that holds the v = 0 row
constexpr int s3_per(bool mixed)
{
    const int lenx = cmaxi(KXM_END, NU - KXP_BEGIN), ny = mixed ? 2 * NRK : NRK + NYX;
    for (int per = 1; per <= NU; ++per)
        if (2 * NRK * cdiv(lenx, per) + ny * cdiv(NU, per) <= BT) return per;
    return NU;
}

template <bool MIXED>
struct MomL {                                                        // sizes and the shared-memory carve-up (offsets in doubles)
    static constexpr int NTG = TG ? 6 : 0;                           // D_1..D_3, E_1..E_3
    static constexpr int NA = MIXED ? 20 : 13 + NTG + (ZROW ? 1 : 0);   // per-thread sums: 6 (x) + 7 (y) [+ 7 (y-) | + 6 (TG) + 1 (v = 0 row)]
    static constexpr int NC = NA + 3;                                // columns after stage 2: 9 (x) + (NA - 6)
    static constexpr int NYO = MIXED ? 2 * NRK : NRK + NYX;          // y outputs of a chunk
    static constexpr int NOUT = 2 * NRK + NYO;
    static constexpr int LENX = cmaxi(KXM_END, NU - KXP_BEGIN);
    static constexpr int PER = s3_per(MIXED);
    static constexpr int NSX = cdiv(LENX, PER), NSY = cdiv(NU, PER);
    static constexpr int PERX = cdiv(LENX, NSX), PERY = cdiv(NU, NSY);
    static constexpr int NITEM = 2 * NRK * NSX + NYO * NSY;
    static constexpr int NUS = NU | 1;                               // odd column stride
    static constexpr int NROW = R * NPT + 1;                         // weight rows incl. zero rows for a ragged chunk
    static constexpr int O_YBUF = NSXM * QB;
    static constexpr int O_PART = O_YBUF + 4 * QB;
    static constexpr int O_COL = O_PART + (R == 1 ? 0 : NA * BT);
    static constexpr int O_FAC = O_COL + pad2c(2 * NC * NUS);
    static constexpr int O_MTAB = O_FAC + pad2c(NFAC * NUS);
    static constexpr int O_IRES = O_MTAB + pad2c(NROW * 6);
    static constexpr int O_BARS = O_IRES + pad2c(2 * NITEM);
    static constexpr int TOTAL = O_BARS + NSXM + 3;
    static constexpr int BYTES = TOTAL * 8;
};

template <bool MIXED>
__device__ __forceinline__ void cell_moments_body(const KArgs &A, const int chunk0)
{
    using L = MomL<MIXED>;
    constexpr int NA = L::NA, NC = L::NC, NOUT = L::NOUT, NUS = L::NUS, NITEM = L::NITEM, NROW = L::NROW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    int b = blockIdx.x;
    const int j = b % GJ; b /= GJ;
    const int s = b % NSTRIP;
    const int chunk = chunk0 + b / NSTRIP;                           // chunks are sorted: [v < 0][v > 0][mixed]
    const int4 ch = c_chunks[chunk];
    // every CTA marches exactly STRIP cells (a compile-time trip count): the last strip of a row that STRIP does not divide
    // starts at GI - STRIP and re-computes a few cells of its neighbour (same inputs, same arithmetic, same bits)
    const int c0 = min(s * STRIP, GI - STRIP), c1 = c0 + STRIP;      // cells [c0, c1)
    const int m0 = ch.x, mc = ch.y;
    const int q0 = m0 * NU, qa = q0 & ~1, qsh = q0 - qa;             // 16-byte aligned copy start; shift of the chunk inside
    const uint32_t bytes = (uint32_t)(pad2c(mc * NU + qsh) * 8);

    double *sm = reinterpret_cast<double *>(smem_raw);
    double *xring = sm;                                              // [NSXM][QB]
    double *ybuf = sm + L::O_YBUF;                                   // [2][2][QB]
    double *part = sm + L::O_PART;                                   // [NA][BT]
    double *col = sm + L::O_COL;                                     // [2][NC][NUS]
    double *fac = sm + L::O_FAC;                                     // [NFAC][NUS]
    double *mtab = sm + L::O_MTAB;                                   // [NROW][6]: w, w v, w v^2, w v^3, w v^4, H(v) / weight of A_0
    double *ires = sm + L::O_IRES;                                   // [2][NITEM] stage-3 item results
    uint64_t *bars = reinterpret_cast<uint64_t *>(sm + L::O_BARS);   // [NSXM] x rows, [2] y stages, [1] part free

    const int tid = threadIdx.x;
    const bool active = tid < NU * R;
    const int k = active ? tid % NU : 0, r = active ? tid / NU : 0;
    const double *fcur = A.fcur;
    const int rows_first = c0 - 1, rows_last = c1;                   // cells c0-1 .. c1 are staged

    // ---- bulk copies (issued by one elected lane)
    auto issue_x = [&](int row) {
        const int sl = (row - rows_first) % NSXM;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(xring + sl * QB, xrow_ptr(fcur, A.ghost, row, j) + qa, bytes, &bars[sl]);
    };
    auto issue_y = [&](int cell) {
        const int buf = (cell - c0) & 1;
        int ystm, ystp;
        const double *ybm = yrow_base(fcur, A.ghost, j - 1, &ystm) + qa, *ybp = yrow_base(fcur, A.ghost, j + 1, &ystp) + qa;
        mbar_expect_tx(&bars[NSXM + buf], 2 * bytes);
        tma_load_1d(ybuf + (buf * 2) * QB, ybm + (size_t)cell * ystm, bytes, &bars[NSXM + buf]);
        tma_load_1d(ybuf + (buf * 2 + 1) * QB, ybp + (size_t)cell * ystp, bytes, &bars[NSXM + buf]);
    };
    if (tid == 0) {
        for (int i = 0; i < NSXM + 2; ++i) mbar_init(&bars[i], 1);
        mbar_init(&bars[NSXM + 2], NW);
        mbar_fence_init();
        for (int row = rows_first; row < rows_first + NSXM && row <= rows_last; ++row) issue_x(row);
        issue_y(c0);
        if (c0 + 1 < c1) issue_y(c0 + 1);
    }
    for (int i = tid; i < NU; i += BT) {
        const double u = c_u[i], w = c_wu[i];
        const double hp = u > 0.0 ? 1.0 : (u < 0.0 ? 0.0 : 0.5);
        double pw = 1.0;
        for (int a = 0; a < 5; ++a) {
            fac[a * NUS + i] = w * hp * pw;
            fac[(5 + a) * NUS + i] = w * (1.0 - hp) * pw;
            if (a < 4) fac[(10 + a) * NUS + i] = w * pw;
            pw *= u;
        }
    }
    for (int i = tid; i < L::O_FAC - L::O_COL; i += BT) col[i] = 0.0;   // stage 3 may read (times a zero factor) entries no cell has written yet
    for (int i = tid; i < NROW; i += BT) {
        const bool in = i < mc;
        const double v = in ? c_v[m0 + i] : 0.0, w = in ? c_wv[m0 + i] : 0.0;
        double *o = mtab + i * 6;
        o[0] = w; o[1] = w * v; o[2] = w * v * v; o[3] = w * v * v * v; o[4] = w * v * v * v * v;
        // MIXED: H(v) (AMB-5); uniform chunks: the weight of A_0, w (w/2 on a v = 0 row: the other half goes to the y- set)
        o[5] = MIXED ? (v > 0.0 ? 1.0 : (v < 0.0 ? 0.0 : 0.5)) : (in && v == 0.0 ? 0.5 * w : w);
    }
    // stage-3 work items of this thread: item = (output v = (set, idx), part h of its k-range); x+ sums u_k >= 0, x- sums u_k <= 0
    constexpr int S3R = cdiv(NITEM, BT);
    int it_f[S3R], it_c[S3R], it_n[S3R];                             // byte offset into fac, into a col buffer; element count
#pragma unroll
    for (int q = 0; q < S3R; ++q) {
        const int it = tid + q * BT;
        int fi = 0, ci = 0, kb = 0, ke = 0, h = 0, per = 1;
        if (it < 2 * NRK * L::NSX) {
            const int v = it / L::NSX, set = v / NRK, idx = v % NRK, c = c_xc[idx];
            h = it % L::NSX; per = L::PERX;
            fi = (set == 0 ? 0 : 5) + c_xa[idx];
            ci = c < 3 ? (set == 0 ? c : 3 + c) : (c < 6 ? 3 + c : 10 + c);   // columns: 0..2 C+B, 3..5 C-B, 6..8 B, 16..18 D (TG)
            kb = set == 0 ? KXP_BEGIN : 0; ke = set == 0 ? NU : KXM_END;
        } else if (it < NITEM) {
            const int w = it - 2 * NRK * L::NSX, v = w / L::NSY;
            h = w % L::NSY; per = L::PERY;
            if (MIXED || v < NRK) {
                const int ys = v / NRK, idx = v % NRK;
                fi = 10 + c_yt[idx];
                ci = 9 + ys * 7 + c_yc[idx];
            } else {                                                 // v = 0 row: M00, M01, M02 of the y- set from the last column
                fi = 10 + (v - NRK);
                ci = NC - 1;
            }
            kb = 0; ke = NU;
        }
        const int b0 = min(kb + h * per, ke), b1 = min(kb + (h + 1) * per, ke);
        it_f[q] = (fi * NUS + b0) * 8; it_c[q] = (ci * NUS + b0) * 8; it_n[q] = b1 - b0;
    }
    // stage-4 outputs of this thread: output v adds its items and stores to (set, idx)
    constexpr int S4R = cdiv(NOUT, BT);
    int o_first[S4R], o_dst[S4R];
#pragma unroll
    for (int q = 0; q < S4R; ++q) {
        const int v = tid + q * BT;
        int set = v / NRK;
        const int idx = v % NRK;
        o_first[q] = set < 2 ? v * L::NSX : 2 * NRK * L::NSX + (v - 2 * NRK) * L::NSY;
        if (!MIXED && set >= 2) set = ch.z > 0 ? 2 : 3;
        o_dst[q] = idx < 13 ? set * 13 + idx : 52 + set * 5 + (idx - 13);    // [4 sets x 13 base sums | 4 sets x 5 T sums]
        if (!MIXED && v >= 3 * NRK) {                                // the three y- outputs of the v = 0 row (flagged chunk only)
            const int e = v - 3 * NRK;
            o_dst[q] = ch.w ? 3 * 13 + (e == 0 ? RW_M00 : (e == 1 ? RW_M01 : RW_M02)) : -1;
        }
    }
    __syncthreads();
    // the factors of a thread's stage-3 items never change along the march: short items keep them in registers (S3REG doubles
    // at most), which halves the shared-memory loads of stage 3 -- the loads with most of this kernel's bank conflicts
    constexpr int S3REG = 32;
    constexpr int S3LEN = cmaxi(L::PERX, L::PERY);
    constexpr bool FREG = S3R * S3LEN <= S3REG;
    double itfac[FREG ? S3R * S3LEN : 1];
    if constexpr (FREG) {
#pragma unroll
        for (int q = 0; q < S3R; ++q)
#pragma unroll
            for (int n = 0; n < S3LEN; ++n)
                itfac[q * S3LEN + n] = n < it_n[q] ? ldsd(reinterpret_cast<const unsigned char *>(fac), it_f[q] + n * 8) : 0.0;
    }

    // per-thread points: row m = r + p*R; byte offsets are thread base + immediates.  A point outside the chunk (the last
    // point when R*NPT > MC, the tail of a ragged chunk) re-reads the chunk's first element and carries a zero weight row
    // (anything it could read beyond the copied bytes is stale shared memory, possibly NaN: 0 x NaN would poison the sums).
    const int qb0 = (qsh + r * NU + k) * 8, wb0 = r * 48;
    constexpr int QSTEP = R * NU * 8, WSTEP = R * 48;
    int qo[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) qo[p] = r + p * R < mc ? p * QSTEP : qsh * 8 - qb0;
#define QOFF(p) ((G_RAGGED == 0 && ((p) + 1) * R <= MC) ? (p) * QSTEP : qo[p])
    const unsigned char *xring_b = reinterpret_cast<const unsigned char *>(xring);
    const unsigned char *ybuf_b = reinterpret_cast<const unsigned char *>(ybuf);
    const unsigned char *mtab_b = reinterpret_cast<const unsigned char *>(mtab) + wb0;
    double fc[NPT], dm[NPT];
    {
        mbar_wait(&bars[0], 0); mbar_wait(&bars[1], 0);
#pragma unroll
        for (int p = 0; p < NPT; ++p) {
            fc[p] = ldsd(xring_b + QBB, qb0 + QOFF(p));
            dm[p] = fc[p] - ldsd(xring_b, qb0 + QOFF(p));
        }
    }
    __syncthreads();                                                 // rows c0-1, c0 consumed
    if (tid == 0) {
        if (rows_first + NSXM <= rows_last) issue_x(rows_first + NSXM);
        if (rows_first + NSXM + 1 <= rows_last) issue_x(rows_first + NSXM + 1);
    }
    const bool ym_miss = beyond_wall_y(j - 1), yp_miss = beyond_wall_y(j + 1);
    const double sy = ch.z > 0 ? 1.0 : -1.0;                         // side of the y-contribution (uniform chunks)
    const double wz = (ZROW && ch.w && r == 0 && active) ? 0.5 * c_wv[m0] : 0.0;
    // pipeline of one iteration a: stage 1 (cell a) -> [wait "part free"] store partials -> BARRIER -> (elected lane: bulk
    // copies of the freed slots) -> stage 2 (cell a) -> stage 3 (cell a - LAG3) -> stage 4 (cell a - LAG3 - 1)
    constexpr int LAG3 = R == 1 ? 0 : 1;
    uint64_t *pfree = &bars[NSXM + 2];
    const int lane = tid & 31;
    constexpr int NXJ = 3 * NU, NYJ = (NA - 6) * NU;                 // stage-2 jobs: (b, k) x-jobs, (i, k) y-jobs
    constexpr int S2X = cdiv(NXJ, BT), S2Y = cdiv(NYJ, BT);
    double *cmom_row = A.cmom + ((size_t)j * GI * NCHUNK + chunk) * CMS;

    int xslot = 2 % NSXM, xphase = 2 / NSXM, ybuf_i = 0, yphase = 0; // ring slot / phase of row a+1 and of y stage a
    int issuer = 0;                                                  // lane 0 of a rotating warp issues the copies of a step
    constexpr int UNROLL_M = STRIP >= 16 ? 2 : 1;                    // measured (C3, C4): -2 %; short strips: +10 %
#pragma unroll UNROLL_M
    for (int a = c0; a < c1 + LAG3 + 1; ++a) {
        if (a < c1) {                                                // stage 1: point sums of cell a
            mbar_wait(&bars[xslot], xphase);                         // row a+1
            mbar_wait(&bars[NSXM + ybuf_i], yphase);
            const unsigned char *xn = xring_b + xslot * QBB + qb0;
            const unsigned char *ym = ybuf_b + ybuf_i * 2 * QBB + qb0, *yp = ym + QBB;
            if (++xslot == NSXM) { xslot = 0; xphase ^= 1; }
            if (ybuf_i) yphase ^= 1;
            ybuf_i ^= 1;
            const bool xm_miss = a == 0 && BCX0 == BC_WALL, xp_miss = a == GI - 1 && BCX1 == BC_WALL;
            double acc[NA];
#pragma unroll
            for (int i = 0; i < NA; ++i) acc[i] = 0.0;
            double zfix = 0.0;                                       // ZROW: the half of the v = 0 row's weight that A_0 does not get
            auto pass = [&](auto fl) {
                constexpr bool FL = decltype(fl)::value;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double fn = ldsd(xn, QOFF(p)), c = fc[p];
                    const double dp = fn - c;
                    double dxm = dm[p], dxp = dp, dym = c - ldsd(ym, QOFF(p)), dyp = ldsd(yp, QOFF(p)) - c;
                    if (FL) {                                        // AMB-13: one-sided slope next to a wall
                        if (xm_miss) dxm = dp; if (xp_miss) dxp = dm[p];
                        if (ym_miss) dym = dyp; if (yp_miss) dyp = dym;
                    }
                    const double hx = vl_half(dxm, dxp), hy = vl_half(dym, dyp);
                    dm[p] = dp; fc[p] = fn;
                    const double2 w01 = ldsd2(mtab_b, p * WSTEP), w23 = ldsd2(mtab_b + 16, p * WSTEP), w4h = ldsd2(mtab_b + 32, p * WSTEP);
                    // x-faces: t = v_m;  C_b = sum wv t^b f_c,  B_b = sum wv t^b h sigma
                    acc[0] = fma(w01.x, c, acc[0]); acc[1] = fma(w01.y, c, acc[1]); acc[2] = fma(w23.x, c, acc[2]);
                    acc[3] = fma(w01.x, hx, acc[3]); acc[4] = fma(w01.y, hx, acc[4]); acc[5] = fma(w23.x, hx, acc[5]);
                    // y-faces: n = v_m;  A_a = sum wv n^a f0 (a = 0..3),  B_a = sum wv n^a h sigma (a = 2..4)
                    if constexpr (!MIXED) {
                        // A_a = sum wv n^a (f_c + sy h sigma) = Cc_a + sy Hy_a: the sums of f_c (Cc_0..2 are the C_b above, Cc_3 in acc[9]) and of
                        // h sigma_y (Hy_0, Hy_1 in acc[6], acc[7]; Hy_2..4 are the B_a) are kept apart and combined once per cell after
                        // the point loop -- 12 accumulations per point instead of 13 and no f0 per point
                        if (ZROW && p == 0) { acc[NA - 1] = wz * (c - hy); zfix = (w01.x - w4h.y) * fma(sy, hy, c); }   // v = 0 row: halves
                        acc[6] = fma(w01.x, hy, acc[6]); acc[7] = fma(w01.y, hy, acc[7]); acc[9] = fma(w23.y, c, acc[9]);
                        acc[10] = fma(w23.x, hy, acc[10]); acc[11] = fma(w23.y, hy, acc[11]); acc[12] = fma(w4h.x, hy, acc[12]);
                        if constexpr (TG) {                          // tangential slopes: D_b = Hy_b (b = 1..3) come for free; E_a = sum wv v^a (h_x sigma_x)
                            acc[18] = fma(w23.y, hx, acc[18]);      // E_3 (E_1, E_2 are B_1, B_2 of the x-sums)
                        }
                    } else {                                         // AMB-5: H(0) = 1/2 sends half of the point to either side
                        const double hp = w4h.y, hm = 1.0 - hp, fp = (c + hy) * hp, fm = (c - hy) * hm, gp = hy * hp, gm = hy * hm;
                        acc[6] = fma(w01.x, fp, acc[6]); acc[7] = fma(w01.y, fp, acc[7]); acc[8] = fma(w23.x, fp, acc[8]);
                        acc[9] = fma(w23.y, fp, acc[9]);
                        acc[10] = fma(w23.x, gp, acc[10]); acc[11] = fma(w23.y, gp, acc[11]); acc[12] = fma(w4h.x, gp, acc[12]);
                        acc[13] = fma(w01.x, fm, acc[13]); acc[14] = fma(w01.y, fm, acc[14]);
                        acc[15] = fma(w23.x, fm, acc[15]); acc[16] = fma(w23.y, fm, acc[16]);
                        acc[17] = fma(w23.x, gm, acc[17]); acc[18] = fma(w23.y, gm, acc[18]);
                        acc[19] = fma(w4h.x, gm, acc[19]);
                    }
                }
            };
            if (xm_miss || xp_miss || ym_miss || yp_miss) pass(true_c{}); else pass(false_c{});
            if constexpr (!MIXED) {                                  // combine: acc[6..9] = A_0..3; TG: acc[13..15] = D_1..3, acc[16], acc[17] = E_1, E_2
                const double hy0 = acc[6], hy1 = acc[7], c3 = acc[9];
                if constexpr (TG) {
                    acc[13] = hy1; acc[14] = acc[10]; acc[15] = acc[11];
                    acc[16] = acc[4]; acc[17] = acc[5];
                }
                acc[6] = fma(sy, hy0, acc[0]) - zfix; acc[7] = fma(sy, hy1, acc[1]); acc[8] = fma(sy, acc[10], acc[2]);
                acc[9] = fma(sy, acc[11], c3);
            }
            if (R == 1) {                                            // the thread's sums are the column sums: stage 2 folded in
                if (active) {
                    double *cc = col + (a & 1) * NC * NUS + k;
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) {
                        cc[bb * NUS] = acc[bb] + acc[3 + bb]; cc[(3 + bb) * NUS] = acc[bb] - acc[3 + bb]; cc[(6 + bb) * NUS] = acc[3 + bb];
                    }
#pragma unroll
                    for (int i = 6; i < NA; ++i) cc[(3 + i) * NUS] = acc[i];
                }
            } else {
                if (a > c0) mbar_wait(pfree, (a - c0 - 1) & 1);      // every warp has read the partials of cell a-1
                double *pp = part + tid;
#pragma unroll
                for (int i = 0; i < NA; ++i) pp[i * BT] = acc[i];
            }
        }
        __syncthreads();                                             // partials of cell a complete; row a+1 and y stage a consumed
        if (tid == issuer && a < c1) {
            if (a + 1 + NSXM <= rows_last) issue_x(a + 1 + NSXM);
            if (a + 2 < c1) issue_y(a + 2);
        }
        issuer += 32;
        if (issuer >= BT) issuer = 0;
        if (R > 1 && a < c1) {                                       // stage 2: column sums of cell a
            const double *pp = part;
            double *cc = col + (a & 1) * NC * NUS;
#pragma unroll
            for (int q = 0; q < S2X; ++q) {                          // x, power b of t: C_b +- B_b for the two sides, B_b
                const int g = tid + q * BT;
                if (g < NXJ) {
                    const int bq = g / NU, kk = g - bq * NU;
                    const double *pc = pp + bq * BT + kk, *pb = pc + 3 * BT;
                    double C = pc[0], Bs = pb[0];
#pragma unroll
                    for (int rr = 1; rr < R; ++rr) { C += pc[rr * NU]; Bs += pb[rr * NU]; }
                    double *o = cc + bq * NUS + kk;
                    o[0] = C + Bs; o[3 * NUS] = C - Bs; o[6 * NUS] = Bs;
                }
            }
            double ysum[S2Y];
#pragma unroll
            for (int q = 0; q < S2Y; ++q) {                          // y sums
                const int g = tid + q * BT;
                if (g < NYJ) {
                    const int iq = g / NU, kk = g - iq * NU;
                    const double *pa = pp + (6 + iq) * BT + kk;
                    double S = pa[0];
#pragma unroll
                    for (int rr = 1; rr < R; ++rr) S += pa[rr * NU];
                    ysum[q] = S;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(pfree);                       // this warp is done with the partials
#pragma unroll
            for (int q = 0; q < S2Y; ++q) {
                const int g = tid + q * BT;
                if (g < NYJ) { const int iq = g / NU, kk = g - iq * NU; cc[(9 + iq) * NUS + kk] = ysum[q]; }
            }
        }
        const int c3 = a - LAG3, c4 = c3 - 1;
        if (c3 >= c0 && c3 < c1) {                                   // stage 3: items (output, k-range) of cell c3
            const unsigned char *cc = reinterpret_cast<const unsigned char *>(col + (c3 & 1) * NC * NUS);
            const unsigned char *fb = reinterpret_cast<const unsigned char *>(fac);
#pragma unroll
            for (int q = 0; q < S3R; ++q) {
                if (tid + q * BT < NITEM) {
                    constexpr int LEN = cmaxi(L::PERX, L::PERY);
                    double sum = 0.0, sum1 = 0.0;                    // two chains
                    if constexpr (FREG) {
                        // no range test per element: beyond the item's range the register factor is zero and the column entry read
                        // instead is a finite number (a neighbouring column, a zeroed pad element or the factor table behind the buffer)
#pragma unroll
                        for (int n = 0; n < LEN; n += 2) {
                            sum = fma(itfac[q * S3LEN + n], ldsd(cc, it_c[q] + n * 8), sum);
                            if (n + 1 < LEN) sum1 = fma(itfac[FREG ? q * S3LEN + n + 1 : 0], ldsd(cc, it_c[q] + (n + 1) * 8), sum1);
                        }
                    } else {
#pragma unroll
                        for (int n = 0; n < LEN; n += 2) {
                            if (n < it_n[q]) sum = fma(ldsd(fb, it_f[q] + n * 8), ldsd(cc, it_c[q] + n * 8), sum);
                            if (n + 1 < LEN && n + 1 < it_n[q]) sum1 = fma(ldsd(fb, it_f[q] + (n + 1) * 8), ldsd(cc, it_c[q] + (n + 1) * 8), sum1);
                        }
                    }
                    ires[(c3 & 1) * NITEM + tid + q * BT] = sum + sum1;
                }
            }
        }
        if (c4 >= c0 && c4 < c1) {                                   // stage 4: add the items of each output of cell c4, store
            const double *ir = ires + (c4 & 1) * NITEM;
            double *dst = cmom_row + (size_t)c4 * (NCHUNK * CMS);
#pragma unroll
            for (int q = 0; q < S4R; ++q) {
                const int v = tid + q * BT;
                if (v < NOUT) {
                    const int ns = v < 2 * NRK ? L::NSX : L::NSY;
                    double sum = ir[o_first[q]];
#pragma unroll
                    for (int h = 1; h < cmaxi(L::NSX, L::NSY); ++h)
                        if (h < ns) sum += ir[o_first[q] + h];
                    if (o_dst[q] >= 0) dst[o_dst[q]] = sum;
                }
            }
        }
    }
}

static_assert(MomL<false>::BYTES == G_SMEM_MOM, "host mirror of the shared-memory layout (ugks_jit.cu) disagrees");
#if G_NMIX > 0
static_assert(MomL<true>::BYTES == G_SMEM_MOMX, "host mirror of the shared-memory layout (ugks_jit.cu) disagrees");
static_assert(!TG, "the tangential reconstruction needs sorted velocity nodes (no mixed-sign chunks)");
#endif

extern "C" __global__ void __launch_bounds__(BT, G_MINB_MOM) k_cell_moments(const KArgs A, const int chunk0)
{
    cell_moments_body<false>(A, chunk0);
}
#if G_NMIX > 0
extern "C" __global__ void __launch_bounds__(BT, G_MINB_MOMX) k_cell_moments_mixed(const KArgs A, const int chunk0)
{
    cell_moments_body<true>(A, chunk0);
}
#endif
