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
//   * sums are tensor products: a thread accumulates sum_m wv v^p (.) for its column (13 sums; weights wv v^p come as
//     broadcast shared-memory loads); three pipelined stages, one per cell step, finish the reduction without an extra
//     barrier: (1) partial sums to shared memory, (2) sum over the R threads of a column, (3) per output one thread (or
//     2 / 4) takes the dot product over k with the factors wu u^a H(+-u).
#include "ugks_common.cuh"
#include <type_traits>

constexpr int NSXM = 3;                                              // x-ring slots
constexpr int NFAC = 13;                                             // factor tables: 5 (x+), 5 (x-), 3 (y)
__constant__ int c_xa[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 2, 3, 4, 2, 2 };   // power of n = u_k of raw sum idx (x sets)
__constant__ int c_xc[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 3, 3, 3, 4, 5 };   // column sum: 0..2 = C_b (+- B_b), 3..5 = B_b
__constant__ int c_yt[NRAW] = { 0, 0, 0, 0, 1, 1, 2, 2, 0, 0, 0, 1, 2 };   // power of t = u_k (y sets)
__constant__ int c_yc[NRAW] = { 0, 1, 2, 3, 0, 1, 0, 1, 4, 5, 6, 4, 4 };   // column sum: A_0..A_3, B_2..B_4

template <int NPT, bool MIXED, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_cell_moments(const UgksParams P, const int cur, const int chunk0)
{
    constexpr int NA = MIXED ? 20 : 13;                              // column sums per thread: 6 (x) + 7 (y) [+ 7 (y-)]
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
    const int Qb = pad2(P.cmax * Nu + 1);
    const uint32_t bytes = (uint32_t)(pad2(mc * Nu + qsh) * sizeof(double));
    const int B = blockDim.x;
    const int nrow = R * NPT + 1;                                    // weight rows incl. a zero row

    double *xring = reinterpret_cast<double *>(smem_raw);            // [NSXM][Qb]
    double *ybuf = xring + (size_t)NSXM * Qb;                        // [2][2][Qb]
    double *part = ybuf + (size_t)4 * Qb;                            // [2][NA][B]
    double *col = part + (size_t)2 * NA * B;                         // [2][NA][Nu]
    double *fac = col + (size_t)2 * NA * Nu;                         // [NFAC][Nu]
    double *mtab = fac + (size_t)pad2(NFAC * Nu);                    // [nrow][6]: w, w v, w v^2, w v^3, w v^4, H(v)
    int4 *desc = reinterpret_cast<int4 *>(mtab + (size_t)pad2(nrow * 6));      // [NOUT] stage-3 output descriptors
    uint64_t *bars = reinterpret_cast<uint64_t *>(desc + NOUT);     // [NSXM] x rows, [2] y stages

    const int tid = threadIdx.x;
    const bool active = tid < Nu * R;
    const int k = active ? tid % Nu : 0, r = active ? tid / Nu : 0;
    const double *fcur = P.f[cur];
    const int rows_first = c0 - 1, rows_last = c1;                   // cells c0-1 .. c1 are staged

    auto issue_x = [&](int row) {
        const int sl = (row - rows_first) % NSXM;
        const double *src = row_ptr<0>(P, fcur, row, j) + qa;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(xring + (size_t)sl * Qb, src, bytes, &bars[sl]);
    };
    auto wait_x = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSXM], (idx / NSXM) & 1);
    };
    auto issue_y = [&](int cell) {
        const int buf = (cell - c0) & 1;
        mbar_expect_tx(&bars[NSXM + buf], 2 * bytes);
        tma_load_1d(ybuf + (size_t)(buf * 2) * Qb, row_ptr<1>(P, fcur, j - 1, cell) + qa, bytes, &bars[NSXM + buf]);
        tma_load_1d(ybuf + (size_t)(buf * 2 + 1) * Qb, row_ptr<1>(P, fcur, j + 1, cell) + qa, bytes, &bars[NSXM + buf]);
    };

    if (tid == 0) {
        for (int i = 0; i < NSXM + 2; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    for (int i = tid; i < Nu; i += B) {
        const double u = P.u[i], w = P.wu[i];
        const double hp = u > 0.0 ? 1.0 : (u < 0.0 ? 0.0 : 0.5);
        double pw = 1.0;
        for (int a = 0; a < 5; ++a) {
            fac[a * Nu + i] = w * hp * pw;
            fac[(5 + a) * Nu + i] = w * (1.0 - hp) * pw;
            if (a < 3) fac[(10 + a) * Nu + i] = w * pw;
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
    __syncthreads();
    if (tid == 0) {
        for (int row = rows_first; row < rows_first + NSXM && row <= rows_last; ++row) issue_x(row);
        issue_y(c0);
        if (c0 + 1 < c1) issue_y(c0 + 1);
    }

    // per-thread points; a point outside the chunk (ragged tail, padding threads) reads a valid value and the zero weight row
    int qoff[NPT], woff[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        const bool valid = active && mm < mc;
        qoff[p] = valid ? qsh + mm * Nu + k : qsh;
        woff[p] = (valid ? mm : nrow - 1) * 6;
    }
    double fc[NPT], dm[NPT];
    {
        wait_x(c0 - 1); wait_x(c0);
        const double *ra = xring, *rb = xring + Qb;
#pragma unroll
        for (int p = 0; p < NPT; ++p) { fc[p] = rb[qoff[p]]; dm[p] = fc[p] - ra[qoff[p]]; }
    }
    __syncthreads();                                                 // rows c0-1, c0 consumed
    if (tid == 0) {
        if (c0 + 2 <= rows_last) issue_x(c0 + 2);
        if (c0 + 3 <= rows_last) issue_x(c0 + 3);
    }
    const bool ym_miss = beyond_wall<1>(P, j - 1), yp_miss = beyond_wall<1>(P, j + 1);
    const double sy = ch.z > 0 ? 1.0 : -1.0;                         // side of the y-contribution (uniform chunks)

    // stage-3 descriptors: output v = (set, idx) -> (factor table, column sums ca (+- cb)); groups of nsplit lanes share an output
    const int nsplit = B >= 4 * NOUT ? 4 : (B >= 2 * NOUT ? 2 : 1);
    const int ngroup = B / nsplit, ov = tid / nsplit, oh = tid % nsplit;
    const int oiter = (NOUT + ngroup - 1) / ngroup;
    for (int v = tid; v < NOUT; v += B) {
        int set = v / NRAW;
        const int idx = v % NRAW;
        int fi, ca, cb, sb;
        if (set < 2) {                                               // x+ / x-: M terms take C_b +- B_b, S terms B_b
            const int c = c_xc[idx];
            fi = (set == 0 ? 0 : 5) + c_xa[idx];
            if (c < 3) { ca = c; cb = 3 + c; sb = set == 0 ? 1 : 2; }
            else { ca = c; cb = c; sb = 0; }
        } else {                                                     // y (uniform chunks: one set; mixed: y+ then y-)
            fi = 10 + c_yt[idx];
            ca = cb = 6 + (set - 2) * 7 + c_yc[idx];
            sb = 0;
            if (!MIXED) set = ch.z > 0 ? 2 : 3;
        }
        desc[v] = make_int4(fi * Nu, ca * Nu, cb * Nu, (sb << 16) | (set * NRAW + idx));
    }
    __syncthreads();

    for (int a = c0; a < c1 + 2; ++a) {
        if (a < c1) {                                                // stage 1: point sums of cell a
            wait_x(a + 1);
            mbar_wait(&bars[NSXM + ((a - c0) & 1)], ((a - c0) >> 1) & 1);
            const double *xn = xring + (size_t)((a + 1 - rows_first) % NSXM) * Qb;
            const double *ym = ybuf + (size_t)(((a - c0) & 1) * 2) * Qb, *yp = ym + Qb;
            const bool xm_miss = beyond_wall<0>(P, a - 1), xp_miss = beyond_wall<0>(P, a + 1);
            double acc[NA];
#pragma unroll
            for (int i = 0; i < NA; ++i) acc[i] = 0.0;
            auto pass = [&](auto fl) {
                constexpr bool FL = decltype(fl)::value;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double fn = xn[qoff[p]], c = fc[p];
                    const double dp = fn - c;
                    double dxm = dm[p], dxp = dp, dym = c - ym[qoff[p]], dyp = yp[qoff[p]] - c;
                    if (FL) {                                        // AMB-13: one-sided slope next to a wall
                        if (xm_miss) dxm = dp; if (xp_miss) dxp = dm[p];
                        if (ym_miss) dym = dyp; if (yp_miss) dyp = dym;
                    }
                    const double hx = vl_half(dxm, dxp), hy = vl_half(dym, dyp);
                    dm[p] = dp; fc[p] = fn;
                    const double2 w01 = *reinterpret_cast<const double2 *>(mtab + woff[p]);
                    const double2 w23 = *reinterpret_cast<const double2 *>(mtab + woff[p] + 2);
                    const double2 w4h = *reinterpret_cast<const double2 *>(mtab + woff[p] + 4);
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
            double *pp = part + (size_t)(a & 1) * NA * B + tid;
#pragma unroll
            for (int i = 0; i < NA; ++i) pp[i * B] = acc[i];
        }
        if (a - 1 >= c0 && a - 1 < c1) {                            // stage 2: column sums of cell a-1
            const double *pp = part + (size_t)((a - 1) & 1) * NA * B;
            double *cc = col + (size_t)((a - 1) & 1) * NA * Nu;
            for (int idx = tid; idx < NA * Nu; idx += B) {
                const int i = idx / Nu, kk = idx - i * Nu;
                double sum = pp[i * B + kk];
                for (int rr = 1; rr < R; ++rr) sum += pp[i * B + rr * Nu + kk];
                cc[idx] = sum;
            }
        }
        if (a - 2 >= c0) {                                           // stage 3: dot products over k of cell a-2
            const double *cc = col + (size_t)(a & 1) * NA * Nu;      // (a-2)&1 == a&1
            const size_t cell = (size_t)j * P.I + (a - 2);
            double *dst = P.cmom + (cell * P.nchunk + chunk) * CMS;
            for (int it = 0; it < oiter; ++it) {
                const int v = it * ngroup + ov;
                const bool on = v < NOUT;
                const int4 d = desc[on ? v : 0];
                const double sb = (d.w >> 16) == 0 ? 0.0 : ((d.w >> 16) == 1 ? 1.0 : -1.0);
                double sum = 0.0;
                if (on) {
                    const double *F = fac + d.x, *ca = cc + d.y, *cb = cc + d.z;
                    for (int kk = oh; kk < Nu; kk += nsplit) sum = fma(F[kk], fma(sb, cb[kk], ca[kk]), sum);
                }
                if (nsplit >= 2) sum += __shfl_xor_sync(0xffffffffu, sum, 1);
                if (nsplit >= 4) sum += __shfl_xor_sync(0xffffffffu, sum, 2);
                if (on && oh == 0) dst[d.w & 0xffff] = sum;
            }
        }
        __syncthreads();
        if (tid == 0 && a < c1) {
            if (a + 4 <= rows_last) issue_x(a + 4);                  // row a+1 is consumed by every thread
            if (a + 2 < c1) issue_y(a + 2);
        }
    }
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32; }

template <bool MIXED>
static size_t smem_cm(const UgksParams &P)
{
    const size_t NA = MIXED ? 20 : 13, NOUT = MIXED ? 4 * NRAW : 3 * NRAW, B = block_threads(P), Qb = pad2(P.cmax * P.Nu + 1);
    const size_t nrow = (size_t)P.R * P.npt + 1;
    return ((NSXM + 4) * Qb + 2 * NA * B + 2 * NA * (size_t)P.Nu + pad2(NFAC * P.Nu) + pad2(nrow * 6) + 2 * NOUT) * sizeof(double)
           + (NSXM + 2) * sizeof(uint64_t);
}
size_t smem_cell_moments(const UgksParams &P) { return smem_cm<true>(P); }

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
    const int T = block_threads(P);
    const int grid = P.J * nstrip * nch;
    const size_t smem = smem_cm<MIXED>(P);
    if (T <= 64) launch_cm<MIXED, 64, 6>(P, cur, chunk0, grid, T, smem, st);
    else if (T <= 128) launch_cm<MIXED, 128, 4>(P, cur, chunk0, grid, T, smem, st);
    else launch_cm<MIXED, 256, 2>(P, cur, chunk0, grid, T, smem, st);
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
    cudaError_t e = set_attr_cm<MIXED, 64, 6>(smem);
    if (e == cudaSuccess) e = set_attr_cm<MIXED, 128, 4>(smem);
    if (e == cudaSuccess) e = set_attr_cm<MIXED, 256, 2>(smem);
    return e;
}
int setup_moments_attributes(const UgksParams &P)
{
    if (smem_cm<true>(P) > 227 * 1024) return 1;
    cudaError_t e = set_attr_cm_all<false>((int)smem_cm<false>(P));
    if (e == cudaSuccess) e = set_attr_cm_all<true>((int)smem_cm<true>(P));
    return e == cudaSuccess ? 0 : 1;
}
