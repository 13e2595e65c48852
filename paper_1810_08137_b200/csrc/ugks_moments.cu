// ugks_moments.cu -- k_face_moments: reconstruction (R) and the velocity-space reductions of S1 and S7
// ("12 times parallel reduction") for every cell face.
//
// One CTA marches along a strip of consecutive faces of one grid line (x-faces of row j, or y-faces of column i)
// for one chunk of velocity rows.  Thread (k, r) owns velocity column k and the NPT rows m = r + p*R.
//   * stencil: each thread keeps its two upwind-side rows in registers and reads ONE new row per face from a
//     4-slot shared-memory ring fed by 1-D TMA bulk copies (cp.async.bulk + mbarrier), two rows in flight.
//   * the 11 distinct moments of f0 and sigma0 are tensor products: per thread only sum_m wv v^p (.) is
//     accumulated (6-7 sums); the reduction is a three-stage pipeline across consecutive faces, one stage per
//     face step and no extra barrier: (1) partial sums to shared memory, (2) sum over the R threads of each
//     column k, (3) one warp applies the k-dependent factors wu u^a once per column and finishes with a
//     transposing shuffle butterfly (16 shuffles for 16 values instead of 5 per value).
#include "ugks_common.cuh"
#include <type_traits>

constexpr int NACC = 7;
constexpr int NSM = 4;       // stencil ring slots: 2 live rows + 2 in flight (8 slots measured no faster: not latency-bound)

__device__ __forceinline__ double vl_half_rcp(double dm, double dp)
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

// upwind state at the face for the moment sums: f0 = f_c + sg * h sigma_c, hs = h sigma_c (O3).
// FL: mm / mp = minus / plus neighbour is a wall (one-sided, AMB-13); mc = the upwind "cell" is the wall itself:
// nothing comes from the fluid on that side, the face sums take 0 there (the wall part is analytic, O9).
template <bool FL>
__device__ __forceinline__ void recon_m(double fm, double fc, double fp, double sg, bool mm, bool mc, bool mp, double &f0, double &hs)
{
    double dm = fc - fm, dp = fp - fc;
    if (FL) { if (mm) dm = dp; if (mp) dp = dm; }
    hs = vl_half_rcp(dm, dp);
    f0 = fma(sg, hs, fc);
    if (FL && mc) { f0 = 0.0; hs = 0.0; }
}

template <int DIR>
__device__ __forceinline__ int miss_mask_m(const UgksParams &P, int a)
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

template <int DIR, int NPT, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_face_moments(const UgksParams P, const int cur)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nline = DIR == 0 ? P.J : P.I;
    const int npos = (DIR == 0 ? P.I : P.J) + 1;
    const int nstrip = (npos + P.strip - 1) / P.strip;
    int b = blockIdx.x;
    const int line = b % nline; b /= nline;
    const int s = b % nstrip;
    const int chunk = b / nstrip;
    const int a0 = s * P.strip, a1 = min(a0 + P.strip, npos);      // faces [a0, a1)
    const int m0 = chunk * P.chunk_m, mc = min(P.chunk_m, P.Nv - m0);
    const int Nu = P.Nu, R = P.R, CM = P.chunk_m, Q = mc * Nu, q0 = m0 * Nu;
    const int Qs = (CM * Nu + 1) & ~1;
    const uint32_t bytes = (uint32_t)(((Q + 1) & ~1) * sizeof(double));
    const int B = blockDim.x;

    double *ring = reinterpret_cast<double *>(smem_raw);            // [NSM][Qs]
    double *part = ring + (size_t)NSM * Qs;                         // [2][NACC][B]   per-thread partial sums
    double *col = part + 2 * NACC * B;                              // [2][NACC][Nu]  per-column sums
    double *un = col + 2 * NACC * Nu;                               // [Nu] u_k, then [Nu] wu_k
    double *wun = un + Nu;
    double *vn = wun + Nu;                                          // [CM] v_m, then [CM] wv_m
    double *wvn = vn + CM;
    double *red = wvn + CM;                                         // [2][32][16] per-warp moment sums
    uint64_t *bars = reinterpret_cast<uint64_t *>(red + 2 * 32 * 16);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = B >> 5;
    const bool active = tid < Nu * R;
    const int k = tid % Nu, r = tid / Nu;
    const double *fcur = P.f[cur];
    const int rows_first = a0 - 2, rows_last = a1;                  // cells a0-2 .. a1 are staged

    auto issue = [&](int row) {
        int miss;
        const int sl = (row - rows_first) % NSM;
        const double *src = row_ptr<DIR>(P, fcur, row, line, &miss) + q0;
        mbar_expect_tx(&bars[sl], bytes);
        tma_load_1d(ring + (size_t)sl * Qs, src, bytes, &bars[sl]);
    };
    auto wait_row = [&](int row) {
        const int idx = row - rows_first;
        mbar_wait(&bars[idx % NSM], (idx / NSM) & 1);
    };

    if (tid == 0) {
        for (int i = 0; i < NSM; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    for (int i = tid; i < Nu; i += B) { un[i] = P.u[i]; wun[i] = P.wu[i]; }
    for (int i = tid; i < mc; i += B) { vn[i] = P.v[m0 + i]; wvn[i] = P.wv[m0 + i]; }
    __syncthreads();
    if (tid == 0)
        for (int row = rows_first; row < rows_first + NSM && row <= rows_last; ++row) issue(row);

    const double uk = un[k];
    // per-thread points; points outside the chunk are clamped onto a valid one and get zero weight
    double vreg[NPT], wreg[NPT], fm[NPT], fc[NPT];
    int qo[NPT];
#pragma unroll
    for (int p = 0; p < NPT; ++p) {
        const int mm = r + p * R;
        const bool valid = active && mm < mc;
        qo[p] = valid ? mm * Nu + k : 0;
        vreg[p] = vn[valid ? mm : 0];
        wreg[p] = valid ? wvn[mm] : 0.0;
    }
    // window shift per point: 0 for n >= 0 (rows a-2, a-1 held, row a read), 1 for n < 0 (rows a-1, a held, a+1 read)
    auto nvel = [&](int p) { return DIR == 0 ? uk : vreg[p]; };
    {
        wait_row(a0 - 2); wait_row(a0 - 1); wait_row(a0);
#pragma unroll
        for (int p = 0; p < NPT; ++p) {
            const int sh = nvel(p) < 0.0 ? 1 : 0;
            fm[p] = ring[(size_t)sh * Qs + qo[p]];
            fc[p] = ring[(size_t)(sh + 1) * Qs + qo[p]];
        }
    }
    __syncthreads();
    if (tid == 0) {
        if (a0 + NSM - 2 <= rows_last) issue(a0 + NSM - 2);
        if (a0 + NSM - 1 <= rows_last) issue(a0 + NSM - 1);
    }
    const double inv_h = 2.0 / (DIR == 0 ? P.dx : P.dy);

    const int nw3 = min(nwarp, (Nu + 31) / 32);                     // warps that own columns in stage 3
    for (int a = a0; a < a1 + 3; ++a) {
        if (a < a1) {                                               // stage 1: point sums of face a
            wait_row(a + 1);
            const double *rA = ring + (size_t)((a - rows_first) % NSM) * Qs;          // row a
            const double *rB = ring + (size_t)((a + 1 - rows_first) % NSM) * Qs;      // row a+1
            const int ms = miss_mask_m<DIR>(P, a);
            double acc[NACC];
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
            auto pass = [&](auto fl) {
                constexpr bool FL = decltype(fl)::value;
#pragma unroll
                for (int p = 0; p < NPT; ++p) {
                    const double n = nvel(p), vm = vreg[p];
                    const bool neg = n < 0.0;
                    const double fn = neg ? rB[qo[p]] : rA[qo[p]];
                    double f0, hs;
                    if (neg) recon_m<FL>(fm[p], fc[p], fn, -1.0, ms & 2, ms & 4, ms & 8, f0, hs);
                    else recon_m<FL>(fm[p], fc[p], fn, 1.0, ms & 1, ms & 2, ms & 4, f0, hs);
                    if (n == 0.0) {                                 // AMB-5: H(0) = 1/2, both sides; sigma0 is never used (x n)
                        double f0r, hsr;
                        recon_m<FL>(fc[p], fn, rB[qo[p]], -1.0, ms & 2, ms & 4, ms & 8, f0r, hsr);
                        f0 = (FL && (ms & 6)) ? 0.0 : 0.5 * (f0 + f0r);
                        hs = 0.0;
                    }
                    fm[p] = fc[p]; fc[p] = fn;
                    const double pw = wreg[p] * f0, sg = wreg[p] * hs, v2 = vm * vm;
                    if (DIR == 0) {                                 // loop variable is t = v_m
                        acc[0] += pw; acc[1] = fma(pw, vm, acc[1]); acc[2] = fma(pw, v2, acc[2]);
                        acc[3] += sg; acc[4] = fma(sg, vm, acc[4]); acc[5] = fma(sg, v2, acc[5]);
                    } else {                                        // loop variable is n = v_m
                        const double pn = pw * vm, sn2 = sg * v2;
                        acc[0] += pw; acc[1] += pn; acc[2] = fma(pn, vm, acc[2]); acc[3] = fma(pn, v2, acc[3]);
                        acc[4] += sn2; acc[5] = fma(sn2, vm, acc[5]); acc[6] = fma(sn2, v2, acc[6]);
                    }
                }
            };
            if (ms == 0) pass(std::false_type{}); else pass(std::true_type{});
            double *pp = part + (size_t)(a & 1) * NACC * B + tid;
#pragma unroll
            for (int i = 0; i < NACC; ++i) pp[i * B] = active ? acc[i] : 0.0;
        }
        if (a - 1 >= a0 && a - 1 < a1) {                            // stage 2: column sums of face a-1
            const double *pp = part + (size_t)((a - 1) & 1) * NACC * B;
            double *cc = col + (size_t)((a - 1) & 1) * NACC * Nu;
            for (int idx = tid; idx < NACC * Nu; idx += B) {
                const int i = idx / Nu, kk = idx - i * Nu;
                double sum = 0.0;
                for (int rr = 0; rr < R; ++rr) sum += pp[i * B + rr * Nu + kk];
                cc[idx] = sum;
            }
        }
        if (a - 2 >= a0 && a - 2 < a1 && warp < nw3) {              // stage 3: k-dependent factors + butterfly, per warp
            const double *cc = col + (size_t)(a & 1) * NACC * Nu;   // (a-2)&1 == a&1
            double o[16];
#pragma unroll
            for (int v = 0; v < 16; ++v) o[v] = 0.0;
            for (int kk = tid; kk < Nu; kk += 32 * nw3) {
                const double w = wun[kk], c = un[kk], c2 = c * c, ws = w * inv_h;
                const double A0 = cc[kk], A1 = cc[Nu + kk], A2 = cc[2 * Nu + kk], A3 = cc[3 * Nu + kk];
                const double B4 = cc[4 * Nu + kk], B5 = cc[5 * Nu + kk], B6 = cc[6 * Nu + kk];
                double M00, M10, M01, M20, M02, M11, M30, M12, S20, S30, S21, S40, S22;
                if (DIR == 0) {                                     // n = u_k = c; A0..A2 = sum wv t^b f0, A3,B4,B5 = sum wv t^b hs
                    M00 = w * A0; M10 = M00 * c; M20 = M10 * c; M30 = M20 * c;
                    M01 = w * A1; M11 = M01 * c; M02 = w * A2; M12 = M02 * c;
                    S20 = ws * c2 * A3; S30 = S20 * c; S40 = S30 * c; S21 = ws * c2 * B4; S22 = ws * c2 * B5;
                } else {                                            // t = u_k = c; A0..A3 = sum wv n^a f0, B4..B6 = sum wv n^(2..4) hs
                    M00 = w * A0; M01 = M00 * c; M02 = M01 * c;
                    M10 = w * A1; M11 = M10 * c; M12 = M11 * c; M20 = w * A2; M30 = w * A3;
                    S20 = ws * B4; S21 = S20 * c; S22 = S21 * c; S30 = ws * B5; S40 = ws * B6;
                }
                o[0] += M00; o[1] += M10; o[2] += M01; o[3] += 0.5 * (M20 + M02); o[4] += M20; o[5] += M11;
                o[6] += 0.5 * (M30 + M12); o[7] += S20; o[8] += S30; o[9] += S21; o[10] += 0.5 * (S40 + S22);
            }
            // transposing butterfly: after the step with offset 2^b the lane keeps the half selected by its bit b
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const bool hi = lane & 16;
                const double send = hi ? o[i] : o[i + 8], keep = hi ? o[i + 8] : o[i];
                o[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const bool hi = lane & 8;
                const double send = hi ? o[i] : o[i + 4], keep = hi ? o[i + 4] : o[i];
                o[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const bool hi = lane & 4;
                const double send = hi ? o[i] : o[i + 2], keep = hi ? o[i + 2] : o[i];
                o[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
            }
            {
                const bool hi = lane & 2;
                const double send = hi ? o[0] : o[1], keep = hi ? o[1] : o[0];
                o[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
            }
            o[0] += __shfl_xor_sync(0xffffffffu, o[0], 1);
            // lane holds moment v = 8*bit4 + 4*bit3 + 2*bit2 + bit1
            const int v = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
            if ((lane & 1) == 0) red[((a & 1) * 32 + warp) * 16 + v] = o[0];
        }
        if (a - 3 >= a0 && tid < 11) {                              // stage 4: sum over the warps of stage 3, store
            const double *rr = red + (size_t)((a - 1) & 1) * 32 * 16 + tid;   // (a-3)&1 == (a-1)&1
            double sum = 0.0;
            for (int w = 0; w < nw3; ++w) sum += rr[w * 16];
            const int fa = a - 3;
            const size_t face = DIR == 0 ? (size_t)line * (P.I + 1) + fa : (size_t)fa * P.I + line;
            P.mom[DIR][(face * P.nchunk + chunk) * NMOM + tid] = sum;
        }
        __syncthreads();
        if (tid == 0 && a < a1 && a + NSM <= rows_last) issue(a + NSM);   // row a is consumed by every thread
    }
}

size_t smem_face_moments(const UgksParams &P)
{
    const size_t Qs = ((size_t)P.chunk_m * P.Nu + 1) & ~(size_t)1;
    const size_t B = ((size_t)P.Nu * P.R + 31) / 32 * 32;
    const size_t tabs = 2 * (size_t)P.Nu + 2 * (size_t)P.chunk_m;
    return (NSM * Qs + 2 * NACC * B + 2 * NACC * (size_t)P.Nu + tabs + 2 * 32 * 16) * sizeof(double) + NSM * sizeof(uint64_t);
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32; }

template <int DIR, int MAXT, int MINB>
static void launch_dir(const UgksParams &P, int cur, int grid, int T, size_t smem, cudaStream_t st)
{
    switch (P.npt) {
#define CASE(N) case N: k_face_moments<DIR, N, MAXT, MINB><<<grid, T, smem, st>>>(P, cur); break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    }
}

int launch_face_moments(const UgksParams &P, int cur, int dir, cudaStream_t st)
{
    const size_t smem = smem_face_moments(P);
    const int nsx = (P.I + 1 + P.strip - 1) / P.strip, nsy = (P.J + 1 + P.strip - 1) / P.strip;
    const int T = block_threads(P);
    const int grid = dir == 0 ? P.J * nsx * P.nchunk : P.I * nsy * P.nchunk;
    if (T <= 128) { if (dir == 0) launch_dir<0, 128, 4>(P, cur, grid, T, smem, st); else launch_dir<1, 128, 4>(P, cur, grid, T, smem, st); }
    else if (T <= 256) { if (dir == 0) launch_dir<0, 256, 2>(P, cur, grid, T, smem, st); else launch_dir<1, 256, 2>(P, cur, grid, T, smem, st); }
    else { if (dir == 0) launch_dir<0, 1024, 1>(P, cur, grid, T, smem, st); else launch_dir<1, 1024, 1>(P, cur, grid, T, smem, st); }
    return 1;
}

template <int DIR, int MAXT, int MINB>
static cudaError_t set_attr_dir(int smem)
{
    cudaError_t e = cudaSuccess;
#define ATTR(N) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_face_moments<DIR, N, MAXT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    ATTR(1) ATTR(2) ATTR(3) ATTR(4) ATTR(5) ATTR(6) ATTR(7) ATTR(8)
#undef ATTR
    return e;
}

int setup_moments_attributes(const UgksParams &P)
{
    const int smem = (int)smem_face_moments(P);
    cudaError_t e = set_attr_dir<0, 128, 4>(smem);
    if (e == cudaSuccess) e = set_attr_dir<1, 128, 4>(smem);
    if (e == cudaSuccess) e = set_attr_dir<0, 256, 2>(smem);
    if (e == cudaSuccess) e = set_attr_dir<1, 256, 2>(smem);
    if (e == cudaSuccess) e = set_attr_dir<0, 1024, 1>(smem);
    if (e == cudaSuccess) e = set_attr_dir<1, 1024, 1>(smem);
    return e == cudaSuccess ? 0 : 1;
}
