// ugks_moments.cu -- k_face_moments: reconstruction (R) and the velocity-space reductions of S1 and S7
// ("12 times parallel reduction") for every cell face.
//
// One CTA marches along a strip of consecutive faces of one grid line (x-faces of row j, or y-faces of
// column i) for one chunk of velocity rows.  The stencil rows i-2..i+1 of f live in a shared-memory ring
// filled by 1-D TMA bulk copies (cp.async.bulk + mbarrier), two rows in flight ahead of the math.
// Thread (k, r) owns velocity column k and the rows m = r, r+R, ...; the sums over m are accumulated per
// thread as  sum_m wv v^p f0  and the k-dependent factor wu u^a is applied once per face (tensor-product
// form of the 11 distinct moments), then warp shuffles and a shared-memory tree finish the reduction.
#include "ugks_common.cuh"

template <int DIR>
__device__ __forceinline__ int cell_missing(const UgksParams &P, int pos)
{
    const int n = DIR == 0 ? P.I : P.J;
    const int lo = DIR == 0 ? 0 : 2;
    return (pos < 0 && P.bc[lo] == BC_WALL) || (pos >= n && P.bc[lo + 1] == BC_WALL);
}

template <int DIR, int MAXT>
__global__ void __launch_bounds__(MAXT) k_face_moments(const UgksParams P, const int cur)
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
    const int Nu = P.Nu, Q = mc * Nu, q0 = m0 * Nu;
    const int Qs = (P.chunk_m * Nu + 1) & ~1;
    const uint32_t bytes = (uint32_t)(((Q + 1) & ~1) * sizeof(double));

    double *ring = reinterpret_cast<double *>(smem_raw);
    double *vt = ring + (size_t)RINGX * Qs;
    double *wvt = vt + P.chunk_m;
    double *red = wvt + P.chunk_m;                                  // [2][32][NMOM]
    uint64_t *bars = reinterpret_cast<uint64_t *>(red + 2 * 32 * NMOM);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
    const bool active = tid < Nu * P.R;
    const int k = tid % Nu, r = tid / Nu;
    const double *fcur = P.f[cur];
    const int rows_first = a0 - 2, rows_last = a1;                  // cells a0-2 .. a1 are staged

    if (tid == 0) {
        for (int i = 0; i < RINGX; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    for (int i = tid; i < mc; i += blockDim.x) {
        vt[i] = (DIR == 0 ? P.v : P.v)[m0 + i];
        wvt[i] = P.wv[m0 + i];
    }
    __syncthreads();
    if (tid == 0) {
        for (int idx = 0; idx < RINGX && rows_first + idx <= rows_last; ++idx) {
            int miss;
            const double *src = row_ptr<DIR>(P, fcur, rows_first + idx, line, &miss) + q0;
            mbar_expect_tx(&bars[idx], bytes);
            tma_load_1d(ring + (size_t)idx * Qs, src, bytes, &bars[idx]);
        }
    }
    const double uk = active ? P.u[k] : 0.0, wuk = active ? P.wu[k] : 0.0;
    const double inv_h = 2.0 / (DIR == 0 ? P.dx : P.dy);

    for (int a = a0; a < a1; ++a) {
        const int idxN = a - a0 + 3;                                // newest row needed: cell a+1
        if (a == a0) for (int idx = 0; idx < 3; ++idx) mbar_wait(&bars[idx % RINGX], (idx / RINGX) & 1);
        mbar_wait(&bars[idxN % RINGX], (idxN / RINGX) & 1);
        const double *rLL = ring + (size_t)((idxN - 3) % RINGX) * Qs;
        const double *rL = ring + (size_t)((idxN - 2) % RINGX) * Qs;
        const double *rR = ring + (size_t)((idxN - 1) % RINGX) * Qs;
        const double *rRR = ring + (size_t)(idxN % RINGX) * Qs;
        const int missLL = cell_missing<DIR>(P, a - 2), missL = cell_missing<DIR>(P, a - 1);
        const int missR = cell_missing<DIR>(P, a), missRR = cell_missing<DIR>(P, a + 1);

        double A0 = 0, A1 = 0, A2 = 0, A3 = 0, B0 = 0, B1 = 0, B2 = 0, B3 = 0, B4 = 0;
        if (active) {
            for (int mm = r; mm < mc; mm += P.R) {
                const int q = mm * Nu + k;
                const double vm = vt[mm], wvm = wvt[mm];
                const double n = DIR == 0 ? uk : vm;
                const double fL = rL[q], fR = rR[q];
                double f0, hs;
                if (n > 0.0) {                                      // upwind cell L
                    if (missL) { f0 = 0.0; hs = 0.0; }
                    else {
                        double dp = fR - fL, dm = fL - rLL[q];
                        if (missLL) dm = dp;                        // AMB-13: one-sided next to a wall
                        if (missR) dp = dm;
                        hs = vl_half(dm, dp);
                        f0 = fL + hs;
                    }
                } else if (n < 0.0) {                               // upwind cell R
                    if (missR) { f0 = 0.0; hs = 0.0; }
                    else {
                        double dm = fR - fL, dp = rRR[q] - fR;
                        if (missL) dm = dp;
                        if (missRR) dp = dm;
                        hs = vl_half(dm, dp);
                        f0 = fR - hs;
                    }
                } else {                                            // AMB-5: H(0) = 1/2; sigma0 never matters (x n)
                    hs = 0.0;
                    if (missL || missR) f0 = 0.0;
                    else {
                        const double dc = fR - fL;
                        const double dmm = missLL ? dc : fL - rLL[q];
                        const double dpp = missRR ? dc : rRR[q] - fR;
                        f0 = 0.5 * ((fL + vl_half(dmm, dc)) + (fR - vl_half(dc, dpp)));
                    }
                }
                const double p = wvm * f0, sg = wvm * hs;
                const double v2 = vm * vm;
                if (DIR == 0) {                                     // loop variable is t = v_m
                    A0 += p; A1 = fma(p, vm, A1); A2 = fma(p, v2, A2);
                    B0 += sg; B1 = fma(sg, vm, B1); B2 = fma(sg, v2, B2);
                } else {                                            // loop variable is n = v_m
                    const double pn = p * vm, sn2 = sg * v2;
                    A0 += p; A1 += pn; A2 = fma(pn, vm, A2); A3 = fma(pn, v2, A3);
                    B2 += sn2; B3 = fma(sn2, vm, B3); B4 = fma(sn2, v2, B4);
                }
            }
        }
        // k-dependent factors: M_ab = sum w n^a t^b f0, S_ab = sum w n^a t^b sigma0
        double o[11];
        {
            const double w = wuk, c = uk, c2 = c * c, ws = wuk * inv_h;
            double M00, M10, M01, M20, M02, M11, M30, M12, S20, S30, S21, S40, S22;
            if (DIR == 0) {                                         // n = u_k = c
                M00 = w * A0; M10 = M00 * c; M20 = M10 * c; M30 = M20 * c;
                M01 = w * A1; M11 = M01 * c; M02 = w * A2; M12 = M02 * c;
                S20 = ws * c2 * B0; S30 = S20 * c; S40 = S30 * c; S21 = ws * c2 * B1; S22 = ws * c2 * B2;
            } else {                                                // t = u_k = c
                M00 = w * A0; M01 = M00 * c; M02 = M01 * c;
                M10 = w * A1; M11 = M10 * c; M12 = M11 * c; M20 = w * A2; M30 = w * A3;
                S20 = ws * B2; S21 = S20 * c; S22 = S21 * c; S30 = ws * B3; S40 = ws * B4;
            }
            o[0] = M00; o[1] = M10; o[2] = M01; o[3] = 0.5 * (M20 + M02); o[4] = M20; o[5] = M11;
            o[6] = 0.5 * (M30 + M12); o[7] = S20; o[8] = S30; o[9] = S21; o[10] = 0.5 * (S40 + S22);
        }
        double *redp = red + (size_t)((a - a0) & 1) * 32 * NMOM;
#pragma unroll
        for (int v = 0; v < 11; ++v) {
            const double sum = warp_sum(o[v]);
            if (lane == 0) redp[warp * NMOM + v] = sum;
        }
        __syncthreads();                                            // ring row a-2 is free, red[par] is complete
        if (tid == 0) {
            const int idx = a - a0 + RINGX;                         // cell a-2+RINGX replaces cell a-2
            if (rows_first + idx <= rows_last && a + 1 < a1) {
                int miss;
                const double *src = row_ptr<DIR>(P, fcur, rows_first + idx, line, &miss) + q0;
                mbar_expect_tx(&bars[idx % RINGX], bytes);
                tma_load_1d(ring + (size_t)(idx % RINGX) * Qs, src, bytes, &bars[idx % RINGX]);
            }
        }
        if (tid < 11) {
            double sum = 0.0;
            for (int w = 0; w < nwarp; ++w) sum += redp[w * NMOM + tid];
            const size_t face = DIR == 0 ? (size_t)line * (P.I + 1) + a : (size_t)a * P.I + line;
            P.mom[DIR][(face * P.nchunk + chunk) * NMOM + tid] = sum;
        }
    }
}

size_t smem_face_moments(const UgksParams &P)
{
    const size_t Qs = ((size_t)P.chunk_m * P.Nu + 1) & ~(size_t)1;
    return (RINGX * Qs + 2 * (size_t)P.chunk_m + 2 * 32 * NMOM) * sizeof(double) + RINGX * sizeof(uint64_t);
}

static int block_threads(const UgksParams &P) { return ((P.Nu * P.R + 31) / 32) * 32; }

int launch_face_moments(const UgksParams &P, int cur, int dir, cudaStream_t st)
{
    const size_t smem = smem_face_moments(P);
    const int nsx = (P.I + 1 + P.strip - 1) / P.strip, nsy = (P.J + 1 + P.strip - 1) / P.strip;
    const int T = block_threads(P);
    if (T <= 256) {
        if (dir == 0) k_face_moments<0, 256><<<P.J * nsx * P.nchunk, T, smem, st>>>(P, cur);
        else k_face_moments<1, 256><<<P.I * nsy * P.nchunk, T, smem, st>>>(P, cur);
    } else {
        if (dir == 0) k_face_moments<0, 1024><<<P.J * nsx * P.nchunk, T, smem, st>>>(P, cur);
        else k_face_moments<1, 1024><<<P.I * nsy * P.nchunk, T, smem, st>>>(P, cur);
    }
    return 1;
}

int setup_moments_attributes(const UgksParams &P)
{
    const int smem = (int)smem_face_moments(P);
    cudaError_t e = cudaFuncSetAttribute(k_face_moments<0, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_face_moments<1, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_face_moments<0, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_face_moments<1, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    return e == cudaSuccess ? 0 : 1;
}
