// radial.cu -- the radial Fourier-Laguerre contraction of the ball transform (step a10 of DESIGN.md).
//
//   forward  (Eq. 7, by Gauss-Laguerre quadrature):  f_{lmp}   = sum_i [q_i K_p(r_i)] f_lm(r_i)
//   inverse  (Eq. 8):                                f_lm(r_i) = sum_p K_p(r_i) f_{lmp}
// and the same with the radial wavelet profile kappa^{j'}(p) folded into the matrix (Eq. A9) on the P_j'-node
// grid of scale j'.  All of them are one real matrix A[R][K] applied to K complex "shell" arrays of `cols` entries:
//
//   out[r][c] (+)= wout[r][l(c)] * sum_k A[r][k] * win[k][l(c)] * in[k][c],      l(c) = c mod Lfull,
//
// where the optional real weights win / wout carry the (p, l)-dependent scaling filter sqrt(4pi/(2l+1)) Phi_{l0p}
// (Eq. 35; it is not separable, reading R9).  A dense fp64 contraction: 64 x 64 output tile per block,
// 4 rows x 4 complex columns per thread, operands staged through shared memory in k-chunks of 16.
#include "kernels.h"

namespace s2w {

namespace {

#define RAD_TR 64   // rows per block
#define RAD_TC 64   // complex columns per block
#define RAD_TK 16   // k-chunk

__global__ void __launch_bounds__(256) radial_kernel(const double *__restrict__ A, int R, int K,
                                                    const cplx *__restrict__ in, cplx *__restrict__ out, size_t cols,
                                                    int Lfull, const double *__restrict__ win,
                                                    const double *__restrict__ wout, int accumulate)
{
    __shared__ double sA[RAD_TK][RAD_TR + 1];
    __shared__ cplx sX[RAD_TK][RAD_TC];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;  // tx: column group, ty: row group
    const size_t c0 = (size_t)blockIdx.x * RAD_TC;
    const int r0 = blockIdx.y * RAD_TR;

    cplx acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = cmake(0.0, 0.0);

    for (int k0 = 0; k0 < K; k0 += RAD_TK) {
        __syncthreads();
        for (int e = threadIdx.x; e < RAD_TK * RAD_TR; e += 256) {
            const int kk = e & (RAD_TK - 1), rr = e >> 4;
            const int r = r0 + rr, k = k0 + kk;
            sA[kk][rr] = (r < R && k < K) ? A[(size_t)r * K + k] : 0.0;
        }
        for (int e = threadIdx.x; e < RAD_TK * RAD_TC; e += 256) {
            const int cc = e & (RAD_TC - 1), kk = e >> 6;
            const size_t c = c0 + cc;
            const int k = k0 + kk;
            cplx v = cmake(0.0, 0.0);
            if (c < cols && k < K) {
                v = in[(size_t)k * cols + c];
                if (win) v = cscale(v, win[(size_t)k * Lfull + (int)(c % (size_t)Lfull)]);
            }
            sX[kk][cc] = v;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < RAD_TK; ++kk) {
            double a[4];
            cplx x[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = sA[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) x[j] = sX[kk][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j].x = fma(a[i], x[j].x, acc[i][j].x);
                    acc[i][j].y = fma(a[i], x[j].y, acc[i][j].y);
                }
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = r0 + ty * 4 + i;
        if (r >= R) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const size_t c = c0 + tx + 16 * j;
            if (c >= cols) continue;
            cplx v = acc[i][j];
            if (wout) v = cscale(v, wout[(size_t)r * Lfull + (int)(c % (size_t)Lfull)]);
            cplx *dst = &out[(size_t)r * cols + c];
            if (accumulate) v = cadd(v, *dst);
            *dst = v;
        }
    }
}

}  // namespace

int launch_radial(const double *A, int R, int K, const cplx *in, cplx *out, size_t cols, int Lfull, const double *win,
                  const double *wout, bool accumulate, cudaStream_t st)
{
    if (R <= 0 || cols == 0) return S2W_OK;
    dim3 grid((unsigned)((cols + RAD_TC - 1) / RAD_TC), (R + RAD_TR - 1) / RAD_TR);
    S2W_LAUNCH_C(S2W_K_RADIAL, radial_kernel, grid, 256, 0, st, A, R, K, in, out, cols, Lfull, win, wout,
                 accumulate ? 1 : 0);
    return S2W_OK;
}

}  // namespace s2w
