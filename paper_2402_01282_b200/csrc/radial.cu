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
// (Eq. 35; it is not separable, reading R9).  A dense fp64 contraction on the FP64 tensor pipe
// (mma.sync.m8n8k4.f64): 64 rows x 64 complex columns per block, operands staged through shared memory.
#include "kernels.h"
#include "smem_attr.cuh"

namespace s2w {

namespace {

#define RAD_TR 64    // rows per block
#define RAD_TC 128   // real columns (64 complex) per block
#define RAD_TK 16    // k-chunk
#define RAD_SA 20    // row stride of the A tile (doubles): the A-fragment reads (8 rows x 4 k) of a half-warp hit 16 bank pairs
#define RAD_SB 132   // row stride of the B tile: 4 k-rows x 8 columns of a fragment land in distinct banks
#define RAD_STAGES 3
#define RAD_STAGE_DOUBLES (RAD_TR * RAD_SA + RAD_TK * RAD_SB)

__device__ __forceinline__ void dmma884_r(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
// asynchronous global -> shared copies (LDGSTS); src_bytes = 0 zero-fills the destination
__device__ __forceinline__ void cp_async8(void *dst, const void *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async16z(void *dst, const void *src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}

// FP64 tensor pipe: D[row][col] += A[row][k] B[k][col] with the complex shell arrays read as 2 cols real columns.
// Block = 64 rows x 128 real columns, 8 warps of 16 rows x 64 columns (2 x 8 accumulator fragments).  The k-chunks of 16
// travel through a ring of three shared-memory stages filled by cp.async two chunks ahead (one barrier per chunk; the
// round-1 kernel staged each chunk with plain loads between two barriers and reached 0.29 of the FP64 peak).  WIN: the
// input weight w_in has to be applied while staging B, so that variant (two launches per ball transform) keeps the
// synchronous staging.
template <bool WIN>
__global__ void __launch_bounds__(256, 2) radial_kernel(const double *__restrict__ A, int R, int K,
                                                       const cplx *__restrict__ in, cplx *__restrict__ out, size_t cols,
                                                       int Lfull, const double *__restrict__ win,
                                                       const double *__restrict__ wout, int accumulate,
                                                       const int2 *__restrict__ krange)
{
    extern __shared__ __align__(16) double s_rad[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int fr = lane >> 2, fk = lane & 3;
    const int wr0 = (warp & 3) * 16, wc0 = (warp >> 2) * 64;  // this warp's rows / real columns inside the block tile
    const size_t dc0 = (size_t)blockIdx.x * RAD_TC;            // first real column of the block
    const int r0 = blockIdx.y * RAD_TR;

    double acc[2][8][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // block-sparse stacked matrices (ball, all radial scales in one launch): only [kbeg, kend) of this row tile holds
    // non-zeros
    const int kbeg = krange ? (krange[blockIdx.y].x / RAD_TK) * RAD_TK : 0;
    const int kend = krange ? min(krange[blockIdx.y].y, K) : K;
    const int nchunk = (kend - kbeg + RAD_TK - 1) / RAD_TK;

    auto stage_async = [&](int ch) {  // chunk ch -> stage ch % RAD_STAGES
        double *sA = s_rad + (size_t)(ch % RAD_STAGES) * RAD_STAGE_DOUBLES, *sB = sA + RAD_TR * RAD_SA;
        const int k0 = kbeg + ch * RAD_TK;
#pragma unroll
        for (int e = threadIdx.x; e < RAD_TR * RAD_TK; e += 256) {
            const int kk = e & (RAD_TK - 1), rr = e >> 4;
            const int r = r0 + rr, k = k0 + kk;
            const bool ok = r < R && k < kend;
            cp_async8(&sA[rr * RAD_SA + kk], ok ? &A[(size_t)r * K + k] : A, ok ? 8 : 0);
        }
#pragma unroll
        for (int e = threadIdx.x; e < RAD_TK * (RAD_TC / 2); e += 256) {
            const int cc = e & (RAD_TC / 2 - 1), kk = e >> 6;
            const size_t c = dc0 / 2 + cc;
            const int k = k0 + kk;
            const bool ok = c < cols && k < kend;
            cp_async16z(&sB[kk * RAD_SB + 2 * cc], ok ? &in[(size_t)k * cols + c] : in, ok ? 16 : 0);
        }
    };
    auto stage_sync = [&](int ch) {
        double *sA = s_rad + (size_t)(ch % RAD_STAGES) * RAD_STAGE_DOUBLES, *sB = sA + RAD_TR * RAD_SA;
        const int k0 = kbeg + ch * RAD_TK;
        for (int e = threadIdx.x; e < RAD_TR * RAD_TK; e += 256) {
            const int kk = e & (RAD_TK - 1), rr = e >> 4;
            const int r = r0 + rr, k = k0 + kk;
            sA[rr * RAD_SA + kk] = (r < R && k < kend) ? A[(size_t)r * K + k] : 0.0;
        }
        for (int e = threadIdx.x; e < RAD_TK * (RAD_TC / 2); e += 256) {
            const int cc = e & (RAD_TC / 2 - 1), kk = e >> 6;
            const size_t c = dc0 / 2 + cc;
            const int k = k0 + kk;
            cplx v = cmake(0.0, 0.0);
            if (c < cols && k < kend) {
                v = in[(size_t)k * cols + c];
                v = cscale(v, win[(size_t)k * Lfull + (int)(c % (size_t)Lfull)]);
            }
            *reinterpret_cast<cplx *>(&sB[kk * RAD_SB + 2 * cc]) = v;
        }
    };

    if (!WIN) {
        for (int ch = 0; ch < RAD_STAGES - 1; ++ch) {
            if (ch < nchunk) stage_async(ch);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
    }
    for (int ch = 0; ch < nchunk; ++ch) {
        if (WIN) {
            __syncthreads();  // the previous chunk has been consumed
            stage_sync(ch);
            __syncthreads();
        } else {
            asm volatile("cp.async.wait_group %0;" ::"n"(RAD_STAGES - 2) : "memory");  // this thread's copies of chunk ch
            __syncthreads();  // everyone's copies of chunk ch have landed; chunk ch - 1 has been consumed by all
            if (ch + RAD_STAGES - 1 < nchunk) stage_async(ch + RAD_STAGES - 1);  // into the stage chunk ch - 1 used
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        const double *sA = s_rad + (size_t)(ch % RAD_STAGES) * RAD_STAGE_DOUBLES, *sB = sA + RAD_TR * RAD_SA;
#pragma unroll
        for (int kq = 0; kq < RAD_TK; kq += 4) {
            const double a0 = sA[(wr0 + fr) * RAD_SA + kq + fk], a1 = sA[(wr0 + 8 + fr) * RAD_SA + kq + fk];
            const double *brow = sB + (kq + fk) * RAD_SB + wc0 + fr;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const double b = brow[8 * j];
                dmma884_r(acc[0][j][0], acc[0][j][1], a0, b);
                dmma884_r(acc[1][j][0], acc[1][j][1], a1, b);
            }
        }
    }
    // D fragment: row fr of the octet, real columns 2 fk + {0, 1} = one complex element
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int r = r0 + wr0 + 8 * i + fr;
        if (r >= R) continue;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const size_t c = (dc0 + wc0 + 8 * j) / 2 + fk;
            if (c >= cols) continue;
            cplx v = cmake(acc[i][j][0], acc[i][j][1]);
            if (wout) v = cscale(v, wout[(size_t)r * Lfull + (int)(c % (size_t)Lfull)]);
            cplx *dst = &out[(size_t)r * cols + c];
            if (accumulate) v = cadd(v, *dst);
            *dst = v;
        }
    }
}

}  // namespace

int launch_radial(const double *A, int R, int K, const cplx *in, cplx *out, size_t cols, int Lfull, const double *win,
                  const double *wout, bool accumulate, cudaStream_t st, const int2 *krange)
{
    if (R <= 0 || cols == 0) return S2W_OK;
    dim3 grid((unsigned)((2 * cols + RAD_TC - 1) / RAD_TC), (R + RAD_TR - 1) / RAD_TR);
    const size_t sm = (size_t)RAD_STAGES * RAD_STAGE_DOUBLES * sizeof(double);
    int rc;
    if (win) {
        if ((rc = set_smem(radial_kernel<true>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RADIAL, radial_kernel<true>, grid, 256, sm, st, A, R, K, in, out, cols, Lfull, win, wout,
                     accumulate ? 1 : 0, krange);
    } else {
        if ((rc = set_smem(radial_kernel<false>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RADIAL, radial_kernel<false>, grid, 256, sm, st, A, R, K, in, out, cols, Lfull, win, wout,
                     accumulate ? 1 : 0, krange);
    }
    return S2W_OK;
}

}  // namespace s2w
