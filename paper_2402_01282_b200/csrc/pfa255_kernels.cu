// pfa255_kernels.cu -- row a8 (alpha, gamma DFT; Eq. 5/47 and Eq. 48, P:68 / P:426-431) for complex signals on grids
// with L_j = 128: 2 L_j - 1 = 255 = 3 x 5 x 17 alpha samples.
//
// The Bluestein kernels (fft16_kernels.cu) turn a length-255 DFT into two power-of-two transforms of length 512 plus
// three chirp products: about 55 000 FP64 instructions per sequence, and ncu showed them at the FP64 pipe (56 % busy,
// DRAM at a quarter of its roof; profiles/r02e_ball_c5.md).  255 is a product of three coprime factors, so the
// prime-factor (Good-Thomas) map turns the DFT into a 3 x 5 x 17 three-dimensional DFT WITHOUT twiddle factors:
//     input   x[n],  n = (85 n1 + 51 n2 + 15 n3) mod 255,          n1 < 3, n2 < 5, n3 < 17
//     output  X[k],  k = (85 k1 + 51 k2 + 120 k3) mod 255          (k = k1 mod 3 = k2 mod 5 = k3 mod 17)
//     n k = 85 n1 k1 + 51 n2 k2 + 15 n3 k3  (mod 255): X = DFT3 x DFT5 x DFT17 of x
// -- 85 + 51 short DFTs in registers and 15 direct 17-point DFTs (even/odd halves: 16 real 8 x 8 products), about
// 11 000 FP64 instructions per sequence, no chirp, no padding.  The index shift m = k - 127 of the harmonic index is a
// rotation of the load index (m = k for k < 128, k - 255 above), not a phase.
//
// A block of 256 threads works on 15 sequences per round: the NN rows n of RB = 15 / NN rings, so the gamma DFT of a ring
// (3 rows <-> 2N-1 samples) is done on the way in / out.  Stage 1: thread (sequence, n3) does the 3 x 5 part of its 15
// elements in registers (255 work items); stage 2: thread (sequence, k1, k2) does the 17-point DFT (225 items); both in
// place in shared memory, so the result sits in natural order k.  F[b][row][t][m + L-1], W[b][g][t][a], complex.
#include "common.cuh"
#include "fft_core.cuh"
#include "kernels.h"
#include "smem_attr.cuh"

namespace s2w {

namespace {

#define PFA_N 255
#define PFA_SEQS 15
#define PFA_STRIDE 257  // elements between the sequences of a round (odd: the lanes of two sequences spread over the banks)

__device__ __forceinline__ int pfa_wrap(int p) { return p >= PFA_N ? p - PFA_N : p; }

__device__ __forceinline__ cplx pfa_cis(int num, int den)  // exp(2 pi i num / den)
{
    int r = num % den;
    if (r < 0) r += den;
    double s, c;
    sincospi(2.0 * (double)r / (double)den, &s, &c);
    return cmake(c, s);
}

#define PFA_S3 0.86602540378443864676   // sin(2 pi / 3)
#define PFA_C51 0.30901699437494742410  // cos(2 pi / 5)
#define PFA_C52 (-0.80901699437494742410)
#define PFA_S51 0.95105651629515357212  // sin(2 pi / 5)
#define PFA_S52 0.58778525229247312917  // sin(4 pi / 5)

// X_k = sum_j x_j e^{-/+ 2 pi i j k / 3} (upper sign: INV = false)
template <bool INV>
__device__ __forceinline__ void pfa_dft3(cplx &x0, cplx &x1, cplx &x2)
{
    const cplx a = cadd(x1, x2), b = csub(x1, x2);
    const cplx t = cmake(fma(-0.5, a.x, x0.x), fma(-0.5, a.y, x0.y));
    const double br = PFA_S3 * b.x, bi = PFA_S3 * b.y;
    x0 = cadd(x0, a);
    x1 = INV ? cmake(t.x - bi, t.y + br) : cmake(t.x + bi, t.y - br);
    x2 = INV ? cmake(t.x + bi, t.y - br) : cmake(t.x - bi, t.y + br);
}

template <bool INV>
__device__ __forceinline__ void pfa_dft5(cplx &x0, cplx &x1, cplx &x2, cplx &x3, cplx &x4)
{
    const cplx a1 = cadd(x1, x4), a2 = cadd(x2, x3), b1 = csub(x1, x4), b2 = csub(x2, x3);
    const cplx A1 = cmake(fma(PFA_C52, a2.x, fma(PFA_C51, a1.x, x0.x)), fma(PFA_C52, a2.y, fma(PFA_C51, a1.y, x0.y)));
    const cplx A2 = cmake(fma(PFA_C51, a2.x, fma(PFA_C52, a1.x, x0.x)), fma(PFA_C51, a2.y, fma(PFA_C52, a1.y, x0.y)));
    const cplx B1 = cmake(fma(PFA_S52, b2.x, PFA_S51 * b1.x), fma(PFA_S52, b2.y, PFA_S51 * b1.y));
    const cplx B2 = cmake(fma(-PFA_S51, b2.x, PFA_S52 * b1.x), fma(-PFA_S51, b2.y, PFA_S52 * b1.y));
    x0 = cadd(x0, cadd(a1, a2));
    // X_k = A_k -/+ i B_k, X_{5-k} = A_k +/- i B_k
    x1 = INV ? cmake(A1.x - B1.y, A1.y + B1.x) : cmake(A1.x + B1.y, A1.y - B1.x);
    x4 = INV ? cmake(A1.x + B1.y, A1.y - B1.x) : cmake(A1.x - B1.y, A1.y + B1.x);
    x2 = INV ? cmake(A2.x - B2.y, A2.y + B2.x) : cmake(A2.x + B2.y, A2.y - B2.x);
    x3 = INV ? cmake(A2.x + B2.y, A2.y - B2.x) : cmake(A2.x - B2.y, A2.y + B2.x);
}

// stage 1: the 3 x 5 part at fixed n3, in place: slot (n1, n2, n3) lives at (85 n1 + 51 n2 + 15 n3) mod 255
template <bool INV>
__device__ __forceinline__ void pfa_stage35(cplx *seq, int n3)
{
    const int b3 = 15 * n3;
    cplx x[3][5];
#pragma unroll
    for (int n1 = 0; n1 < 3; ++n1)
#pragma unroll
        for (int n2 = 0; n2 < 5; ++n2) x[n1][n2] = seq[pfa_wrap(b3 + (85 * n1 + 51 * n2) % PFA_N)];
#pragma unroll
    for (int n2 = 0; n2 < 5; ++n2) pfa_dft3<INV>(x[0][n2], x[1][n2], x[2][n2]);
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1) pfa_dft5<INV>(x[k1][0], x[k1][1], x[k1][2], x[k1][3], x[k1][4]);
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1)
#pragma unroll
        for (int k2 = 0; k2 < 5; ++k2) seq[pfa_wrap(b3 + (85 * k1 + 51 * k2) % PFA_N)] = x[k1][k2];
}

// stage 2: the 17-point DFT over n3 at fixed (k1, k2): reads (base + 15 n3) mod 255, writes X[k] at its natural position
// k = (base + 120 k3) mod 255 -- the same 17 positions, read completely before the first store
template <bool INV>
__device__ __forceinline__ void pfa_stage17(cplx *seq, int base)
{
    cplx a[8], b[8];
    const cplx x0 = seq[base];
#pragma unroll
    for (int j = 1; j <= 8; ++j) {
        const cplx p = seq[pfa_wrap(base + 15 * j)], q = seq[pfa_wrap(base + (15 * (17 - j)) % PFA_N)];
        a[j - 1] = cadd(p, q);
        b[j - 1] = csub(p, q);
    }
#include "pfa255_dft17.inc"
}

// the two transform stages of a round of PFA_SEQS sequences (block-wide barriers inside)
template <bool INV>
__device__ __forceinline__ void pfa_round(cplx *buf)
{
    const int tid = threadIdx.x;
    __syncthreads();
    if (tid < PFA_SEQS * 17) pfa_stage35<INV>(buf + (tid / 17) * PFA_STRIDE, tid % 17);
    __syncthreads();
    if (tid < PFA_SEQS * 15) {
        const int j = tid % 15;
        pfa_stage17<INV>(buf + (tid / 15) * PFA_STRIDE, (85 * (j / 5) + 51 * (j % 5)) % PFA_N);
    }
    __syncthreads();
}

// analysis side: F -> W(gamma_g, beta_t, alpha_a) = sum_{m,n} F_mn(beta_t) e^{i(m alpha_a + n gamma_g)}
template <int NN>
__global__ void __launch_bounds__(256, 3) so3_inv_pfa255_kernel(const cplx *__restrict__ F, cplx *__restrict__ W,
                                                               size_t sig_stride, So3Args A, int L)
{
    constexpr int RB = PFA_SEQS / NN;
    extern __shared__ cplx buf[];
    __shared__ cplx gph[NN * 64];
    const int n = PFA_N, ng = 2 * A.N - 1, tid = threadIdx.x;
    const cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * n;
    cplx *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    for (int e = tid; e < NN * ng; e += 256) gph[e] = pfa_cis(A.n_val[e / ng] * (e % ng), ng);
    if (tid < n) {
        const int mo = (L - 1) + (tid < L ? tid : tid - n);  // DFT index k = tid <-> m = k or k - 255
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int t = blockIdx.x * RB + r;
#pragma unroll
            for (int i = 0; i < NN; ++i)
                buf[(r * NN + i) * PFA_STRIDE + tid] =
                    t < L ? Fb[((size_t)A.n_row[i] * L + t) * n + mo] : cmake(0.0, 0.0);
        }
    }
    pfa_round<true>(buf);
    if (tid < n) {
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int t = blockIdx.x * RB + r;
            if (t >= L) continue;
            cplx v[NN];
#pragma unroll
            for (int i = 0; i < NN; ++i) v[i] = buf[(r * NN + i) * PFA_STRIDE + tid];
            cplx *Wr = Wb + (size_t)t * n + tid;
            for (int g = 0; g < ng; ++g) {
                cplx o = cmul(gph[g], v[0]);
#pragma unroll
                for (int i = 1; i < NN; ++i) o = cadd(o, cmul(gph[i * ng + g], v[i]));
                Wr[(size_t)g * plane] = o;
            }
        }
    }
}

// synthesis side: F_mn(beta_t) = 1/(n_a n_g) sum_{a,g} W e^{-i(m alpha_a + n gamma_g)}
template <int NN>
__global__ void __launch_bounds__(256, 3) so3_fwd_pfa255_kernel(const cplx *__restrict__ W, cplx *__restrict__ F,
                                                               size_t sig_stride, So3Args A, int L)
{
    constexpr int RB = PFA_SEQS / NN;
    extern __shared__ cplx buf[];
    __shared__ cplx gph[NN * 64];
    const int n = PFA_N, ng = 2 * A.N - 1, tid = threadIdx.x;
    const double scale = 1.0 / ((double)ng * (double)n);
    cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * n;
    const cplx *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    for (int e = tid; e < NN * ng; e += 256) gph[e] = pfa_cis(-A.n_val[e / ng] * (e % ng), ng);
    __syncthreads();
    if (tid < n) {
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int t = blockIdx.x * RB + r;
            cplx y[NN];
#pragma unroll
            for (int i = 0; i < NN; ++i) y[i] = cmake(0.0, 0.0);
            if (t < L) {
                const cplx *Wr = Wb + (size_t)t * n + tid;
                for (int g = 0; g < ng; ++g) {
                    const cplx wv = Wr[(size_t)g * plane];
#pragma unroll
                    for (int i = 0; i < NN; ++i) y[i] = cadd(y[i], cmul(gph[i * ng + g], wv));
                }
            }
#pragma unroll
            for (int i = 0; i < NN; ++i) buf[(r * NN + i) * PFA_STRIDE + tid] = cscale(y[i], scale);
        }
    }
    pfa_round<false>(buf);
    if (tid < n) {
        const int mo = (L - 1) + (tid < L ? tid : tid - n);
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int t = blockIdx.x * RB + r;
            if (t >= L) continue;
#pragma unroll
            for (int i = 0; i < NN; ++i) {
                const cplx v = buf[(r * NN + i) * PFA_STRIDE + tid];
                if (A.f_transposed)
                    Fb[((size_t)A.n_row[i] * n + mo) * L + t] = v;   // [row][m][t]: runs of RB rings per (row, m)
                else
                    Fb[((size_t)A.n_row[i] * L + t) * n + mo] = v;
            }
        }
    }
}

// a1 ring FFTs (Eqs. 2-3) of complex signals on the 255-sample grids (the ball's shells): 15 rings per block;
// layouts and normalisation as ring_fwd16_kernel / ring_inv16_kernel (fft16_kernels.cu): pixel rows [batch][L][n], row r of
// the spectrum array holds F_m at [m + L-1]
__global__ void __launch_bounds__(256, 3) ring_fwd_pfa255_kernel(const cplx *__restrict__ in, cplx *__restrict__ out, int nrows,
                                                                size_t sig_stride, int L)
{
    extern __shared__ cplx buf[];
    const int n = PFA_N, tid = threadIdx.x;
    const double inv_n = 1.0 / (double)n;
    if (tid < n) {
#pragma unroll
        for (int q = 0; q < PFA_SEQS; ++q) {
            const int r = blockIdx.x * PFA_SEQS + q;
            buf[q * PFA_STRIDE + tid] =
                r < nrows ? in[(size_t)(r / L) * sig_stride + (size_t)(r % L) * n + tid] : cmake(0.0, 0.0);
        }
    }
    pfa_round<false>(buf);
    if (tid < n) {
        const int mo = (L - 1) + (tid < L ? tid : tid - n);
#pragma unroll
        for (int q = 0; q < PFA_SEQS; ++q) {
            const int r = blockIdx.x * PFA_SEQS + q;
            if (r < nrows) out[(size_t)r * n + mo] = cscale(buf[q * PFA_STRIDE + tid], inv_n);
        }
    }
}

__global__ void __launch_bounds__(256, 3) ring_inv_pfa255_kernel(const cplx *__restrict__ in, cplx *__restrict__ out, int nrows,
                                                                size_t sig_stride, int L)
{
    extern __shared__ cplx buf[];
    const int n = PFA_N, tid = threadIdx.x;
    if (tid < n) {
        const int mo = (L - 1) + (tid < L ? tid : tid - n);
#pragma unroll
        for (int q = 0; q < PFA_SEQS; ++q) {
            const int r = blockIdx.x * PFA_SEQS + q;
            buf[q * PFA_STRIDE + tid] = r < nrows ? in[(size_t)r * n + mo] : cmake(0.0, 0.0);
        }
    }
    pfa_round<true>(buf);
    if (tid < n) {
#pragma unroll
        for (int q = 0; q < PFA_SEQS; ++q) {
            const int r = blockIdx.x * PFA_SEQS + q;
            if (r < nrows) out[(size_t)(r / L) * sig_stride + (size_t)(r % L) * n + tid] = buf[q * PFA_STRIDE + tid];
        }
    }
}

template <int NN>
int so3_pfa255_t(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, int L, cudaStream_t st)
{
    constexpr int RB = PFA_SEQS / NN;
    const size_t sm = (size_t)PFA_SEQS * PFA_STRIDE * sizeof(cplx);
    int rc;
    for (int b0 = 0; b0 < batch; b0 += 65535) {
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        if (b0) {
            set_error("launch_so3_pfa255: more than 65535 signals per launch");
            return S2W_EUNSUPPORTED;
        }
        dim3 grid((L + RB - 1) / RB, nb);
        if (fwd) {
            if ((rc = set_smem(so3_fwd_pfa255_kernel<NN>, sm))) return rc;
            S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_fwd_pfa255_kernel<NN>), grid, 256, sm, st, (const cplx *)in, (cplx *)out,
                         sig_stride, A, L);
        } else {
            if ((rc = set_smem(so3_inv_pfa255_kernel<NN>, sm))) return rc;
            S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_inv_pfa255_kernel<NN>), grid, 256, sm, st, (const cplx *)in, (cplx *)out,
                         sig_stride, A, L);
        }
    }
    return S2W_OK;
}

}  // namespace

bool so3_pfa255_supported(const So3Args &A, const FftTab &T)
{
    static const bool on = [] {
        const char *e = getenv("S2W_PFA");
        return !(e && e[0] == '0');
    }();
    return on && T.n == PFA_N && T.L == 128 && T.nt == T.L && A.nn >= 1 && A.nn <= 3 && 2 * A.N - 1 <= 64;
}

bool ring_pfa255_supported(bool real, const FftTab &T)
{
    static const bool on = [] {
        const char *e = getenv("S2W_PFA");
        return !(e && e[0] == '0');
    }();
    return on && !real && T.n == PFA_N && T.L == 128 && T.nt == T.L;
}

// complex signals, nrows = batch x L rings of 255 samples; the caller checks ring_pfa255_supported
int launch_ring_pfa255(bool fwd, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T, cudaStream_t st)
{
    const size_t sm = (size_t)PFA_SEQS * PFA_STRIDE * sizeof(cplx);
    const int grid = (nrows + PFA_SEQS - 1) / PFA_SEQS;
    int rc;
    if (fwd) {
        if ((rc = set_smem(ring_fwd_pfa255_kernel, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_fwd_pfa255_kernel, grid, 256, sm, st, (const cplx *)in, (cplx *)out, nrows, sig_stride,
                     T.L);
    } else {
        if ((rc = set_smem(ring_inv_pfa255_kernel, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_inv_pfa255_kernel, grid, 256, sm, st, (const cplx *)in, (cplx *)out, nrows, sig_stride,
                     T.L);
    }
    return S2W_OK;
}

// complex signals on the McEwen-Wiaux grid of L_j = 128; the caller checks so3_pfa255_supported
int launch_so3_pfa255(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                      cudaStream_t st)
{
    if (A.nn == 1) return so3_pfa255_t<1>(fwd, in, out, sig_stride, A, batch, T.L, st);
    if (A.nn == 2) return so3_pfa255_t<2>(fwd, in, out, sig_stride, A, batch, T.L, st);
    return so3_pfa255_t<3>(fwd, in, out, sig_stride, A, batch, T.L, st);
}

}  // namespace s2w
