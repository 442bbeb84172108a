// ring_fft.cu -- batched odd-length fp64 DFTs along phi / alpha (steps a1 and a8 of DESIGN.md) and the MW
// theta-quadrature reweighting (step a2), all as Bluestein chirp convolutions on fft_core.cuh.
//
//   a1  F_m(theta_t) = (1/n) sum_p f(theta_t, phi_p) e^{-i m phi_p},  n = 2L-1                      (Eq. 2)
//   a8  W(gamma_g, beta_t, alpha_a) = sum_{m,n} F_mn(beta_t) e^{i(m alpha_a + n gamma_g)}            (Eq. 5/47)
//       F_mn(beta_t) = 1/(n_a n_g) sum_{a,g} W e^{-i(m alpha_a + n gamma_g)}                         (Eq. 48)
//   a2  h = fold(DFT^-1(w * DFT(extend(F))))  per (m,n) column along theta                          (R3)
//
// Real signals: W real  <=>  F_{-m,-n} = conj(F_mn).  The harmonic-side arrays then hold m = 0..L-1 only, two real
// rings share one complex DFT in a1, and a8 transforms only the rows n >= 0.
#include <cstdlib>

#include "fft_core.cuh"
#include "kernels.h"
#include "smem_attr.cuh"

namespace s2w {

namespace {

__device__ __forceinline__ cplx cis_2pi_frac(int num, int den)  // exp(2 pi i num/den), num reduced mod den
{
    int r = num % den;
    if (r < 0) r += den;
    double s, c;
    sincospi(2.0 * (double)r / (double)den, &s, &c);
    return cmake(c, s);
}

// ---------------------------------------------------------------------------------------------------------------
// a1 forward: pixels -> F_m.  Real: one block per pair of rows, out[row][m], m = 0..L-1.
//                              Complex: one block per row, out[row][m+L-1].
// ---------------------------------------------------------------------------------------------------------------
template <bool REAL>
__global__ void __launch_bounds__(256, 3) ring_fwd_kernel(const void *__restrict__ in, cplx *__restrict__ out, int nrows,
                                                      size_t sig_stride, FftTab T)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const double inv_n = 1.0 / (double)n;
    if (REAL) {
        const int r0 = 2 * blockIdx.x, r1 = r0 + 1;
        const bool has1 = r1 < nrows;
        const double *x0 = (const double *)in + (size_t)(r0 / T.nt) * sig_stride + (size_t)(r0 % T.nt) * n;
        const double *x1 = (const double *)in + (size_t)(r1 / T.nt) * sig_stride + (size_t)(r1 % T.nt) * n;
        for (int p = threadIdx.x; p < M; p += blockDim.x) {
            cplx v = cmake(0.0, 0.0);
            if (p < n) v = cmul(cmake(x0[p], has1 ? x1[p] : 0.0), __ldg(&T.chirp[p]));
            buf[S2W_PAD(p)] = v;
        }
        __syncthreads();
        fft_convolve<true>(buf, T, s_tw, T.bhat_m);
        for (int k = threadIdx.x; k < n; k += blockDim.x) buf[S2W_PAD(k)] = cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]));
        __syncthreads();
        for (int m = threadIdx.x; m < L; m += blockDim.x) {
            cplx a = buf[S2W_PAD(m)], b = cconj(buf[S2W_PAD(m == 0 ? 0 : n - m)]);
            cplx s = cadd(a, b), d = csub(a, b);
            out[(size_t)r0 * L + m] = cscale(s, 0.5 * inv_n);
            if (has1) out[(size_t)r1 * L + m] = cmake(0.5 * inv_n * d.y, -0.5 * inv_n * d.x);
        }
    } else {
        const int r0 = blockIdx.x;
        const cplx *x0 = (const cplx *)in + (size_t)(r0 / T.nt) * sig_stride + (size_t)(r0 % T.nt) * n;
        for (int p = threadIdx.x; p < M; p += blockDim.x) {
            cplx v = cmake(0.0, 0.0);
            if (p < n) v = cmul(x0[p], __ldg(&T.chirp[p]));
            buf[S2W_PAD(p)] = v;
        }
        __syncthreads();
        fft_convolve<true>(buf, T, s_tw, T.bhat_m);
        for (int mi = threadIdx.x; mi < n; mi += blockDim.x) {
            int m = mi - (L - 1);
            int k = m < 0 ? m + n : m;
            out[(size_t)r0 * n + mi] = cscale(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k])), inv_n);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a1 inverse: F_m -> pixels, f = sum_m F_m e^{i m phi_p}.
// ---------------------------------------------------------------------------------------------------------------
template <bool REAL>
__global__ void __launch_bounds__(256, 3) ring_inv_kernel(const cplx *__restrict__ in, void *__restrict__ out, int nrows,
                                                      size_t sig_stride, FftTab T)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    if (REAL) {
        const int r0 = 2 * blockIdx.x, r1 = r0 + 1;
        const bool has1 = r1 < nrows;
        const cplx *X0 = in + (size_t)r0 * L;
        const cplx *X1 = in + (size_t)r1 * L;
        for (int k = threadIdx.x; k < M; k += blockDim.x) {
            cplx v = cmake(0.0, 0.0);
            if (k < n) {
                int m = k < L ? k : n - k;  // |m|
                cplx a = X0[m], b = has1 ? X1[m] : cmake(0.0, 0.0);
                if (k >= L) {
                    a = cconj(a);
                    b = cconj(b);
                }
                // Z_k = A_k + i B_k
                v = cmulc(cmake(a.x - b.y, a.y + b.x), __ldg(&T.chirp[k]));
            }
            buf[S2W_PAD(k)] = v;
        }
        __syncthreads();
        fft_convolve<true>(buf, T, s_tw, T.bhat_p);
        double *y0 = (double *)out + (size_t)(r0 / T.nt) * sig_stride + (size_t)(r0 % T.nt) * n;
        double *y1 = (double *)out + (size_t)(r1 / T.nt) * sig_stride + (size_t)(r1 % T.nt) * n;
        for (int p = threadIdx.x; p < n; p += blockDim.x) {
            cplx z = cmulc(buf[S2W_PAD(p)], __ldg(&T.chirp[p]));
            y0[p] = z.x;
            if (has1) y1[p] = z.y;
        }
    } else {
        const int r0 = blockIdx.x;
        const cplx *X0 = in + (size_t)r0 * n;
        for (int k = threadIdx.x; k < M; k += blockDim.x) {
            cplx v = cmake(0.0, 0.0);
            if (k < n) {
                int m = k < L ? k : k - n;
                v = cmulc(X0[m + L - 1], __ldg(&T.chirp[k]));
            }
            buf[S2W_PAD(k)] = v;
        }
        __syncthreads();
        fft_convolve<true>(buf, T, s_tw, T.bhat_p);
        cplx *y0 = (cplx *)out + (size_t)(r0 / T.nt) * sig_stride + (size_t)(r0 % T.nt) * n;
        for (int p = threadIdx.x; p < n; p += blockDim.x) y0[p] = cmulc(buf[S2W_PAD(p)], __ldg(&T.chirp[p]));
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a8 analysis: F[b][row][t][mi] -> W[b][g][t][a].  One block per (b, t); loops over the rows n of the scale.
// Real: rows n >= 0 only: V_n(a) = sum_m F_mn e^{i m alpha_a} with F_{-m,n} = conj(F_{m,-n});
//       W = sum_{n>=0} c_n Re(e^{i n gamma_g} V_n), c_0 = 1, c_n = 2.
// ---------------------------------------------------------------------------------------------------------------
// Few gamma samples (real: 2N-1 <= 9, complex: 2N-1 <= 5): no read-modify-write of the gamma planes.  The transforms
// V_n(alpha) of all rows but the last are parked in the ring's own output planes (real: row i in planes 2i, 2i+1;
// complex: row i in plane i), the pass of the last row reads them back -- each thread its own alpha samples, so
// program order is all the ordering needed -- and writes every plane once.
template <bool REAL, bool MULTI>
__device__ __forceinline__ void so3_inv_few(const cplx *__restrict__ F, void *__restrict__ W, size_t sig_stride,
                                            const So3Args &A, const FftTab &T, int rpb, cplx *buf0, const cplx *s_tw,
                                            cplx *gph)
{
    constexpr int NG = REAL ? 9 : 5;  // most gamma samples
    constexpr int NP = 4;             // most parked rows
    const int n = T.n, L = T.L, M = T.M;
    const int bstride = fft_padded_len(M);
    const int tpr = MULTI ? blockDim.x / rpb : blockDim.x;
    const int rl = MULTI ? threadIdx.x / tpr : 0, tl = MULTI ? threadIdx.x - rl * tpr : threadIdx.x;
    cplx *buf = buf0 + (size_t)rl * bstride;
    const int t = MULTI ? blockIdx.x * rpb + rl : blockIdx.x, b = blockIdx.y;
    const bool has = MULTI ? t < T.nt : true;
    const int Md = REAL ? L : n;
    const int ng = 2 * A.N - 1;
    const size_t plane = (size_t)T.nt * n;
    const cplx *Fb = F + (size_t)b * A.nrows * T.nt * Md;
    int nproc = 0;
    for (int q = 0; q < A.nn; ++q) {
        if (REAL && A.n_val[q] < 0) continue;
        for (int g = threadIdx.x; g < ng; g += blockDim.x) {
            cplx ph = cis_2pi_frac(A.n_val[q] * g, ng);
            if (REAL && A.n_val[q] != 0) ph = cscale(ph, 2.0);  // W = V_0 + 2 Re sum_{n>0} e^{i n gamma} V_n
            gph[nproc * ng + g] = ph;
        }
        ++nproc;
    }
    int i = 0;
    for (int q = 0; q < A.nn; ++q) {
        const int nv = A.n_val[q];
        if (REAL && nv < 0) continue;
        const cplx *Fp = Fb + ((size_t)A.n_row[q] * T.nt + t) * Md;   // row of n
        const cplx *Fm = Fb + ((size_t)A.n_rowm[q] * T.nt + t) * Md;  // row of -n
        for (int k0 = tl; k0 < M; k0 += 4 * tpr) {  // four elements at a time, loads first
            cplx x[4], c[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = k0 + j * tpr;
                const int kk = (k < n && has) ? k : 0;
                if (REAL)
                    x[j] = *(kk < L ? Fp + kk : Fm + (n - kk));
                else
                    x[j] = Fp[(kk < L ? kk : kk - n) + L - 1];
                c[j] = __ldg(&T.chirp[kk]);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = k0 + j * tpr;
                if (k >= M) continue;
                const cplx v = (REAL && k >= L) ? cconj(x[j]) : x[j];
                buf[S2W_PAD(k)] = (k < n && has) ? cmulc(v, c[j]) : cmake(0.0, 0.0);
            }
        }
        __syncthreads();
        if (MULTI)
            fft_convolve_b<true>(buf0, T, s_tw, T.bhat_p, rpb, bstride);
        else
            fft_convolve<true>(buf, T, s_tw, T.bhat_p);
        for (int a = tl; a < (has ? n : 0); a += tpr) {
            const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));
            if (REAL) {
                double *Wr = (double *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                if (i + 1 < nproc) {
                    Wr[(size_t)(2 * i) * plane] = v.x;
                    Wr[(size_t)(2 * i + 1) * plane] = v.y;
                } else {
                    double sc[2 * NP];
#pragma unroll
                    for (int k = 0; k < 2 * NP; ++k) sc[k] = k < 2 * i ? Wr[(size_t)k * plane] : 0.0;
                    double out[NG];
#pragma unroll
                    for (int g = 0; g < NG; ++g) {
                        const cplx ph = gph[i * ng + (g < ng ? g : 0)];
                        out[g] = ph.x * v.x - ph.y * v.y;
                    }
#pragma unroll
                    for (int j = 0; j < NP; ++j)
                        if (j < i) {
#pragma unroll
                            for (int g = 0; g < NG; ++g) {
                                const cplx ph = gph[j * ng + (g < ng ? g : 0)];
                                out[g] += ph.x * sc[2 * j] - ph.y * sc[2 * j + 1];
                            }
                        }
#pragma unroll
                    for (int g = 0; g < NG; ++g)
                        if (g < ng) Wr[(size_t)g * plane] = out[g];
                }
            } else {
                cplx *Wc = (cplx *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                if (i + 1 < nproc) {
                    Wc[(size_t)i * plane] = v;
                } else {
                    cplx sc[NP];
#pragma unroll
                    for (int k = 0; k < NP; ++k) sc[k] = k < i ? Wc[(size_t)k * plane] : cmake(0.0, 0.0);
                    cplx out[NG];
#pragma unroll
                    for (int g = 0; g < NG; ++g) out[g] = cmul(gph[i * ng + (g < ng ? g : 0)], v);
#pragma unroll
                    for (int j = 0; j < NP; ++j)
                        if (j < i) {
#pragma unroll
                            for (int g = 0; g < NG; ++g) out[g] = cadd(out[g], cmul(gph[j * ng + (g < ng ? g : 0)], sc[j]));
                        }
#pragma unroll
                    for (int g = 0; g < NG; ++g)
                        if (g < ng) Wc[(size_t)g * plane] = out[g];
                }
            }
        }
        ++i;
        __syncthreads();
    }
}

// MULTI: rpb rings per block (small grids), tpr = blockDim / rpb threads per ring; otherwise one ring per block.
template <bool REAL, bool MULTI>
__global__ void __launch_bounds__(256, 3) so3_inv_kernel(const cplx *__restrict__ F, void *__restrict__ W, size_t sig_stride,
                                                     So3Args A, FftTab T, int rpb)
{
    extern __shared__ cplx buf0[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const int bstride = fft_padded_len(M);
    const int tpr = MULTI ? blockDim.x / rpb : blockDim.x;
    const int rl = MULTI ? threadIdx.x / tpr : 0, tl = MULTI ? threadIdx.x - rl * tpr : threadIdx.x;
    cplx *buf = buf0 + (size_t)rl * bstride;
    const int t = MULTI ? blockIdx.x * rpb + rl : blockIdx.x, b = blockIdx.y;
    const bool has = MULTI ? t < T.nt : true;
    const int Md = REAL ? L : n;
    const int ng = 2 * A.N - 1;
    const cplx *Fb = F + (size_t)b * A.nrows * T.nt * Md;
    __shared__ cplx gph[2 * S2W_MAX_N];
    if (ng <= (REAL ? 9 : 5)) {
        so3_inv_few<REAL, MULTI>(F, W, sig_stride, A, T, rpb, buf0, s_tw, gph);
        return;
    }
    bool first = true;
    for (int q = 0; q < A.nn; ++q) {
        const int nv = A.n_val[q];
        if (REAL && nv < 0) continue;
        if (threadIdx.x < ng) gph[threadIdx.x] = cis_2pi_frac(nv * (int)threadIdx.x, ng);
        const cplx *Fp = Fb + ((size_t)A.n_row[q] * T.nt + t) * Md;   // row of n
        const cplx *Fm = Fb + ((size_t)A.n_rowm[q] * T.nt + t) * Md;  // row of -n
        for (int k = tl; k < M; k += tpr) {
            cplx v = cmake(0.0, 0.0);
            if (k < n && has) {
                if (REAL) {
                    v = k < L ? Fp[k] : cconj(Fm[n - k]);
                } else {
                    int m = k < L ? k : k - n;
                    v = Fp[m + L - 1];
                }
                v = cmulc(v, __ldg(&T.chirp[k]));
            }
            buf[S2W_PAD(k)] = v;
        }
        __syncthreads();
        if (MULTI)
            fft_convolve_b<true>(buf0, T, s_tw, T.bhat_p, rpb, bstride);
        else
            fft_convolve<true>(buf, T, s_tw, T.bhat_p);
        // one pass over alpha: the chirp product once, then all gamma planes with their loads issued together
        for (int a = tl; a < (has ? n : 0); a += tpr) {
            const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));
            if (REAL) {
                double *Wr = (double *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                const double cn = nv == 0 ? 1.0 : 2.0;
                const double vx = cn * v.x, vy = cn * v.y;
                for (int g0 = 0; g0 < ng; g0 += 9) {
                    double old[9];
#pragma unroll
                    for (int k = 0; k < 9; ++k)
                        old[k] = (!first && g0 + k < ng) ? Wr[(size_t)(g0 + k) * T.nt * n] : 0.0;
#pragma unroll
                    for (int k = 0; k < 9; ++k)
                        if (g0 + k < ng) {
                            const cplx ph = gph[g0 + k];
                            Wr[(size_t)(g0 + k) * T.nt * n] = old[k] + (ph.x * vx - ph.y * vy);
                        }
                }
            } else {
                cplx *Wc = (cplx *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                for (int g0 = 0; g0 < ng; g0 += 5) {
                    cplx old[5];
#pragma unroll
                    for (int k = 0; k < 5; ++k)
                        old[k] = (!first && g0 + k < ng) ? Wc[(size_t)(g0 + k) * T.nt * n] : cmake(0.0, 0.0);
#pragma unroll
                    for (int k = 0; k < 5; ++k)
                        if (g0 + k < ng) Wc[(size_t)(g0 + k) * T.nt * n] = cadd(old[k], cmul(gph[g0 + k], v));
                }
            }
        }
        first = false;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a8 synthesis: W[b][g][t][a] -> F[b][row][t][mi], F_mn = 1/(n_a n_g) sum_{a,g} W e^{-i(m alpha_a + n gamma_g)}.
// The gamma sum is done first in pixel space, V_n(a) = (1/n_g) sum_g e^{-i n gamma_g} W(g,t,a), then one DFT per row.
// Real: rows n >= 0; the row of -n follows from F_{m,-n} = conj(F_{-m,n}).
// ---------------------------------------------------------------------------------------------------------------
// Few gamma samples (real: 2N-1 <= 9, complex: 2N-1 <= 5): the gamma planes of a ring are read ONCE.  The gamma sums
// of all rows, Y_n(alpha) = 1/(2N-1) sum_g e^{-i n gamma_g} W(alpha, gamma_g), are formed together; the first row goes
// straight into the shared-memory buffer, the others are parked, chirp applied, in their own output rows (real:
// F_{., n} and F_{., -n}, 2L >= 2L-1 slots, which is why a row n = 0 goes first; complex: the row's 2L-1 slots) and
// fetched back -- each thread its own alpha samples -- when their convolution is due.
template <bool REAL, bool MULTI>
__device__ __forceinline__ void so3_fwd_few(const void *__restrict__ W, cplx *__restrict__ F, size_t sig_stride,
                                            const So3Args &A, const FftTab &T, int rpb, cplx *buf0, const cplx *s_tw,
                                            cplx *gph)
{
    constexpr int NG = REAL ? 9 : 5;
    constexpr int NR = 5;  // most rows
    const int n = T.n, L = T.L, M = T.M;
    const int bstride = fft_padded_len(M);
    const int tpr = MULTI ? blockDim.x / rpb : blockDim.x;
    const int rl = MULTI ? threadIdx.x / tpr : 0, tl = MULTI ? threadIdx.x - rl * tpr : threadIdx.x;
    cplx *buf = buf0 + (size_t)rl * bstride;
    const int t = MULTI ? blockIdx.x * rpb + rl : blockIdx.x, b = blockIdx.y;
    const bool has = MULTI ? t < T.nt : true;
    const int Md = REAL ? L : n;
    const int ng = 2 * A.N - 1;
    const size_t plane = (size_t)T.nt * n;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)b * A.nrows * T.nt * Md;
    __shared__ int s_nv[NR], s_rowp[NR], s_rowm[NR];
    int nproc = 0;
    for (int pass = 0; pass < 2; ++pass)  // a row n = 0 first
        for (int q = 0; q < A.nn; ++q) {
            const int nv = A.n_val[q];
            if ((REAL && nv < 0) || (pass == 0) != (nv == 0)) continue;
            for (int g = threadIdx.x; g < ng; g += blockDim.x) gph[nproc * ng + g] = cis_2pi_frac(-nv * g, ng);
            if (threadIdx.x == 0) {
                s_nv[nproc] = nv;
                s_rowp[nproc] = A.n_row[q];
                s_rowm[nproc] = A.n_rowm[q];
            }
            ++nproc;
        }
    __syncthreads();
    // gather pass
    for (int a = tl; a < M; a += tpr) {
        if (a >= n || !has) {
            buf[S2W_PAD(a)] = cmake(0.0, 0.0);
            continue;
        }
        const cplx ch = __ldg(&T.chirp[a]);
        double wr[NG];
        cplx wc[REAL ? 1 : NG];
        if (REAL) {
            const double *Wr = (const double *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
#pragma unroll
            for (int g = 0; g < NG; ++g) wr[g] = g < ng ? Wr[(size_t)g * plane] : 0.0;
        } else {
            const cplx *Wc = (const cplx *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
#pragma unroll
            for (int g = 0; g < NG; ++g) wc[g] = g < ng ? Wc[(size_t)g * plane] : cmake(0.0, 0.0);
        }
#pragma unroll
        for (int i = 0; i < NR; ++i)
            if (i < nproc) {
                cplx y = cmake(0.0, 0.0);
#pragma unroll
                for (int g = 0; g < NG; ++g) {
                    const cplx ph = gph[i * ng + (g < ng ? g : 0)];
                    if (REAL) {
                        y.x = fma(ph.x, wr[g], y.x);
                        y.y = fma(ph.y, wr[g], y.y);
                    } else {
                        y = cadd(y, cmul(ph, wc[g]));
                    }
                }
                y = cmul(cscale(y, inv_ng), ch);
                if (i == 0)
                    buf[S2W_PAD(a)] = y;
                else if (REAL)
                    Fb[((size_t)(a < L ? s_rowp[i] : s_rowm[i]) * T.nt + t) * Md + (a < L ? a : a - L)] = y;
                else
                    Fb[((size_t)s_rowp[i] * T.nt + t) * Md + a] = y;
            }
    }
    __syncthreads();
    for (int i = 0; i < nproc; ++i) {
        cplx *Fp = Fb + ((size_t)s_rowp[i] * T.nt + t) * Md;
        cplx *Fm = Fb + ((size_t)s_rowm[i] * T.nt + t) * Md;
        if (i > 0) {
            for (int a = tl; a < M; a += tpr) {
                cplx v = cmake(0.0, 0.0);
                if (a < n && has) v = REAL ? (a < L ? Fp[a] : Fm[a - L]) : Fp[a];
                buf[S2W_PAD(a)] = v;
            }
            __syncthreads();
        }
        if (MULTI)
            fft_convolve_b<true>(buf0, T, s_tw, T.bhat_m, rpb, bstride);
        else
            fft_convolve<true>(buf, T, s_tw, T.bhat_m);
        if (REAL) {
            const int nv = s_nv[i];
            for (int m = tl; m < (has ? L : 0); m += tpr) {
                Fp[m] = cscale(cmul(buf[S2W_PAD(m)], __ldg(&T.chirp[m])), inv_n);
                if (nv != 0) {
                    int k = m == 0 ? 0 : n - m;
                    Fm[m] = cscale(cconj(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]))), inv_n);
                }
            }
        } else {
            // the row is also this ring's parking slot of the NEXT rows' values only; its own were consumed above
            for (int mi = tl; mi < (has ? n : 0); mi += tpr) {
                int m = mi - (L - 1);
                int k = m < 0 ? m + n : m;
                Fp[mi] = cscale(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k])), inv_n);
            }
        }
        __syncthreads();
    }
}

template <bool REAL, bool MULTI>
__global__ void __launch_bounds__(256, 3) so3_fwd_kernel(const void *__restrict__ W, cplx *__restrict__ F, size_t sig_stride,
                                                     So3Args A, FftTab T, int rpb)
{
    extern __shared__ cplx buf0[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const int bstride = fft_padded_len(M);
    const int tpr = MULTI ? blockDim.x / rpb : blockDim.x;
    const int rl = MULTI ? threadIdx.x / tpr : 0, tl = MULTI ? threadIdx.x - rl * tpr : threadIdx.x;
    cplx *buf = buf0 + (size_t)rl * bstride;
    const int t = MULTI ? blockIdx.x * rpb + rl : blockIdx.x, b = blockIdx.y;
    const bool has = MULTI ? t < T.nt : true;
    const int Md = REAL ? L : n;
    const int ng = 2 * A.N - 1;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)b * A.nrows * T.nt * Md;
    __shared__ cplx gph[2 * S2W_MAX_N];
    if (ng <= (REAL ? 9 : 5)) {
        so3_fwd_few<REAL, MULTI>(W, F, sig_stride, A, T, rpb, buf0, s_tw, gph);
        return;
    }
    for (int q = 0; q < A.nn; ++q) {
        const int nv = A.n_val[q];
        if (REAL && nv < 0) continue;
        if (threadIdx.x < ng) gph[threadIdx.x] = cis_2pi_frac(-nv * (int)threadIdx.x, ng);
        __syncthreads();
        for (int a = tl; a < M; a += tpr) {
            cplx v = cmake(0.0, 0.0);
            if (a < n && has) {
                if (REAL) {
                    const double *Wr = (const double *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                    for (int g0 = 0; g0 < ng; g0 += 9) {
                        double wv[9];
#pragma unroll
                        for (int k = 0; k < 9; ++k) wv[k] = g0 + k < ng ? Wr[(size_t)(g0 + k) * T.nt * n] : 0.0;
#pragma unroll
                        for (int k = 0; k < 9; ++k)
                            if (g0 + k < ng) {
                                const cplx ph = gph[g0 + k];
                                v.x = fma(ph.x, wv[k], v.x);
                                v.y = fma(ph.y, wv[k], v.y);
                            }
                    }
                } else {
                    const cplx *Wc = (const cplx *)W + so3_base(A, b, sig_stride) + (size_t)t * n + a;
                    for (int g0 = 0; g0 < ng; g0 += 5) {
                        cplx wv[5];
#pragma unroll
                        for (int k = 0; k < 5; ++k)
                            wv[k] = g0 + k < ng ? Wc[(size_t)(g0 + k) * T.nt * n] : cmake(0.0, 0.0);
#pragma unroll
                        for (int k = 0; k < 5; ++k)
                            if (g0 + k < ng) v = cadd(v, cmul(gph[g0 + k], wv[k]));
                    }
                }
                v = cmul(cscale(v, inv_ng), __ldg(&T.chirp[a]));
            }
            buf[S2W_PAD(a)] = v;
        }
        __syncthreads();
        if (MULTI)
            fft_convolve_b<true>(buf0, T, s_tw, T.bhat_m, rpb, bstride);
        else
            fft_convolve<true>(buf, T, s_tw, T.bhat_m);
        cplx *Fp = Fb + ((size_t)A.n_row[q] * T.nt + t) * Md;
        cplx *Fm = Fb + ((size_t)A.n_rowm[q] * T.nt + t) * Md;
        if (REAL) {
            for (int m = tl; m < (has ? L : 0); m += tpr) {
                Fp[m] = cscale(cmul(buf[S2W_PAD(m)], __ldg(&T.chirp[m])), inv_n);
                if (nv != 0) {
                    int k = m == 0 ? 0 : n - m;
                    Fm[m] = cscale(cconj(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]))), inv_n);
                }
            }
        } else {
            for (int mi = tl; mi < (has ? n : 0); mi += tpr) {
                int m = mi - (L - 1);
                int k = m < 0 ? m + n : m;
                Fp[mi] = cscale(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k])), inv_n);
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a8 for REAL signals on the large grids: one block per PAIR of rings.  The row n = 0 has a Hermitian spectrum
// (F_{-m,0} = conj F_{m,0}) and a real transform, so the two rings share one complex DFT (ring t0 in the real part,
// ring t0+1 in the imaginary part), as in a1; the rows n > 0 are done ring by ring.  5 instead of 6 convolutions per
// ring pair at N = 5.
// ---------------------------------------------------------------------------------------------------------------
// Fill of one Bluestein buffer from a half-stored Hermitian row pair: buf[k] = conj(chirp[k]) x, x = Fp[k] for k < L,
// conj(Fm[n-k]) for L <= k < n, 0 for k >= n.  Four elements per thread at a time, loads first (one unconditional
// load each through a selected pointer), so that a thread waits for global memory once per four elements.
__device__ __forceinline__ void fill_row_pm(cplx *buf, const cplx *__restrict__ Fp, const cplx *__restrict__ Fm,
                                            const cplx *__restrict__ chirp, int n, int L, int M)
{
    for (int k0 = threadIdx.x; k0 < M; k0 += 4 * blockDim.x) {
        cplx x[4], c[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int k = k0 + j * blockDim.x;
            const int kk = k < n ? k : 0;
            x[j] = *(kk < L ? Fp + kk : Fm + (n - kk));
            c[j] = __ldg(&chirp[kk]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int k = k0 + j * blockDim.x;
            if (k >= M) continue;
            cplx v = k >= L ? cconj(x[j]) : x[j];
            buf[S2W_PAD(k)] = k < n ? cmulc(v, c[j]) : cmake(0.0, 0.0);
        }
    }
}

// The same for at most 9 gamma samples (N <= 5), without read-modify-write of the gamma planes: the rows are done
// ring by ring, the transforms V_n(alpha) of all rows but the last are parked in the ring's own output planes (V_0 in
// plane 0, row i in planes 2i+1, 2i+2: at most 2N-3 of the 2N-1 planes), and the pass of the last row reads them back
// -- each thread its own alpha samples, so program order is all the ordering needed -- and writes every plane once:
//   W(alpha, gamma_g) = V_0(alpha) + 2 Re sum_{n>0} e^{i n gamma_g} V_n(alpha).
__device__ __forceinline__ void so3_inv_pair_few(const cplx *__restrict__ F, double *__restrict__ W, size_t sig_stride,
                                                 const So3Args &A, const FftTab &T, cplx *buf, const cplx *s_tw,
                                                 cplx *gph)
{
    const int n = T.n, L = T.L, M = T.M;
    const int t0 = 2 * blockIdx.x, b = blockIdx.y;
    const bool has1 = t0 + 1 < L;
    const int ng = 2 * A.N - 1;
    const cplx *Fb = F + (size_t)b * A.nrows * L * L;
    double *Wb = W + so3_base(A, b, sig_stride);
    const size_t plane = (size_t)L * n;
    int q0 = -1, np = 0;  // the row n = 0 and the number of rows n > 0
    for (int q = 0; q < A.nn; ++q) {
        if (A.n_val[q] == 0) q0 = q;
        if (A.n_val[q] > 0) {
            for (int g = threadIdx.x; g < ng; g += blockDim.x) gph[np * ng + g] = cis_2pi_frac(A.n_val[q] * g, ng);
            ++np;
        }
    }
    if (q0 >= 0) {
        const cplx *X0 = Fb + ((size_t)A.n_row[q0] * L + t0) * L, *X1 = has1 ? X0 + L : X0;
        for (int k0 = threadIdx.x; k0 < M; k0 += 4 * blockDim.x) {  // four elements at a time, loads first
            cplx xa[4], xc[4], ch[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = k0 + j * blockDim.x;
                const int kk = k < n ? k : 0, m = kk < L ? kk : n - kk;
                xa[j] = X0[m];
                xc[j] = X1[m];
                ch[j] = __ldg(&T.chirp[kk]);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = k0 + j * blockDim.x;
                if (k >= M) continue;
                cplx a = xa[j], c = has1 ? xc[j] : cmake(0.0, 0.0);
                if (k >= L) {
                    a = cconj(a);
                    c = cconj(c);
                }
                buf[S2W_PAD(k)] = k < n ? cmulc(cmake(a.x - c.y, a.y + c.x), ch[j]) : cmake(0.0, 0.0);
            }
        }
        __syncthreads();
        fft_convolve<true>(buf, T, s_tw, T.bhat_p);
        for (int a = threadIdx.x; a < n; a += blockDim.x) {
            const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));  // V_0 of ring t0 + i V_0 of ring t0+1
            double *Wr = Wb + (size_t)t0 * n + a;
            for (int g = 0; g < (np ? 1 : ng); ++g) {
                Wr[g * plane] = v.x;
                if (has1) Wr[g * plane + n] = v.y;
            }
        }
        __syncthreads();
    }
    for (int r = 0; r < (has1 ? 2 : 1); ++r) {
        const int t = t0 + r;
        int i = 0;
        for (int q = 0; q < A.nn; ++q) {
            if (A.n_val[q] <= 0) continue;
            const cplx *Fp = Fb + ((size_t)A.n_row[q] * L + t) * L;
            const cplx *Fm = Fb + ((size_t)A.n_rowm[q] * L + t) * L;
            fill_row_pm(buf, Fp, Fm, T.chirp, n, L, M);
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_p);
            if (i + 1 < np) {
                for (int a = threadIdx.x; a < n; a += blockDim.x) {
                    const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));
                    double *Wr = Wb + (size_t)t * n + a;
                    Wr[(2 * i + 1) * plane] = v.x;
                    Wr[(2 * i + 2) * plane] = v.y;
                }
            } else {
                for (int a = threadIdx.x; a < n; a += blockDim.x) {
                    const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));
                    double *Wr = Wb + (size_t)t * n + a;
                    double sc[7];
#pragma unroll
                    for (int s = 0; s < 7; ++s) sc[s] = 0.0;
                    if (q0 >= 0) sc[0] = Wr[0];
#pragma unroll
                    for (int s = 1; s < 7; ++s)
                        if (s < 2 * np - 1) sc[s] = Wr[s * plane];
                    double out[9];
#pragma unroll
                    for (int g = 0; g < 9; ++g) {
                        const cplx ph = gph[(np - 1) * ng + (g < ng ? g : 0)];
                        out[g] = fma(2.0, ph.x * v.x - ph.y * v.y, sc[0]);
                    }
#pragma unroll
                    for (int j = 0; j < 3; ++j)
                        if (j + 1 < np) {
#pragma unroll
                            for (int g = 0; g < 9; ++g) {
                                const cplx ph = gph[j * ng + (g < ng ? g : 0)];
                                out[g] = fma(2.0, ph.x * sc[2 * j + 1] - ph.y * sc[2 * j + 2], out[g]);
                            }
                        }
#pragma unroll
                    for (int g = 0; g < 9; ++g)
                        if (g < ng) Wr[g * plane] = out[g];
                }
            }
            __syncthreads();
            ++i;
        }
    }
}

__global__ void __launch_bounds__(256, 3) so3_inv_pair_kernel(const cplx *__restrict__ F, double *__restrict__ W,
                                                             size_t sig_stride, So3Args A, FftTab Tin)
{
    // dynamic shared memory: the Bluestein buffer, the twiddles (own split, tw_own_entries), and for 2N-1 > 9 the gamma
    // phases; static shared memory stays small enough for three blocks per SM at M = 4096 (so3_launch)
    extern __shared__ cplx buf[];
    FftTab T = Tin;
    cplx *s_tw = buf + fft_padded_len(T.M);
    __shared__ cplx s_gph[36];
    cplx *gph = 2 * A.N - 1 <= 9 ? s_gph : s_tw + tw_own_entries(T.logM);
    tw_stage_own(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const int t0 = 2 * blockIdx.x, b = blockIdx.y;
    const bool has1 = t0 + 1 < L;
    const int ng = 2 * A.N - 1;
    const cplx *Fb = F + (size_t)b * A.nrows * L * L;
    double *Wb = W + so3_base(A, b, sig_stride);
    const size_t plane = (size_t)L * n;
    if (ng <= 9) {
        so3_inv_pair_few(F, W, sig_stride, A, T, buf, s_tw, gph);
        return;
    }
    bool first = true;
    for (int q = 0; q < A.nn; ++q) {
        const int nv = A.n_val[q];
        if (nv < 0) continue;
        if (nv == 0) {
            const cplx *X0 = Fb + ((size_t)A.n_row[q] * L + t0) * L, *X1 = X0 + L;
            for (int k = threadIdx.x; k < M; k += blockDim.x) {
                cplx v = cmake(0.0, 0.0);
                if (k < n) {
                    const int m = k < L ? k : n - k;
                    cplx a = X0[m], c = has1 ? X1[m] : cmake(0.0, 0.0);
                    if (k >= L) {
                        a = cconj(a);
                        c = cconj(c);
                    }
                    v = cmulc(cmake(a.x - c.y, a.y + c.x), __ldg(&T.chirp[k]));
                }
                buf[S2W_PAD(k)] = v;
            }
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_p);
            for (int a = threadIdx.x; a < n; a += blockDim.x) {
                const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));  // V_0 of ring t0 + i V_0 of ring t0+1
                double *Wr = Wb + (size_t)t0 * n + a;
                for (int g = 0; g < ng; ++g) {
                    Wr[g * plane] = first ? v.x : Wr[g * plane] + v.x;
                    if (has1) Wr[g * plane + n] = first ? v.y : Wr[g * plane + n] + v.y;
                }
            }
            first = false;
            __syncthreads();
            continue;
        }
        if (threadIdx.x < ng) gph[threadIdx.x] = cis_2pi_frac(nv * (int)threadIdx.x, ng);
        for (int r = 0; r < (has1 ? 2 : 1); ++r) {
            const int t = t0 + r;
            const cplx *Fp = Fb + ((size_t)A.n_row[q] * L + t) * L;
            const cplx *Fm = Fb + ((size_t)A.n_rowm[q] * L + t) * L;
            for (int k = threadIdx.x; k < M; k += blockDim.x) {
                cplx v = cmake(0.0, 0.0);
                if (k < n) v = cmulc(k < L ? Fp[k] : cconj(Fm[n - k]), __ldg(&T.chirp[k]));
                buf[S2W_PAD(k)] = v;
            }
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_p);
            for (int a = threadIdx.x; a < n; a += blockDim.x) {
                const cplx v = cmulc(buf[S2W_PAD(a)], __ldg(&T.chirp[a]));
                double *Wr = Wb + (size_t)t * n + a;
                const double vx = 2.0 * v.x, vy = 2.0 * v.y;
                for (int g0 = 0; g0 < ng; g0 += 9) {
                    double old[9];
#pragma unroll
                    for (int k = 0; k < 9; ++k) old[k] = (!first && g0 + k < ng) ? Wr[(g0 + k) * plane] : 0.0;
#pragma unroll
                    for (int k = 0; k < 9; ++k)
                        if (g0 + k < ng) {
                            const cplx ph = gph[g0 + k];
                            Wr[(g0 + k) * plane] = old[k] + (ph.x * vx - ph.y * vy);
                        }
                }
            }
            __syncthreads();
        }
        first = false;
    }
}

// The analysis counterpart for at most 9 gamma samples: the gamma planes of a ring are read ONCE; the gamma sums of
// all its rows, Y_n(alpha) = 1/(2N-1) sum_g e^{-i n gamma_g} W(alpha, gamma_g), are formed together, the row n = 0
// goes straight into the shared-memory buffer (ring t0 real part, ring t0+1 imaginary part) and the rows n > 0 are
// parked, chirp applied, in the ring's own output rows F_{., n}, F_{., -n} (2L >= 2L-1 entries), from where the fill
// of that row's convolution takes them back -- each thread its own alpha samples -- before the row is overwritten.
__device__ __forceinline__ void so3_fwd_pair_few(const double *__restrict__ W, cplx *__restrict__ F, size_t sig_stride,
                                                 const So3Args &A, const FftTab &T, cplx *buf, const cplx *s_tw,
                                                 cplx *gph)
{
    const int n = T.n, L = T.L, M = T.M;
    const int t0 = 2 * blockIdx.x, b = blockIdx.y;
    const bool has1 = t0 + 1 < L;
    const int ng = 2 * A.N - 1;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)b * A.nrows * L * L;
    const double *Wb = W + so3_base(A, b, sig_stride);
    const size_t plane = (size_t)L * n;
    __shared__ int s_rowp[4], s_rowm[4];
    int q0 = -1, np = 0;
    for (int q = 0; q < A.nn; ++q) {
        if (A.n_val[q] == 0) q0 = q;
        if (A.n_val[q] > 0) {
            for (int g = threadIdx.x; g < ng; g += blockDim.x) gph[np * ng + g] = cis_2pi_frac(-A.n_val[q] * g, ng);
            if (threadIdx.x == 0) {
                s_rowp[np] = A.n_row[q];
                s_rowm[np] = A.n_rowm[q];
            }
            ++np;
        }
    }
    __syncthreads();
    // gather pass: every gamma plane of both rings once, the 2 x 9 loads of an alpha sample issued together
    const double *W0 = Wb + (size_t)t0 * n, *W1 = Wb + (size_t)(has1 ? t0 + 1 : t0) * n;
    for (int a = threadIdx.x; a < M; a += blockDim.x) {
        if (a >= n) {
            buf[S2W_PAD(a)] = cmake(0.0, 0.0);
            continue;
        }
        const cplx ch = __ldg(&T.chirp[a]);
        double wv[2][9];
#pragma unroll
        for (int g = 0; g < 9; ++g) {
            const size_t o = a + (size_t)(g < ng ? g : 0) * plane;
            wv[0][g] = W0[o];
            wv[1][g] = W1[o];
        }
#pragma unroll
        for (int g = 0; g < 9; ++g) {
            if (g >= ng) wv[0][g] = 0.0;
            if (g >= ng || !has1) wv[1][g] = 0.0;
        }
        double y0 = 0.0, y1 = 0.0;
#pragma unroll
        for (int g = 0; g < 9; ++g) {
            y0 += wv[0][g];
            y1 += wv[1][g];
        }
        buf[S2W_PAD(a)] = cmul(cscale(cmake(y0, y1), inv_ng), ch);
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            if (r == 1 && !has1) continue;
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (i < np) {
                    cplx y = cmake(0.0, 0.0);
#pragma unroll
                    for (int g = 0; g < 9; ++g) {
                        const cplx ph = gph[i * ng + (g < ng ? g : 0)];
                        y.x = fma(ph.x, wv[r][g], y.x);
                        y.y = fma(ph.y, wv[r][g], y.y);
                    }
                    y = cmul(cscale(y, inv_ng), ch);
                    cplx *dst = a < L ? Fb + ((size_t)s_rowp[i] * L + t0 + r) * L + a
                                      : Fb + ((size_t)s_rowm[i] * L + t0 + r) * L + (a - L);
                    *dst = y;
                }
        }
    }
    __syncthreads();
    if (q0 >= 0) {
        fft_convolve<true>(buf, T, s_tw, T.bhat_m);
        for (int k = threadIdx.x; k < n; k += blockDim.x) buf[S2W_PAD(k)] = cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]));
        __syncthreads();
        cplx *F0 = Fb + ((size_t)A.n_row[q0] * L + t0) * L, *F1 = F0 + L;
        for (int m = threadIdx.x; m < L; m += blockDim.x) {
            const cplx a = buf[S2W_PAD(m)], c = cconj(buf[S2W_PAD(m == 0 ? 0 : n - m)]);
            const cplx sm = cadd(a, c), df = csub(a, c);
            F0[m] = cscale(sm, 0.5 * inv_n);
            if (has1) F1[m] = cmake(0.5 * inv_n * df.y, -0.5 * inv_n * df.x);
        }
        __syncthreads();
    }
    for (int r = 0; r < (has1 ? 2 : 1); ++r) {
        const int t = t0 + r;
        for (int i = 0; i < np; ++i) {
            cplx *Fp = Fb + ((size_t)s_rowp[i] * L + t) * L;
            cplx *Fm = Fb + ((size_t)s_rowm[i] * L + t) * L;
            for (int a0 = threadIdx.x; a0 < M; a0 += 4 * blockDim.x) {  // four at a time, loads first
                cplx x[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int a = a0 + j * blockDim.x;
                    const int aa = a < n ? a : 0;
                    x[j] = *(aa < L ? Fp + aa : Fm + (aa - L));
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int a = a0 + j * blockDim.x;
                    if (a < M) buf[S2W_PAD(a)] = a < n ? x[j] : cmake(0.0, 0.0);
                }
            }
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_m);
            for (int m = threadIdx.x; m < L; m += blockDim.x) {
                Fp[m] = cscale(cmul(buf[S2W_PAD(m)], __ldg(&T.chirp[m])), inv_n);
                const int k = m == 0 ? 0 : n - m;
                Fm[m] = cscale(cconj(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]))), inv_n);
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(256, 3) so3_fwd_pair_kernel(const double *__restrict__ W, cplx *__restrict__ F,
                                                             size_t sig_stride, So3Args A, FftTab Tin)
{
    // dynamic shared memory: the Bluestein buffer, the twiddles (own split, tw_own_entries), and for 2N-1 > 9 the gamma
    // phases; static shared memory stays small enough for three blocks per SM at M = 4096 (so3_launch)
    extern __shared__ cplx buf[];
    FftTab T = Tin;
    cplx *s_tw = buf + fft_padded_len(T.M);
    __shared__ cplx s_gph[36];
    cplx *gph = 2 * A.N - 1 <= 9 ? s_gph : s_tw + tw_own_entries(T.logM);
    tw_stage_own(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const int t0 = 2 * blockIdx.x, b = blockIdx.y;
    const bool has1 = t0 + 1 < L;
    const int ng = 2 * A.N - 1;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)b * A.nrows * L * L;
    const double *Wb = W + so3_base(A, b, sig_stride);
    const size_t plane = (size_t)L * n;
    if (ng <= 9) {
        so3_fwd_pair_few(W, F, sig_stride, A, T, buf, s_tw, gph);
        return;
    }
    for (int q = 0; q < A.nn; ++q) {
        const int nv = A.n_val[q];
        if (nv < 0) continue;
        if (nv == 0) {
            for (int a = threadIdx.x; a < M; a += blockDim.x) {
                cplx v = cmake(0.0, 0.0);
                if (a < n) {
                    const double *Wr = Wb + (size_t)t0 * n + a;
                    for (int g0 = 0; g0 < ng; g0 += 9) {
                        double w0[9], w1[9];
#pragma unroll
                        for (int k = 0; k < 9; ++k) {
                            w0[k] = g0 + k < ng ? Wr[(g0 + k) * plane] : 0.0;
                            w1[k] = (has1 && g0 + k < ng) ? Wr[(g0 + k) * plane + n] : 0.0;
                        }
#pragma unroll
                        for (int k = 0; k < 9; ++k) {
                            v.x += w0[k];
                            v.y += w1[k];
                        }
                    }
                    v = cmul(cscale(v, inv_ng), __ldg(&T.chirp[a]));
                }
                buf[S2W_PAD(a)] = v;
            }
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_m);
            for (int k = threadIdx.x; k < n; k += blockDim.x) buf[S2W_PAD(k)] = cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]));
            __syncthreads();
            cplx *F0 = Fb + ((size_t)A.n_row[q] * L + t0) * L, *F1 = F0 + L;
            for (int m = threadIdx.x; m < L; m += blockDim.x) {
                const cplx a = buf[S2W_PAD(m)], c = cconj(buf[S2W_PAD(m == 0 ? 0 : n - m)]);
                const cplx sm = cadd(a, c), df = csub(a, c);
                F0[m] = cscale(sm, 0.5 * inv_n);
                if (has1) F1[m] = cmake(0.5 * inv_n * df.y, -0.5 * inv_n * df.x);
            }
            __syncthreads();
            continue;
        }
        if (threadIdx.x < ng) gph[threadIdx.x] = cis_2pi_frac(-nv * (int)threadIdx.x, ng);
        __syncthreads();
        for (int r = 0; r < (has1 ? 2 : 1); ++r) {
            const int t = t0 + r;
            for (int a = threadIdx.x; a < M; a += blockDim.x) {
                cplx v = cmake(0.0, 0.0);
                if (a < n) {
                    const double *Wr = Wb + (size_t)t * n + a;
                    for (int g0 = 0; g0 < ng; g0 += 9) {
                        double wv[9];
#pragma unroll
                        for (int k = 0; k < 9; ++k) wv[k] = g0 + k < ng ? Wr[(g0 + k) * plane] : 0.0;
#pragma unroll
                        for (int k = 0; k < 9; ++k)
                            if (g0 + k < ng) {
                                const cplx ph = gph[g0 + k];
                                v.x = fma(ph.x, wv[k], v.x);
                                v.y = fma(ph.y, wv[k], v.y);
                            }
                    }
                    v = cmul(cscale(v, inv_ng), __ldg(&T.chirp[a]));
                }
                buf[S2W_PAD(a)] = v;
            }
            __syncthreads();
            fft_convolve<true>(buf, T, s_tw, T.bhat_m);
            cplx *Fp = Fb + ((size_t)A.n_row[q] * L + t) * L;
            cplx *Fm = Fb + ((size_t)A.n_rowm[q] * L + t) * L;
            for (int m = threadIdx.x; m < L; m += blockDim.x) {
                Fp[m] = cscale(cmul(buf[S2W_PAD(m)], __ldg(&T.chirp[m])), inv_n);
                const int k = m == 0 ? 0 : n - m;
                Fm[m] = cscale(cconj(cmul(buf[S2W_PAD(k)], __ldg(&T.chirp[k]))), inv_n);
            }
            __syncthreads();
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a2 reweighting of one theta-column F[.][t][mi] (stride Md) of parity sigma = (-1)^{m+n}, in place (R3):
//   (ii)  extend to n = 2L-1 rings by F(theta_{n-1-t}) = sigma F(theta_t)
//   (iii) Fh(k) = 1/n sum_t F(theta_t) e^{-i k theta_t},  theta_t = pi(2t+1)/n,  |k| <= L-1
//   (iv)  G(k') = sum_k Fh(k) w(k + k')
//   (v)   g(theta_t) = sum_k' G(k') e^{-i k' theta_t}
//   (vi)  h(theta_t) = g(theta_t) + sigma g(theta_{n-1-t}),  t < L-1;   h(theta_{L-1}) = g(theta_{L-1})
// Three chained chirp convolutions with no reordering in between: (iii) is evaluated at k = L-1-i, i = 0..n-1, as a
// sign(+) DFT of the modulated column, which makes (iv) a plain convolution xr * w landing at slot i' = k' + L-1, and
// (v) a sign(-) DFT over i' with an output modulation; the four phase tables rw_* absorb chirps and modulations.
// One block per column.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) reweight_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A, FftTab T)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, L = T.L, M = T.M;
    const int mi = blockIdx.x, q = blockIdx.y, b = blockIdx.z;
    const int m = A.isReal ? mi : mi - (L - 1);
    const int nv = A.n_val[q];
    const double sigma = ((m + nv) & 1) ? -1.0 : 1.0;
    const cplx *col = F + ((size_t)b * A.nrows + A.n_row[q]) * (size_t)L * A.Md + mi;
    cplx *colT = Ft + (((size_t)b * A.nrows + A.n_row[q]) * A.Md + mi) * (size_t)L;  // [b][row][mi][t]: t contiguous
    for (int t = threadIdx.x; t < M; t += blockDim.x) {
        cplx v = cmake(0.0, 0.0);
        if (t < n) {
            v = t < L ? col[(size_t)t * A.Md] : cscale(col[(size_t)(n - 1 - t) * A.Md], sigma);
            v = cmul(v, __ldg(&T.rw_in1[t]));
        }
        buf[S2W_PAD(t)] = v;
    }
    __syncthreads();
    fft_convolve(buf, T, s_tw, T.bhat_p);
    for (int i = threadIdx.x; i < M; i += blockDim.x)
        buf[S2W_PAD(i)] = i < n ? cmul(buf[S2W_PAD(i)], __ldg(&T.rw_out1[i])) : cmake(0.0, 0.0);
    __syncthreads();
    fft_convolve(buf, T, s_tw, T.what);
    for (int i = threadIdx.x; i < M; i += blockDim.x)
        buf[S2W_PAD(i)] = i < n ? cmul(buf[S2W_PAD(i)], __ldg(&T.rw_in3[i])) : cmake(0.0, 0.0);
    __syncthreads();
    fft_convolve(buf, T, s_tw, T.bhat_m);
    for (int t = threadIdx.x; t < L; t += blockDim.x) {
        cplx g0 = cmul(buf[S2W_PAD(t)], __ldg(&T.rw_out3[t]));
        if (t < L - 1) {
            int tb = n - 1 - t;
            cplx g1 = cmul(buf[S2W_PAD(tb)], __ldg(&T.rw_out3[tb]));
            g0 = cmake(fma(sigma, g1.x, g0.x), fma(sigma, g1.y, g0.y));
        }
        colT[t] = g0;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a2 in Toeplitz/Hankel form.  On the extended grid of n = 2L-1 rings the operator of R3 (iii)-(v),
//   K[t,s] = sum_{k,k'} w(k+k') e^{-i(k theta_s + k' theta_t)} = int_0^pi D_n(theta-theta_t) D_n(theta-theta_s) sin(theta) dtheta
// (D_n the Dirichlet kernel), is Cauchy-like:  K[t,s] = (-1)^{t-s} (c_t - c_s) / sin(pi (t-s)/n),  t != s.
// Folding the extension and the fold (vi) into it, with a_t = (-1)^t, delta_t = c_t - c_{n-1-t}, on rings t, s < L-1:
//   n h_t = a_t [ delta_t ((T - sigma H) u1)_t - ((T + sigma H) u2)_t ] + (K_tt + K_{n-1-t,n-1-t}) x_t + v_sigma[t] x_{L-1},
//   u1 = a x,  u2 = delta a x,  T[t,s] = 1/sin(pi (t-s)/n) (0 on the diagonal),  H[t,s] = 1/sin(pi (t+s+1)/n),
// and the pole ring t = L-1 (its own mirror image) is a plain dot product with a tabulated row.  T u and H u are
// linear convolutions of length-(L-1) sequences: four power-of-two FFTs of length M2 >= 2L-3 per column (H u uses
// the spectrum of u at -k), instead of three Bluestein convolutions (six FFTs of length 2 M2).  All tables (c_t, the
// diagonal, pole row and column) are computed in long double at plan creation; no chirps, so the result is also more
// accurate (2e-16 at L = 1024).  One block per column; both sequences go through each FFT pass together.
// ---------------------------------------------------------------------------------------------------------------
#define RW_MAXPT 8  // ring values a thread keeps in registers (L <= 8 * blockDim)
template <int PT>  // ring values a thread keeps in registers: L <= PT * blockDim
__global__ void __launch_bounds__(256, 3) reweight_th_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A,
                                                            RwTab R)
{
    extern __shared__ cplx buf[];
    // twiddles: a two-level split of W_M^k on the transform's own length (k = 32 hi + lo, M / 32 + 32 entries) instead
    // of the plan-wide table's split (up to 192 entries): the 1.5 KB are what lets a third block fit on an SM at L = 1024
    constexpr int TWN = 64 * (PT / 4) + 32;
    __shared__ cplx s_tw[TWN];
    __shared__ cplx s_part[8];
    __shared__ cplx s_pole[2];
    FftTab T = R.fft;
    {
        const int nh = T.M >> 5;
        for (int i = threadIdx.x; i < nh; i += blockDim.x) s_tw[i] = R.fft.tw[(i << 5) * R.fft.twmul];
        // (M < 32: only the first M entries exist -- reading on ran past the end of the plan's twiddle table, a fault that
        // showed or not with the neighbouring allocations; entry 0 = 1 then also serves as the single "high" entry)
        if (threadIdx.x < 32 && (int)threadIdx.x < T.M) s_tw[nh + threadIdx.x] = R.fft.tw[threadIdx.x * R.fft.twmul];
        T.twmul = 1;
        T.twmask = T.M - 1;
        T.twlo = 5;
    }
    const int L = R.L, Lm = L - 1, M = T.M;
    const int bstride = fft_padded_len(M);
    cplx *b1 = buf, *b2 = buf + bstride;
    const int mi = blockIdx.x, q = blockIdx.y, b = blockIdx.z;
    const int m = A.isReal ? mi : mi - (L - 1);
    const int nv = A.n_val[q];
    const int par = ((m + nv) & 1) ? 1 : 0;  // 0: sigma = +1, 1: sigma = -1
    // M = 512 PT (always, see launch_reweight_th): the outermost radix-8 pass of both transforms has stride
    // M / 8 = NI * 256, so its butterflies touch exactly the rings t = threadIdx.x + 256 j this thread holds in xs[]
    // (inputs 4..7 are the zero padding) -- the first forward pass runs straight from the registers, the last inverse
    // pass feeds the epilogue from them: no zero fill, and 2 writes + 2 reads of the buffers less per column
    constexpr int NI = PT / 4;
    const bool fused = M == 512 * PT && blockDim.x == 256;
    const double sigma = par ? -1.0 : 1.0;
    const cplx *col = F + ((size_t)b * A.nrows + A.n_row[q]) * (size_t)L * A.Md + mi;
    cplx *colT = Ft + (((size_t)b * A.nrows + A.n_row[q]) * A.Md + mi) * (size_t)L;  // [b][row][mi][t]: t contiguous
    const double *rp = R.rpole + par * L, *vp = R.vpole + par * L;

    cplx xs[PT];
    cplx dot = cmake(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < PT; ++k) {
        const int t = threadIdx.x + k * blockDim.x;
        cplx x = cmake(0.0, 0.0);
        if (t < L) {
            x = col[(size_t)t * A.Md];
            const double r = rp[t];
            dot.x = fma(r, x.x, dot.x);
            dot.y = fma(r, x.y, dot.y);
        }
        xs[k] = x;
        if (t == Lm) s_pole[0] = x;
    }
    if (!fused) {
        for (int t = threadIdx.x; t < M; t += blockDim.x) {  // zero padding (and the slots filled below)
            b1[S2W_PAD(t)] = cmake(0.0, 0.0);
            b2[S2W_PAD(t)] = cmake(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < PT; ++k) {
            const int t = threadIdx.x + k * blockDim.x;
            if (t < Lm) {
                const cplx u1 = (t & 1) ? cscale(xs[k], -1.0) : xs[k];
                b1[S2W_PAD(t)] = u1;
                b2[S2W_PAD(t)] = cscale(u1, R.delta[t]);
            }
        }
    }
    // pole-ring dot product: warp shuffle, then across warps
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
        dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
    }
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = dot;
    __syncthreads();
    if (fused) {
        const int per = M >> 3;
#pragma unroll
        for (int c = 0; c < NI; ++c) {
            const int idx = threadIdx.x + c * 256;
            cplx w[8];
            twiddle_powers<8>(tw_lookup(s_tw, T, idx), w);
#pragma unroll
            for (int sq = 0; sq < 2; ++sq) {
                cplx v[8];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int t = idx + k * per;  // = threadIdx.x + 256 (c + k NI)
                    cplx u = cmake(0.0, 0.0);
                    if (t < Lm) {
                        u = (t & 1) ? cscale(xs[c + k * NI], -1.0) : xs[c + k * NI];
                        if (sq) u = cscale(u, R.delta[t]);
                    }
                    v[k] = u;
                }
#pragma unroll
                for (int k = 4; k < 8; ++k) v[k] = cmake(0.0, 0.0);
                Bfly<8, false>::run(v);
#pragma unroll
                for (int j = 1; j < 8; ++j) v[j] = cmul(v[j], w[j]);
                cplx *bq = buf + sq * bstride;
#pragma unroll
                for (int k = 0; k < 8; ++k) bq[S2W_PAD(idx + k * per)] = v[k];
            }
        }
        __syncthreads();
        for (int logS = T.logM - 3; logS >= 3; logS -= 3) {
            dif_pass_b<8>(buf, M, logS, T, s_tw, 2, bstride);
            __syncthreads();
        }
        if (T.logM % 3 == 2) {
            dif_pass_b<4>(buf, M, 2, T, s_tw, 2, bstride);
            __syncthreads();
        } else if (T.logM % 3 == 1) {
            dif_pass_b<2>(buf, M, 1, T, s_tw, 2, bstride);
            __syncthreads();
        }
    } else {
        fft_dif_full_b(buf, T, s_tw, 2, bstride);
    }
    // spectra of T u -/+ sigma H u: Y(k) = That(k) U(k) -/+ sigma Ghat(k) U(-k)
    for (int i = threadIdx.x; i < R.npairs; i += blockDim.x) {
        const int2 pp = __ldg(&R.pairs[i]);
        const int p = pp.x, pn = pp.y;
        const cplx tp = __ldg(&R.TG[4 * i]), gp = cscale(__ldg(&R.TG[4 * i + 1]), sigma);
        const cplx tn = __ldg(&R.TG[4 * i + 2]), gn = cscale(__ldg(&R.TG[4 * i + 3]), sigma);
        const cplx u1p = b1[S2W_PAD(p)], u1n = b1[S2W_PAD(pn)], u2p = b2[S2W_PAD(p)], u2n = b2[S2W_PAD(pn)];
        b1[S2W_PAD(p)] = csub(cmul(tp, u1p), cmul(gp, u1n));
        b2[S2W_PAD(p)] = cadd(cmul(tp, u2p), cmul(gp, u2n));
        if (pn != p) {
            b1[S2W_PAD(pn)] = csub(cmul(tn, u1n), cmul(gn, u1p));
            b2[S2W_PAD(pn)] = cadd(cmul(tn, u2n), cmul(gn, u2p));
        }
    }
    __syncthreads();
    const cplx xpole = s_pole[0];
    if (fused) {
        if (T.logM % 3 == 2) {
            dit_pass_b<4>(buf, M, 2, T, s_tw, 2, bstride);
            __syncthreads();
        } else if (T.logM % 3 == 1) {
            dit_pass_b<2>(buf, M, 1, T, s_tw, 2, bstride);
            __syncthreads();
        }
        for (int logS = T.logM % 3 + 3; logS < T.logM; logS += 3) {
            dit_pass_b<8>(buf, M, logS, T, s_tw, 2, bstride);
            __syncthreads();
        }
        const int per = M >> 3;
#pragma unroll
        for (int c = 0; c < NI; ++c) {
            const int idx = threadIdx.x + c * 256;
            cplx w[8];
            twiddle_powers<8>(tw_lookup(s_tw, T, idx), w);
            cplx y1[4];
            {
                cplx v[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = b1[S2W_PAD(idx + k * per)];
#pragma unroll
                for (int j = 1; j < 8; ++j) v[j] = cmulc(v[j], w[j]);
                Bfly<8, true>::run(v);
#pragma unroll
                for (int k = 0; k < 4; ++k) y1[k] = v[k];
            }
            cplx v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = b2[S2W_PAD(idx + k * per)];
#pragma unroll
            for (int j = 1; j < 8; ++j) v[j] = cmulc(v[j], w[j]);
            Bfly<8, true>::run(v);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int t = idx + k * per;
                const cplx x = xs[c + k * NI];
                if (t < Lm) {
                    const double dl = R.delta[t], ds = R.dsum[t], vv = vp[t];
                    cplx h = cmake(fma(dl, y1[k].x, -v[k].x), fma(dl, y1[k].y, -v[k].y));
                    if (t & 1) h = cscale(h, -1.0);
                    h.x += fma(ds, x.x, vv * xpole.x);
                    h.y += fma(ds, x.y, vv * xpole.y);
                    colT[t] = h;
                } else if (t == Lm) {
                    cplx acc = cmake(0.0, 0.0);
                    for (int wi = 0; wi < (int)(blockDim.x >> 5); ++wi) acc = cadd(acc, s_part[wi]);
                    colT[t] = acc;
                }
            }
        }
        return;
    }
    fft_dit_full_b(buf, T, s_tw, 2, bstride);
#pragma unroll
    for (int k = 0; k < PT; ++k) {
        const int t = threadIdx.x + k * blockDim.x;
        if (t < Lm) {
            const cplx y1 = b1[S2W_PAD(t)], y2 = b2[S2W_PAD(t)];
            const double dl = R.delta[t], ds = R.dsum[t], v = vp[t];
            cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
            if (t & 1) h = cscale(h, -1.0);
            h.x += fma(ds, xs[k].x, v * xpole.x);
            h.y += fma(ds, xs[k].y, v * xpole.y);
            colT[t] = h;
        } else if (t == Lm) {
            cplx acc = cmake(0.0, 0.0);
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) acc = cadd(acc, s_part[w]);
            colT[t] = acc;
        }
    }
}

// The same for the small grids of the multiresolution / ball scale loops (M2 <= 1024): cpb = 2048 / M2 columns per block,
// tpc = 256 / cpb threads per column, all 2 cpb sequences through each FFT pass together -- one column per block would
// spend its time in per-block set-up and barriers there.
#define RW_MAXCPB 128
__global__ void __launch_bounds__(256, 2) reweight_th_multi_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft,
                                                                  RwArgs A, RwTab R, int cpb, int ncolumns)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, R.fft);
    __shared__ double s_dot[RW_MAXCPB][2];
    __shared__ cplx s_pole[RW_MAXCPB];
    const FftTab &T = R.fft;
    const int L = R.L, Lm = L - 1, M = T.M;
    const int bstride = fft_padded_len(M);
    const int tpc = blockDim.x / cpb, cl = threadIdx.x / tpc, tl = threadIdx.x - cl * tpc;
    cplx *b1 = buf + (size_t)(2 * cl) * bstride, *b2 = b1 + bstride;
    const int colid = blockIdx.x * cpb + cl;
    const bool has = colid < ncolumns;
    const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
    const int m = A.isReal ? mi : mi - (L - 1);
    const int nv = has ? A.n_val[q] : 0;
    const int par = ((m + nv) & 1) ? 1 : 0;
    const double sigma = par ? -1.0 : 1.0;
    const int row = has ? A.n_row[q] : 0;
    const cplx *col = F + ((size_t)b * A.nrows + row) * (size_t)L * A.Md + mi;
    cplx *colT = Ft + (((size_t)b * A.nrows + row) * A.Md + mi) * (size_t)L;
    const double *rp = R.rpole + par * L, *vp = R.vpole + par * L;

    if (threadIdx.x < cpb) s_dot[threadIdx.x][0] = s_dot[threadIdx.x][1] = 0.0;
    cplx xs[RW_MAXPT];
    cplx dot = cmake(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < RW_MAXPT; ++k) {
        const int t = tl + k * tpc;
        cplx x = cmake(0.0, 0.0);
        if (t < L && has) {
            x = col[(size_t)t * A.Md];
            const double r = rp[t];
            dot.x = fma(r, x.x, dot.x);
            dot.y = fma(r, x.y, dot.y);
            if (t == Lm) s_pole[cl] = x;
        }
        xs[k] = x;
    }
    for (int t = tl; t < M; t += tpc) {
        b1[S2W_PAD(t)] = cmake(0.0, 0.0);
        b2[S2W_PAD(t)] = cmake(0.0, 0.0);
    }
    __syncthreads();  // zeroed buffers and s_dot are visible
#pragma unroll
    for (int k = 0; k < RW_MAXPT; ++k) {
        const int t = tl + k * tpc;
        if (t < Lm) {
            const cplx u1 = (t & 1) ? cscale(xs[k], -1.0) : xs[k];
            b1[S2W_PAD(t)] = u1;
            b2[S2W_PAD(t)] = cscale(u1, R.delta[t]);
        }
    }
    {   // pole-ring dot product: shuffle tree over the lanes of a column inside a warp, then shared atomics
        const int w = tpc < 32 ? tpc : 32;  // a power of two; columns never straddle a w-lane group
        for (int o = w >> 1; o > 0; o >>= 1) {
            dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
            dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
        }
        if ((threadIdx.x & (w - 1)) == 0) {
            atomicAdd(&s_dot[cl][0], dot.x);
            atomicAdd(&s_dot[cl][1], dot.y);
        }
    }
    __syncthreads();
    fft_dif_full_b(buf, T, s_tw, 2 * cpb, bstride);
    for (int i = tl; i < R.npairs; i += tpc) {
        const int2 pp = __ldg(&R.pairs[i]);
        const int p = pp.x, pn = pp.y;
        const cplx tp = __ldg(&R.TG[4 * i]), gp = cscale(__ldg(&R.TG[4 * i + 1]), sigma);
        const cplx tn = __ldg(&R.TG[4 * i + 2]), gn = cscale(__ldg(&R.TG[4 * i + 3]), sigma);
        const cplx u1p = b1[S2W_PAD(p)], u1n = b1[S2W_PAD(pn)], u2p = b2[S2W_PAD(p)], u2n = b2[S2W_PAD(pn)];
        b1[S2W_PAD(p)] = csub(cmul(tp, u1p), cmul(gp, u1n));
        b2[S2W_PAD(p)] = cadd(cmul(tp, u2p), cmul(gp, u2n));
        if (pn != p) {
            b1[S2W_PAD(pn)] = csub(cmul(tn, u1n), cmul(gn, u1p));
            b2[S2W_PAD(pn)] = cadd(cmul(tn, u2n), cmul(gn, u2p));
        }
    }
    __syncthreads();
    fft_dit_full_b(buf, T, s_tw, 2 * cpb, bstride);
    if (!has) return;
    const cplx xpole = s_pole[cl];
#pragma unroll
    for (int k = 0; k < RW_MAXPT; ++k) {
        const int t = tl + k * tpc;
        if (t < Lm) {
            const cplx y1 = b1[S2W_PAD(t)], y2 = b2[S2W_PAD(t)];
            const double dl = R.delta[t], ds = R.dsum[t], v = vp[t];
            cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
            if (t & 1) h = cscale(h, -1.0);
            h.x += fma(ds, xs[k].x, v * xpole.x);
            h.y += fma(ds, xs[k].y, v * xpole.y);
            colT[t] = h;
        } else if (t == Lm) {
            colT[t] = cmake(s_dot[cl][0], s_dot[cl][1]);
        }
    }
}

// plan-time: in-place forward transform (natural in, digit-reversed out) of one length-M array, one block
__global__ void __launch_bounds__(256) fft_forward_kernel(cplx *data, FftTab T)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    for (int e = threadIdx.x; e < T.M; e += blockDim.x) buf[S2W_PAD(e)] = data[e];
    __syncthreads();
    fft_dif_full(buf, T, s_tw);
    for (int e = threadIdx.x; e < T.M; e += blockDim.x) data[e] = buf[S2W_PAD(e)];
}

// ---------------------------------------------------------------------------------------------------------------
// plan-time table kernels
// ---------------------------------------------------------------------------------------------------------------
__global__ void twiddle_kernel(cplx *tw, int Mtab)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < Mtab) {
        double s, c;
        sincospi(-2.0 * (double)k / (double)Mtab, &s, &c);
        tw[k] = cmake(c, s);
    }
}

// exp(i pi num/n) with the integer num reduced mod 2n exactly
__device__ __forceinline__ cplx cis_pi_frac(long long num, int n)
{
    long long r = num % (2LL * n);
    if (r < 0) r += 2LL * n;
    double s, c;
    sincospi((double)r / (double)n, &s, &c);
    return cmake(c, s);
}

// chirp[j] = exp(-i pi j^2/n); reweighting phase tables (see reweight_kernel):
//   rw_in1[t]  = exp(i pi [t^2 - (L-1)(2t+1)]/n)       rw_out1[i] = exp(i pi (i + i^2)/n) / n
//   rw_in3[i]  = exp(-i pi (i + i^2)/n)                rw_out3[t] = exp(i pi [(L-1)(2t+1) - t^2]/n)
__global__ void chirp_kernel(cplx *chirp, cplx *rw_in1, cplx *rw_out1, cplx *rw_in3, cplx *rw_out3, int n, int L)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    long long jj = (long long)j * j, mod = (long long)(L - 1) * (2 * j + 1);
    chirp[j] = cis_pi_frac(-jj, n);
    rw_in1[j] = cis_pi_frac(jj - mod, n);
    rw_out1[j] = cscale(cis_pi_frac(j + jj, n), 1.0 / (double)n);
    rw_in3[j] = cis_pi_frac(-(j + jj), n);
    rw_out3[j] = cis_pi_frac(mod - jj, n);
}

// kind 0: b[d mod M] = exp(+i pi d^2/n)/M, |d| < n   (forward DFT);  kind 1: conjugate (inverse DFT);
// kind 2: w(q)/M, |q| < n:  2/(1-q^2) for even q, +-i pi/2 for q = +-1, 0 otherwise   (R3 (iv)).
// One block; transforms in place (digit-reversed output) and writes khat[M].
__global__ void __launch_bounds__(256) kernel_spectrum_kernel(cplx *khat, int kind, FftTab T)
{
    extern __shared__ cplx buf[];
    __shared__ cplx s_tw[S2W_TW_SMEM];
    tw_stage(s_tw, T);
    const int n = T.n, M = T.M;
    const double invM = 1.0 / (double)M;
    for (int e = threadIdx.x; e < M; e += blockDim.x) buf[S2W_PAD(e)] = cmake(0.0, 0.0);
    __syncthreads();
    for (int e = threadIdx.x; e < 2 * n - 1; e += blockDim.x) {
        int d = e - (n - 1);
        cplx v;
        if (kind == 2) {
            if ((d & 1) == 0)
                v = cmake(2.0 / (1.0 - (double)d * (double)d), 0.0);
            else if (d == 1)
                v = cmake(0.0, 1.5707963267948966192);
            else if (d == -1)
                v = cmake(0.0, -1.5707963267948966192);
            else
                v = cmake(0.0, 0.0);
        } else {
            long long r = ((long long)d * d) % (2LL * n);
            double s, c;
            sincospi((double)r / (double)n, &s, &c);
            v = cmake(c, kind == 0 ? s : -s);
        }
        int slot = d < 0 ? d + M : d;
        buf[S2W_PAD(slot)] = cscale(v, invM);
    }
    __syncthreads();
    fft_dif_full(buf, T, s_tw);
    for (int e = threadIdx.x; e < M; e += blockDim.x) khat[e] = buf[S2W_PAD(e)];
}

// dst[b][c][r] = src[b][r][c] for nb matrices of R x C complex values: the adjoint transforms move
// between the ring-major layout F[n][t][m] of the FFT kernels and the column-major layout Ft[n][m][t] of the forward
// contraction without the reweighting kernel that normally does it.  32 x 32 tiles through padded shared memory.
__global__ void __launch_bounds__(256) transpose_kernel(const cplx *__restrict__ src, cplx *__restrict__ dst, int R, int C,
                                                       const double *__restrict__ w)
{
    __shared__ cplx tile[32][33];
    const size_t base = (size_t)blockIdx.z * R * C;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int k = ty; k < 32; k += 8) {
        const int r = r0 + k, c = c0 + tx;
        if (r < R && c < C) tile[k][tx] = w ? cscale(src[base + (size_t)r * C + c], w[r]) : src[base + (size_t)r * C + c];
    }
    __syncthreads();
    for (int k = ty; k < 32; k += 8) {
        const int c = c0 + k, r = r0 + tx;
        if (r < R && c < C) dst[base + (size_t)c * R + r] = tile[tx][k];
    }
}

size_t fft_smem_bytes(const FftTab &T) { return (size_t)fft_padded_len(T.M) * sizeof(cplx); }

}  // namespace

// ---- host launchers -------------------------------------------------------------------------------------------

// S2W_FFT16=0 in the environment keeps the radix-8 kernels (before / after measurements); read once
static bool use_fft16()
{
    static const bool on = [] {
        const char *e = getenv("S2W_FFT16");
        return !(e && e[0] == '0');
    }();
    return on;
}

int launch_twiddles(cplx *tw, int Mtab, cudaStream_t st)
{
    S2W_LAUNCH(twiddle_kernel, (Mtab + 255) / 256, 256, 0, st, tw, Mtab);
    return S2W_OK;
}

int launch_fft_tables(const FftTab &T, cplx *chirp, cplx *rw_in1, cplx *rw_out1, cplx *rw_in3, cplx *rw_out3,
                      cplx *bhat_m, cplx *bhat_p, cplx *what, cudaStream_t st)
{
    S2W_LAUNCH(chirp_kernel, (T.n + 255) / 256, 256, 0, st, chirp, rw_in1, rw_out1, rw_in3, rw_out3, T.n, T.L);
    size_t sm = fft_smem_bytes(T);
    int rc = set_smem(kernel_spectrum_kernel, sm);
    if (rc) return rc;
    S2W_LAUNCH(kernel_spectrum_kernel, 1, 256, sm, st, bhat_m, 0, T);
    S2W_LAUNCH(kernel_spectrum_kernel, 1, 256, sm, st, bhat_p, 1, T);
    S2W_LAUNCH(kernel_spectrum_kernel, 1, 256, sm, st, what, 2, T);
    return S2W_OK;
}

int launch_ring_fwd(bool real, const void *in, cplx *out, int B, int Lg, size_t sig_stride, const FftTab &T,
                    cudaStream_t st)
{
    const int nrows = B * T.nt;
    (void)Lg;
    if (nrows <= 0) return S2W_OK;
    if (ring_pfa4095_supported(real, T)) return launch_ring_pfa4095(true, in, out, nrows, sig_stride, T, st);
    if (ring_pfa255_supported(real, T)) return launch_ring_pfa255(true, in, out, nrows, sig_stride, T, st);
    if (T.nt == T.L && T.bhat16_m && f16_supported(T.M) && use_fft16())
        return launch_ring16(true, real, in, out, nrows, sig_stride, T, st);
    size_t sm = fft_smem_bytes(T);
    int rc;
    if (real) {
        if ((rc = set_smem(ring_fwd_kernel<true>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_fwd_kernel<true>, (nrows + 1) / 2, 256, sm, st, in, out, nrows, sig_stride, T);
    } else {
        if ((rc = set_smem(ring_fwd_kernel<false>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_fwd_kernel<false>, nrows, 256, sm, st, in, out, nrows, sig_stride, T);
    }
    return S2W_OK;
}

int launch_ring_inv(bool real, const cplx *in, void *out, int B, int Lg, size_t sig_stride, const FftTab &T,
                    cudaStream_t st)
{
    const int nrows = B * T.nt;
    (void)Lg;
    if (nrows <= 0) return S2W_OK;
    if (ring_pfa4095_supported(real, T)) return launch_ring_pfa4095(false, in, out, nrows, sig_stride, T, st);
    if (ring_pfa255_supported(real, T)) return launch_ring_pfa255(false, in, out, nrows, sig_stride, T, st);
    if (T.nt == T.L && T.bhat16_m && f16_supported(T.M) && use_fft16())
        return launch_ring16(false, real, in, out, nrows, sig_stride, T, st);
    size_t sm = fft_smem_bytes(T);
    int rc;
    if (real) {
        if ((rc = set_smem(ring_inv_kernel<true>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_inv_kernel<true>, (nrows + 1) / 2, 256, sm, st, in, out, nrows, sig_stride, T);
    } else {
        if ((rc = set_smem(ring_inv_kernel<false>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, ring_inv_kernel<false>, nrows, 256, sm, st, in, out, nrows, sig_stride, T);
    }
    return S2W_OK;
}

static int seqs_per_block(int fit, long long total, int cap);


template <bool REAL, bool MULTI>
static int so3_launch_t(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch,
                        const FftTab &T, int rpb, cudaStream_t st)
{
    size_t sm = (size_t)rpb * fft_smem_bytes(T);
    dim3 grid((T.nt + rpb - 1) / rpb, batch);
    int rc;
    if (fwd) {
        if ((rc = set_smem(so3_fwd_kernel<REAL, MULTI>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_fwd_kernel<REAL, MULTI>), grid, 256, sm, st, in, (cplx *)out, sig_stride, A, T,
                     rpb);
    } else {
        if ((rc = set_smem(so3_inv_kernel<REAL, MULTI>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_inv_kernel<REAL, MULTI>), grid, 256, sm, st, (const cplx *)in, out, sig_stride, A,
                     T, rpb);
    }
    return S2W_OK;
}

static int so3_launch(bool fwd, bool real, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch,
                      const FftTab &T, cudaStream_t st)
{
    const bool mw = T.nt == T.L;  // the radix-16 and ring-pair kernels are written for McEwen-Wiaux grids (L rings)
    if (mw && real && so3_pfa4095_supported(A, T)) return launch_so3_pfa4095(fwd, in, out, sig_stride, A, batch, T, st);
    if (mw && real && 2 * A.N - 1 <= 9 && T.bhat16_m && T.M >= 1024 && f16_supported(T.M) && use_fft16())
        return launch_so3_pair16(fwd, in, out, sig_stride, A, batch, T, st);
    if (mw && !real && so3_pfa255_supported(A, T)) return launch_so3_pfa255(fwd, in, out, sig_stride, A, batch, T, st);
    if (mw && !real && so3_c16_supported(A, T) && use_fft16())
        return launch_so3_c16(fwd, in, out, sig_stride, A, batch, T, st);
    const int rpb = seqs_per_block(4096 / T.M, (long long)T.nt * batch, 32);
    if (mw && rpb == 1 && real) {  // large grids, real signals: ring pairs (the n = 0 row shares one transform)
        const int ng = 2 * A.N - 1;
        size_t sm = ((size_t)fft_padded_len(T.M) + tw_own_entries(T.logM) + (ng <= 9 ? 0 : ng)) * sizeof(cplx);
        dim3 grid((T.L + 1) / 2, batch);
        int rc;
        if (fwd) {
            if ((rc = set_smem(so3_fwd_pair_kernel, sm))) return rc;
            S2W_LAUNCH_C(S2W_K_SO3_FFT, so3_fwd_pair_kernel, grid, 256, sm, st, (const double *)in, (cplx *)out,
                         sig_stride, A, T);
        } else {
            if ((rc = set_smem(so3_inv_pair_kernel, sm))) return rc;
            S2W_LAUNCH_C(S2W_K_SO3_FFT, so3_inv_pair_kernel, grid, 256, sm, st, (const cplx *)in, (double *)out,
                         sig_stride, A, T);
        }
        return S2W_OK;
    }
    if (rpb > 1)
        return real ? so3_launch_t<true, true>(fwd, in, out, sig_stride, A, batch, T, rpb, st)
                    : so3_launch_t<false, true>(fwd, in, out, sig_stride, A, batch, T, rpb, st);
    return real ? so3_launch_t<true, false>(fwd, in, out, sig_stride, A, batch, T, 1, st)
                : so3_launch_t<false, false>(fwd, in, out, sig_stride, A, batch, T, 1, st);
}

int launch_so3_inv(bool real, const cplx *F, void *W, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st)
{
    return so3_launch(false, real, F, W, sig_stride, A, batch, T, st);
}

bool so3_fwd_writes_transposed(bool real, const So3Args &A, const FftTab &T)
{
    return T.nt == T.L && !real && so3_pfa255_supported(A, T);  // the first branch of so3_launch
}

int launch_so3_fwd(bool real, const void *W, size_t sig_stride, cplx *F, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st)
{
    if (A.f_transposed && !so3_fwd_writes_transposed(real, A, T)) {
        set_error("launch_so3_fwd: transposed output is not available for this grid");
        return S2W_EINVAL;
    }
    return so3_launch(true, real, W, F, sig_stride, A, batch, T, st);
}

int launch_fft_forward(cplx *data, const FftTab &T, cudaStream_t st)
{
    size_t sm = fft_smem_bytes(T);
    int rc = set_smem(fft_forward_kernel, sm);
    if (rc) return rc;
    S2W_LAUNCH(fft_forward_kernel, 1, 256, sm, st, data, T);
    return S2W_OK;
}

// sequences per block on small grids: as many as fit the shared-memory budget of one full-size sequence, but never so
// many that the launch drops below ~6 blocks per SM
static int seqs_per_block(int fit, long long total, int cap)
{
    int s = fit < 1 ? 1 : (fit > cap ? cap : fit);
    while (s > 1 && total / s < 900) s >>= 1;
    return s;
}

int launch_transpose(const cplx *src, cplx *dst, int R, int C, int nb, cudaStream_t st, const double *w)
{
    if (R <= 0 || C <= 0 || nb <= 0) return S2W_OK;
    for (int b0 = 0; b0 < nb; b0 += 65535) {  // gridDim.z limit
        const int nz = nb - b0 < 65535 ? nb - b0 : 65535;
        dim3 grid((C + 31) / 32, (R + 31) / 32, nz);
        S2W_LAUNCH_C(w ? S2W_K_REWEIGHT : S2W_K_OTHER, transpose_kernel, grid, 256, 0, st, src + (size_t)b0 * R * C,
                     dst + (size_t)b0 * R * C, R, C, w);
    }
    return S2W_OK;
}

int launch_reweight_th(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const RwTab &R, cudaStream_t st)
{
    if (A.nn <= 0) return S2W_OK;
    if (R.TG16 && R.fft.M >= 256 && R.fft.M <= 4096 && use_fft16()) return launch_reweight16(F, Ft, A, batch, R, st);
    const int ncol = A.Md * A.nn * batch;
    const int cpb = seqs_per_block(2048 / R.fft.M, ncol, RW_MAXCPB);
    size_t sm = 2 * (size_t)cpb * fft_padded_len(R.fft.M) * sizeof(cplx);
    int rc;
    if (cpb > 1) {
        if ((rc = set_smem(reweight_th_multi_kernel, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight_th_multi_kernel, (ncol + cpb - 1) / cpb, 256, sm, st, F, Ft, A, R, cpb,
                     ncol);
        return S2W_OK;
    }
    dim3 grid(A.Md, A.nn, batch);
    if (R.L <= 4 * 256) {  // four values per thread: no spills under the 80-register cap of three blocks per SM
        if ((rc = set_smem(reweight_th_kernel<4>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight_th_kernel<4>, grid, 256, sm, st, F, Ft, A, R);
        return S2W_OK;
    }
    if ((rc = set_smem(reweight_th_kernel<RW_MAXPT>, sm))) return rc;
    S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight_th_kernel<RW_MAXPT>, grid, 256, sm, st, F, Ft, A, R);
    return S2W_OK;
}

int launch_reweight(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const FftTab &T, cudaStream_t st)
{
    if (A.nn <= 0) return S2W_OK;
    size_t sm = fft_smem_bytes(T);
    int rc = set_smem(reweight_kernel, sm);
    if (rc) return rc;
    dim3 grid(A.Md, A.nn, batch);
    S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight_kernel, grid, 256, sm, st, F, Ft, A, T);
    return S2W_OK;
}

}  // namespace s2w
