// fft16_kernels.cu -- rows a8 (alpha, gamma FFT) and a2 (theta reweighting) on the register-fed radix-16 core of
// fft16_core.cuh, for Bluestein / Toeplitz lengths 1024, 2048 and 4096 (grids with 129 <= L_j <= 1024: every grid that
// matters for the time of BASELINE configs 2, 3 and 5).  Other lengths stay on the radix-8 kernels of ring_fft.cu.
//
//   a8  W(gamma_g, beta_t, alpha_a) = sum_{m,n} F_mn(beta_t) e^{i(m alpha_a + n gamma_g)}            (Eq. 5/47)
//       F_mn(beta_t) = 1/(n_a n_g) sum_{a,g} W e^{-i(m alpha_a + n gamma_g)}                         (Eq. 48)
//   a2  h = reweight(F) per (m, n) column along theta, Toeplitz/Hankel form                          (R3)
//
// A block works on NB = 4096 / M sequences at a time ("round").  Thread tid owns elements tid + 256 c (c < M/512) of
// every sequence of a round: it loads them from global memory (coalesced), and gets the same elements of the result
// back in registers.
#include "fft16_core.cuh"
#include "kernels.h"
#include "smem_attr.cuh"

namespace s2w {

namespace {

__device__ __forceinline__ cplx cis_2pi(int num, int den)  // exp(2 pi i num/den), num reduced mod den
{
    int r = num % den;
    if (r < 0) r += den;
    double s, c;
    sincospi(2.0 * (double)r / (double)den, &s, &c);
    return cmake(c, s);
}

// rows n = 0 / n > 0 of a real-signal launch, and the gamma phases e^{+- i n gamma_g} of the rows n > 0
struct RowSet {
    int q0, np;
};
__device__ __forceinline__ RowSet so3_rows(const So3Args &A, int sign, cplx *gph, int *s_rowp, int *s_rowm)
{
    const int ng = 2 * A.N - 1;
    RowSet r;
    r.q0 = -1;
    r.np = 0;
    for (int q = 0; q < A.nn; ++q) {
        if (A.n_val[q] == 0) r.q0 = q;
        if (A.n_val[q] > 0 && r.np < 4) {
            for (int g = threadIdx.x; g < ng; g += blockDim.x) gph[r.np * ng + g] = cis_2pi(sign * A.n_val[q] * g, ng);
            if (threadIdx.x == 0) {
                s_rowp[r.np] = A.n_row[q];
                s_rowm[r.np] = A.n_rowm[q];
            }
            ++r.np;
        }
    }
    return r;
}

// The I/O stages around a round work on the thread's 8 elements e = q HR + c (sequence q, element tid + 256 c) in ROLLED
// loops over batches of 4 (or 2), loads first: fully unrolled they keep the addresses and loaded values of all 8 elements
// live at once and spill (ptxas: 0.8-1.6 KB of local memory per thread, as much LSU traffic as the transform itself).
// XE(h, j) is element 4h + j of the register array x[NB][R1] for a rolled h and an unrolled j: one select per register.
#define XE_GET(x, HRv, h, j) ((h) ? (x)[(4 + (j)) / (HRv)][(4 + (j)) % (HRv)] : (x)[(j) / (HRv)][(j) % (HRv)])
#define XE_SET(x, HRv, h, j, val)                                   \
    do {                                                            \
        const cplx _v = (val);                                      \
        if (h)                                                      \
            (x)[(4 + (j)) / (HRv)][(4 + (j)) % (HRv)] = _v;         \
        else                                                        \
            (x)[(j) / (HRv)][(j) % (HRv)] = _v;                     \
    } while (0)

// the same for batches of 2: element 2h + j, h = 0..3 rolled, j = 0..1 unrolled
#define X2_AT(x, HRv, e) (x)[(e) / (HRv)][(e) % (HRv)]
#define X2_GET(x, HRv, h, j) \
    ((h) == 0 ? X2_AT(x, HRv, j) : (h) == 1 ? X2_AT(x, HRv, 2 + (j)) : (h) == 2 ? X2_AT(x, HRv, 4 + (j)) : X2_AT(x, HRv, 6 + (j)))
#define X2_SET(x, HRv, h, j, val)                   \
    do {                                            \
        const cplx _v = (val);                      \
        if ((h) == 0) X2_AT(x, HRv, j) = _v;        \
        if ((h) == 1) X2_AT(x, HRv, 2 + (j)) = _v;  \
        if ((h) == 2) X2_AT(x, HRv, 4 + (j)) = _v;  \
        if ((h) == 3) X2_AT(x, HRv, 6 + (j)) = _v;  \
    } while (0)

// ---------------------------------------------------------------------------------------------------------------
// a8 analysis, real signals, 2N-1 <= 9: F[b][row][t][m >= 0] -> W[b][g][t][a] (real).  A block owns NB PAIRS of rings.
// Round 0: the rows n = 0 of a pair's two rings share one transform (X_t0 + i X_t1, Hermitian in m); then one round
// per row n > 0 and ring parity.  Until a ring's last row the transforms V_n(alpha) are parked in the ring's own output
// planes (each thread reads back only what it wrote), and every plane is written once in the last round.
// ---------------------------------------------------------------------------------------------------------------
template <int R1>
__global__ void __launch_bounds__(256, 2) so3_inv_pair16_kernel(const cplx *__restrict__ F, double *__restrict__ W,
                                                               size_t sig_stride, So3Args A, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 / 2;
    extern __shared__ cplx buf[];
    __shared__ cplx gph[36];
    __shared__ int s_rowp[4], s_rowm[4];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L, ng = 2 * A.N - 1;
    const cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * L;
    double *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    const RowSet rs = so3_rows(A, +1, gph, s_rowp, s_rowm);
    const int q0 = rs.q0, np = rs.np;
    __syncthreads();
    cplx x[NB][R1];
    if (q0 >= 0) {
        const cplx *Xrow = Fb + (size_t)A.n_row[q0] * L * L;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            cplx a[4], cc[4], ch[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t0 = 2 * (blockIdx.x * NB + q), k = threadIdx.x + 256 * c;
                const int kk = (k < n && t0 < L) ? k : 0, m = kk < L ? kk : n - kk;
                const cplx *X0 = Xrow + (size_t)(t0 < L ? t0 : 0) * L;
                a[j] = X0[m];
                cc[j] = X0[(t0 + 1 < L ? L : 0) + m];
                ch[j] = __ldg(&T.chirp[kk]);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t0 = 2 * (blockIdx.x * NB + q), k = threadIdx.x + 256 * c;
                cplx av = a[j], cv = t0 + 1 < L ? cc[j] : cmake(0.0, 0.0);
                if (k >= L) {
                    av = cconj(av);
                    cv = cconj(cv);
                }
                XE_SET(x, HR, h, j, (k < n && t0 < L) ? cmulc(cmake(av.x - cv.y, av.y + cv.x), ch[j]) : cmake(0.0, 0.0));
            }
        }
        f16_convolve_half<R1>(buf, x, T.bhat16_p, tw);
        const int nplanes = np ? 1 : ng;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t0 = 2 * (blockIdx.x * NB + q), a = threadIdx.x + 256 * c;
                if (a < n && t0 < L) {
                    const cplx v = cmulc(XE_GET(x, HR, h, j), __ldg(&T.chirp[a]));  // V_0 of ring t0 + i V_0 of ring t0+1
                    double *Wr = Wb + (size_t)t0 * n + a;
                    for (int g = 0; g < nplanes; ++g) {
                        Wr[g * plane] = v.x;
                        if (t0 + 1 < L) Wr[g * plane + n] = v.y;
                    }
                }
            }
        }
    }
#pragma unroll 1
    for (int ri = 0; ri < 2 * np; ++ri) {
        const int r = ri / np, i = ri - r * np;
        const cplx *Fp = Fb + (size_t)s_rowp[i] * L * L, *Fm = Fb + (size_t)s_rowm[i] * L * L;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            cplx v[4], ch[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, k = threadIdx.x + 256 * c;
                const int kk = (k < n && t < L) ? k : 0;
                const size_t ro = (size_t)(t < L ? t : 0) * L;
                v[j] = *(kk < L ? Fp + ro + kk : Fm + ro + (n - kk));
                ch[j] = __ldg(&T.chirp[kk]);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, k = threadIdx.x + 256 * c;
                const cplx vv = k >= L ? cconj(v[j]) : v[j];
                XE_SET(x, HR, h, j, (k < n && t < L) ? cmulc(vv, ch[j]) : cmake(0.0, 0.0));
            }
        }
        f16_convolve_half<R1>(buf, x, T.bhat16_p, tw);
        if (i + 1 < np) {  // park V_n in planes 2i+1, 2i+2 of the ring
#pragma unroll 1
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int e = 4 * h + j, q = e / HR, c = e % HR;
                    const int t = 2 * (blockIdx.x * NB + q) + r, a = threadIdx.x + 256 * c;
                    if (a < n && t < L) {
                        const cplx v = cmulc(XE_GET(x, HR, h, j), __ldg(&T.chirp[a]));
                        double *Wr = Wb + (size_t)t * n + a;
                        Wr[(2 * i + 1) * plane] = v.x;
                        Wr[(2 * i + 2) * plane] = v.y;
                    }
                }
            }
            continue;
        }
#pragma unroll 1
        for (int h = 0; h < 4; ++h) {  // last row of the ring: every gamma plane written once; two elements at a time
            cplx xv[2];
            double sc[2][7];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                xv[j] = X2_GET(x, HR, h, j);
                const int e = 2 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, a = threadIdx.x + 256 * c;
                const bool on = a < n && t < L;
                const double *Wr = Wb + (on ? (size_t)t * n + a : 0);
#pragma unroll
                for (int s = 0; s < 7; ++s) sc[j][s] = 0.0;
                if (q0 >= 0) sc[j][0] = Wr[0];
#pragma unroll
                for (int s = 1; s < 7; ++s)
                    if (s < 2 * np - 1) sc[j][s] = Wr[s * plane];
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int e = 2 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, a = threadIdx.x + 256 * c;
                if (a >= n || t >= L) continue;
                const cplx v = cmulc(xv[j], __ldg(&T.chirp[a]));
                double *Wr = Wb + (size_t)t * n + a;
                double out[9];
#pragma unroll
                for (int g = 0; g < 9; ++g) {
                    const cplx ph = gph[(np - 1) * ng + (g < ng ? g : 0)];
                    out[g] = fma(2.0, ph.x * v.x - ph.y * v.y, sc[j][0]);
                }
#pragma unroll
                for (int jj = 0; jj < 3; ++jj)
                    if (jj + 1 < np) {
#pragma unroll
                        for (int g = 0; g < 9; ++g) {
                            const cplx ph = gph[jj * ng + (g < ng ? g : 0)];
                            out[g] = fma(2.0, ph.x * sc[j][2 * jj + 1] - ph.y * sc[j][2 * jj + 2], out[g]);
                        }
                    }
#pragma unroll
                for (int g = 0; g < 9; ++g)
                    if (g < ng) Wr[g * plane] = out[g];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a8 synthesis, real signals, 2N-1 <= 9: W[b][g][t][a] -> F[b][row][t][m >= 0].  The gamma planes of a ring cross the
// memory system once: the gather forms the gamma sums Y_n(alpha) of all rows, feeds the row n = 0 (ring t0 real part,
// ring t0+1 imaginary part) straight into round 0 and parks the rows n > 0, chirp applied, in the ring's own output
// rows F_{., n}, F_{., -n} (2L >= 2L-1 entries), from where that row's round takes them back (same thread).
// ---------------------------------------------------------------------------------------------------------------
template <int R1>
__global__ void __launch_bounds__(256, 2) so3_fwd_pair16_kernel(const double *__restrict__ W, cplx *__restrict__ F,
                                                               size_t sig_stride, So3Args A, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 / 2, M = R1 * 256;
    extern __shared__ cplx buf[];
    __shared__ cplx gph[36];
    __shared__ int s_rowp[4], s_rowm[4];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L, ng = 2 * A.N - 1;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * L;
    const double *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    const RowSet rs = so3_rows(A, -1, gph, s_rowp, s_rowm);
    const int q0 = rs.q0, np = rs.np;
    __syncthreads();
    // gather: every gamma plane of both rings of a pair once, two alpha samples (36 loads) at a time
#pragma unroll 1
    for (int h = 0; h < 4; ++h) {
        double wv[2][2][9];
        cplx ch[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int e = 2 * h + j, q = e / HR, c = e % HR;
            const int t0 = 2 * (blockIdx.x * NB + q), a = threadIdx.x + 256 * c;
            const int aa = a < n ? a : 0;
            const double *W0 = Wb + (size_t)(t0 < L ? t0 : 0) * n + aa, *W1 = Wb + (size_t)(t0 + 1 < L ? t0 + 1 : 0) * n + aa;
            ch[j] = __ldg(&T.chirp[aa]);
#pragma unroll
            for (int g = 0; g < 9; ++g) {
                const size_t o = (size_t)(g < ng ? g : 0) * plane;
                wv[j][0][g] = W0[o];
                wv[j][1][g] = W1[o];
            }
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int e = 2 * h + j, q = e / HR, c = e % HR;
            const int t0 = 2 * (blockIdx.x * NB + q), a = threadIdx.x + 256 * c;
            const bool has0 = t0 < L && a < n, has1 = t0 + 1 < L && a < n;
#pragma unroll
            for (int g = 0; g < 9; ++g) {
                if (g >= ng || !has0) wv[j][0][g] = 0.0;
                if (g >= ng || !has1) wv[j][1][g] = 0.0;
            }
            double y0 = 0.0, y1 = 0.0;
#pragma unroll
            for (int g = 0; g < 9; ++g) {
                y0 += wv[j][0][g];
                y1 += wv[j][1][g];
            }
            // round 0's input goes through the thread's own column slot of the buffer, not through 32 live registers: with
            // them the 38 loads of a batch spilled, and a spill store of a just-loaded value waits for that load -- the
            // batch's loads went out one DRAM round trip after the other (43 % of the kernel's samples sat here)
            buf[F16_PAD(q * M + a)] = cmul(cscale(cmake(y0, y1), inv_ng), ch[j]);
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (r == 0 ? !has0 : !has1) continue;
                for (int i = 0; i < np; ++i) {
                    cplx y = cmake(0.0, 0.0);
#pragma unroll
                    for (int g = 0; g < 9; ++g) {
                        const cplx ph = gph[i * ng + (g < ng ? g : 0)];
                        y.x = fma(ph.x, wv[j][r][g], y.x);
                        y.y = fma(ph.y, wv[j][r][g], y.y);
                    }
                    y = cmul(cscale(y, inv_ng), ch[j]);
                    cplx *dst = a < L ? Fb + ((size_t)s_rowp[i] * L + t0 + r) * L + a
                                      : Fb + ((size_t)s_rowm[i] * L + t0 + r) * L + (a - L);
                    *dst = y;
                }
            }
        }
    }
    cplx x[NB][R1];
    if (q0 >= 0) {
#pragma unroll
        for (int q = 0; q < NB; ++q)
#pragma unroll
            for (int c = 0; c < HR; ++c) x[q][c] = buf[F16_PAD(q * M + threadIdx.x + 256 * c)];
        f16_convolve_half<R1>(buf, x, T.bhat16_m, tw);
        // u(k) = chirp(k) y(k) back into the thread's own column slots, then F0[m], F1[m] from u(m), u(n - m)
#pragma unroll
        for (int q = 0; q < NB; ++q)
#pragma unroll
            for (int c = 0; c < HR; ++c) {
                const int k = threadIdx.x + 256 * c;
                buf[F16_PAD(q * M + k)] = cmul(x[q][c], __ldg(&T.chirp[k < n ? k : 0]));
            }
        __syncthreads();
#pragma unroll 1
        for (int q = 0; q < NB; ++q) {
            const int t0 = 2 * (blockIdx.x * NB + q);
            if (t0 >= L) continue;
            const bool has1 = t0 + 1 < L;
            cplx *F0 = Fb + ((size_t)A.n_row[q0] * L + t0) * L, *F1 = F0 + L;
            for (int m = threadIdx.x; m < L; m += 256) {
                const cplx a = buf[F16_PAD(q * M + m)], c = cconj(buf[F16_PAD(q * M + (m == 0 ? 0 : n - m))]);
                const cplx sm = cadd(a, c), df = csub(a, c);
                F0[m] = cscale(sm, 0.5 * inv_n);
                if (has1) F1[m] = cmake(0.5 * inv_n * df.y, -0.5 * inv_n * df.x);
            }
        }
        __syncthreads();
    }
#pragma unroll 1
    for (int ri = 0; ri < 2 * np; ++ri) {
        const int r = ri / np, i = ri - r * np;
        cplx *Fp = Fb + (size_t)s_rowp[i] * L * L, *Fm = Fb + (size_t)s_rowm[i] * L * L;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            cplx v[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, a = threadIdx.x + 256 * c;
                const int aa = (a < n && t < L) ? a : 0;
                const size_t ro = (size_t)(t < L ? t : 0) * L;
                v[j] = *(aa < L ? Fp + ro + aa : Fm + ro + (aa - L));
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, a = threadIdx.x + 256 * c;
                XE_SET(x, HR, h, j, (a < n && t < L) ? v[j] : cmake(0.0, 0.0));
            }
        }
        f16_convolve_half<R1>(buf, x, T.bhat16_m, tw);
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int e = 4 * h + j, q = e / HR, c = e % HR;
                const int t = 2 * (blockIdx.x * NB + q) + r, k = threadIdx.x + 256 * c;
                if (k >= n || t >= L) continue;
                const cplx u = cscale(cmul(XE_GET(x, HR, h, j), __ldg(&T.chirp[k])), inv_n);
                const size_t ro = (size_t)t * L;
                if (k < L) Fp[ro + k] = u;
                if (k == 0 || k >= L) Fm[ro + (k == 0 ? 0 : n - k)] = cconj(u);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a2 on the radix-16 core: the Toeplitz/Hankel form of DESIGN.md 6.3 (see reweight_th_kernel in ring_fft.cu for the
// algebra), M2 = R1 * 256 = 2048 or 1024.  A block owns NC = 8 / R1 columns, two sequences each (u1 = a x, u2 = delta a x);
// thread tid holds the ring values x_t, t = tid + 256 c, of its columns in registers from the first load to the last
// store.  The spectra U(k) and U(-k) meet between the innermost forward and inverse passes: position
// p = j1 256 + j2 16 + j3 holds k = j1 + R1 (j2 + 16 j3), so the partners of a thread's 16 contiguous positions are 16
// contiguous positions of another thread, in reverse order.
// ---------------------------------------------------------------------------------------------------------------
template <int R1>
__global__ void __launch_bounds__(256, 2) reweight16_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A,
                                                           RwTab R, int ncolumns)
{
    constexpr int NB = 16 / R1, NC = NB / 2, HR = R1 >= 2 ? R1 / 2 : 1, M = R1 * 256;
    extern __shared__ cplx buf[];
    __shared__ cplx s_part[NC][8];
    __shared__ cplx s_pole[NC];
    const F16Tw tw = f16_twiddles<R1>();
    const int L = R.L, Lm = L - 1;
    cplx xs[NC][HR];
    cplx x[NB][R1];
    int par_of[NC];
    cplx *colT_of[NC];
#pragma unroll
    for (int ci = 0; ci < NC; ++ci) {
        const int colid = blockIdx.x * NC + ci;
        const bool has = colid < ncolumns;
        const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
        const int m = A.isReal ? mi : mi - (L - 1);
        const int nv = has ? A.n_val[q] : 0, row = has ? A.n_row[q] : 0;
        const int par = ((m + nv) & 1) ? 1 : 0;  // 0: sigma = +1, 1: sigma = -1
        par_of[ci] = par;
        const cplx *col = F + ((size_t)(has ? b : 0) * A.nrows + row) * (size_t)L * A.Md + (has ? mi : 0);
        colT_of[ci] = has ? Ft + (((size_t)b * A.nrows + row) * A.Md + mi) * (size_t)L : nullptr;
        const double *rp = R.rpole + par * L;
        cplx dot = cmake(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int t = threadIdx.x + 256 * c;
            cplx xv = cmake(0.0, 0.0);
            if (t < L && has) {
                xv = col[(size_t)t * A.Md];
                const double r = rp[t];
                dot.x = fma(r, xv.x, dot.x);
                dot.y = fma(r, xv.y, dot.y);
            }
            xs[ci][c] = xv;
            if (t == Lm) s_pole[ci] = xv;
            cplx u1 = cmake(0.0, 0.0), u2 = u1;
            if (t < Lm) {
                u1 = (t & 1) ? cscale(xv, -1.0) : xv;
                u2 = cscale(u1, R.delta[t]);
            }
            x[2 * ci][c] = u1;
            x[2 * ci + 1][c] = u2;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
            dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
        }
        if ((threadIdx.x & 31) == 0) s_part[ci][threadIdx.x >> 5] = dot;
    }
#pragma unroll
    for (int q = 0; q < NB; ++q) f16_pass1_fwd<R1, (R1 > 1)>(buf, q, x[q], tw);
    __syncthreads();
    f16_pass2_fwd(buf, tw);
    __syncwarp();
    f16_pass3_fwd(buf);
    __syncthreads();
    {
        const int hw = threadIdx.x >> 4, j2 = threadIdx.x & 15;
        const int sq = hw / R1, j1 = hw % R1;                       // sequence, sub-block inside it
        const int j1p = (R1 - j1) % R1, j2p = j1 ? 15 - j2 : (16 - j2) & 15;
        const bool shifted = j1 == 0 && j2 == 0;                    // partner of j3 is (16 - j3) % 16, else 15 - j3
        cplx *own = buf + F16_PAD(hw * 256 + j2 * 16);
        const cplx *prt = buf + F16_PAD(sq * M + j1p * 256 + j2p * 16);
        const cplx *tg = R.TG16 + (j1 * 256 + j2);                   // [2][M2] in the storage order F16_TPOS
        double sg = par_of[0] ? -1.0 : 1.0;
#pragma unroll
        for (int ci = 1; ci < NC; ++ci)
            if ((sq >> 1) == ci) sg = par_of[ci] ? -1.0 : 1.0;
        if (!(sq & 1)) sg = -sg;                                    // u1: T - sigma H, u2: T + sigma H
        cplx v[16];
#pragma unroll
        for (int j3 = 0; j3 < 16; ++j3) {
            const cplx u = own[j3], un = prt[shifted ? (16 - j3) & 15 : 15 - j3];
            const cplx th = __ldg(&tg[16 * j3]), gh = cscale(__ldg(&tg[M + 16 * j3]), sg);
            v[j3] = cadd(cmul(th, u), cmul(gh, un));
        }
        __syncthreads();                                            // every partner value has been read
        bfly16<true>(v);
#pragma unroll
        for (int j3 = 0; j3 < 16; ++j3) own[j3] = v[j3];
    }
    __syncwarp();
    f16_pass2_inv(buf, tw);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NB; ++q) f16_pass1_inv<R1, (R1 > 1)>(buf, q, x[q], tw);
#pragma unroll
    for (int ci = 0; ci < NC; ++ci) {
        cplx *colT = colT_of[ci];
        if (!colT) continue;
        const double *vp = R.vpole + par_of[ci] * L;
        const cplx xpole = s_pole[ci];
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int t = threadIdx.x + 256 * c;
            if (t < Lm) {
                const cplx y1 = x[2 * ci][c], y2 = x[2 * ci + 1][c];
                const double dl = R.delta[t], ds = R.dsum[t], vv = vp[t];
                cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
                if (t & 1) h = cscale(h, -1.0);
                h.x += fma(ds, xs[ci][c].x, vv * xpole.x);
                h.y += fma(ds, xs[ci][c].y, vv * xpole.y);
                colT[t] = h;
            } else if (t == Lm) {
                cplx acc = cmake(0.0, 0.0);
                for (int w = 0; w < 8; ++w) acc = cadd(acc, s_part[ci][w]);
                colT[t] = acc;
            }
        }
    }
}

__device__ __forceinline__ void rw_cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

template <int R1>
__global__ void __launch_bounds__(256, 2) reweight16p_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A,
                                                           RwTab R, int ncolumns)
{
    constexpr int NB = 16 / R1, NC = NB / 2, HR = R1 >= 2 ? R1 / 2 : 1, M = R1 * 256;
    extern __shared__ cplx buf[];
    __shared__ cplx s_part[NC][8];
    __shared__ cplx s_pole[NC];
    const F16Tw tw = f16_twiddles<R1>();
    const int L = R.L, Lm = L - 1;
    // persistent blocks: the ring values of the NEXT column group arrive by cp.async in a staging area (NC x L <= 1024
    // values) while the current group is transformed -- the strided column reads (one 16-byte element per ring, Md
    // elements apart) were the exposed latency at the head of every block
    cplx *stg = buf + F16_BUF;
    const int ngroups = (ncolumns + NC - 1) / NC;
    auto prefetch = [&](int grp) {
#pragma unroll
        for (int ci = 0; ci < NC; ++ci) {
            const int colid = grp * NC + ci;
            if (colid >= ncolumns) continue;
            const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
            const cplx *col = F + ((size_t)b * A.nrows + A.n_row[q]) * (size_t)L * A.Md + mi;
#pragma unroll
            for (int c = 0; c < HR; ++c) {
                const int t = threadIdx.x + 256 * c;
                if (t < L) rw_cp_async16(stg + ci * L + t, col + (size_t)t * A.Md);
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if ((int)blockIdx.x < ngroups) prefetch(blockIdx.x);
    for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();  // the staged values of every thread; the previous group's use of buf, s_part, s_pole
    cplx xs[NC][HR];
    cplx x[NB][R1];
    int par_of[NC];
    cplx *colT_of[NC];
#pragma unroll
    for (int ci = 0; ci < NC; ++ci) {
        const int colid = grp * NC + ci;
        const bool has = colid < ncolumns;
        const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
        const int m = A.isReal ? mi : mi - (L - 1);
        const int nv = has ? A.n_val[q] : 0, row = has ? A.n_row[q] : 0;
        const int par = ((m + nv) & 1) ? 1 : 0;  // 0: sigma = +1, 1: sigma = -1
        par_of[ci] = par;
        colT_of[ci] = has ? Ft + (((size_t)b * A.nrows + row) * A.Md + mi) * (size_t)L : nullptr;
        const double *rp = R.rpole + par * L;
        cplx dot = cmake(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int t = threadIdx.x + 256 * c;
            cplx xv = cmake(0.0, 0.0);
            if (t < L && has) {
                xv = stg[ci * L + t];
                const double r = rp[t];
                dot.x = fma(r, xv.x, dot.x);
                dot.y = fma(r, xv.y, dot.y);
            }
            xs[ci][c] = xv;
            if (t == Lm) s_pole[ci] = xv;
            cplx u1 = cmake(0.0, 0.0), u2 = u1;
            if (t < Lm) {
                u1 = (t & 1) ? cscale(xv, -1.0) : xv;
                u2 = cscale(u1, R.delta[t]);
            }
            x[2 * ci][c] = u1;
            x[2 * ci + 1][c] = u2;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
            dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
        }
        if ((threadIdx.x & 31) == 0) s_part[ci][threadIdx.x >> 5] = dot;
    }
    __syncthreads();  // every thread has taken its staged values
    if (grp + (int)gridDim.x < ngroups) prefetch(grp + gridDim.x);
#pragma unroll
    for (int q = 0; q < NB; ++q) f16_pass1_fwd<R1, (R1 > 1)>(buf, q, x[q], tw);
    __syncthreads();
    f16_pass2_fwd(buf, tw);
    __syncwarp();
    f16_pass3_fwd(buf);
    __syncthreads();
    {
        const int hw = threadIdx.x >> 4, j2 = threadIdx.x & 15;
        const int sq = hw / R1, j1 = hw % R1;                       // sequence, sub-block inside it
        const int j1p = (R1 - j1) % R1, j2p = j1 ? 15 - j2 : (16 - j2) & 15;
        const bool shifted = j1 == 0 && j2 == 0;                    // partner of j3 is (16 - j3) % 16, else 15 - j3
        cplx *own = buf + F16_PAD(hw * 256 + j2 * 16);
        const cplx *prt = buf + F16_PAD(sq * M + j1p * 256 + j2p * 16);
        const cplx *tg = R.TG16 + (j1 * 256 + j2);                   // [2][M2] in the storage order F16_TPOS
        double sg = par_of[0] ? -1.0 : 1.0;
#pragma unroll
        for (int ci = 1; ci < NC; ++ci)
            if ((sq >> 1) == ci) sg = par_of[ci] ? -1.0 : 1.0;
        if (!(sq & 1)) sg = -sg;                                    // u1: T - sigma H, u2: T + sigma H
        cplx v[16];
#pragma unroll
        for (int j3 = 0; j3 < 16; ++j3) {
            const cplx u = own[j3], un = prt[shifted ? (16 - j3) & 15 : 15 - j3];
            const cplx th = __ldg(&tg[16 * j3]), gh = cscale(__ldg(&tg[M + 16 * j3]), sg);
            v[j3] = cadd(cmul(th, u), cmul(gh, un));
        }
        __syncthreads();                                            // every partner value has been read
        bfly16<true>(v);
#pragma unroll
        for (int j3 = 0; j3 < 16; ++j3) own[j3] = v[j3];
    }
    __syncwarp();
    f16_pass2_inv(buf, tw);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NB; ++q) f16_pass1_inv<R1, (R1 > 1)>(buf, q, x[q], tw);
#pragma unroll
    for (int ci = 0; ci < NC; ++ci) {
        cplx *colT = colT_of[ci];
        if (!colT) continue;
        const double *vp = R.vpole + par_of[ci] * L;
        const cplx xpole = s_pole[ci];
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int t = threadIdx.x + 256 * c;
            if (t < Lm) {
                const cplx y1 = x[2 * ci][c], y2 = x[2 * ci + 1][c];
                const double dl = R.delta[t], ds = R.dsum[t], vv = vp[t];
                cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
                if (t & 1) h = cscale(h, -1.0);
                h.x += fma(ds, xs[ci][c].x, vv * xpole.x);
                h.y += fma(ds, xs[ci][c].y, vv * xpole.y);
                colT[t] = h;
            } else if (t == Lm) {
                cplx acc = cmake(0.0, 0.0);
                for (int w = 0; w < 8; ++w) acc = cadd(acc, s_part[ci][w]);
                colT[t] = acc;
            }
        }
    }
    }  // column groups
}

// a2 at Toeplitz length 4096 (the grid of L_j = 2048, BASELINE config 4): one column per block; its two sequences
// u1 = a x and u2 = delta a x go through the one 4096-element buffer one after the other (y1 waits in registers), the
// thread keeps the ring values x_t, t = tid + 256 c (c < 8), in registers throughout.  Same algebra and tables as above.
__global__ void __launch_bounds__(256, 2) reweight16w_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A,
                                                            RwTab R, int ncolumns)
{
    constexpr int R1 = 16, HR = 8, M = R1 * 256;
    extern __shared__ cplx buf[];
    __shared__ cplx s_part[8];
    __shared__ cplx s_pole;
    const F16Tw tw = f16_twiddles<R1>();
    const int L = R.L, Lm = L - 1;
    for (int colid = blockIdx.x; colid < ncolumns; colid += gridDim.x) {  // resident blocks walk over the columns
    const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
    const int m = A.isReal ? mi : mi - (L - 1);
    const int par = ((m + A.n_val[q]) & 1) ? 1 : 0;  // 0: sigma = +1, 1: sigma = -1
    const cplx *col = F + ((size_t)b * A.nrows + A.n_row[q]) * (size_t)L * A.Md + mi;
    cplx *colT = Ft + (((size_t)b * A.nrows + A.n_row[q]) * A.Md + mi) * (size_t)L;
    const double *rp = R.rpole + par * L, *vp = R.vpole + par * L;
    cplx xs[HR], x[1][R1];
    cplx *sy1 = buf + F16_BUF + threadIdx.x;  // y1 of the first sequence waits here (own slots: element tid + 256 c)
    cplx dot = cmake(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < HR; ++c) {
        const int t = threadIdx.x + 256 * c;
        cplx xv = cmake(0.0, 0.0);
        if (t < L) {
            xv = col[(size_t)t * A.Md];
            const double r = rp[t];
            dot.x = fma(r, xv.x, dot.x);
            dot.y = fma(r, xv.y, dot.y);
        }
        xs[c] = xv;
        if (t == Lm) s_pole = xv;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
        dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
    }
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = dot;
#pragma unroll 1
    for (int sq = 0; sq < 2; ++sq) {
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int t = threadIdx.x + 256 * c;
            cplx u = cmake(0.0, 0.0);
            if (t < Lm) {
                u = (t & 1) ? cscale(xs[c], -1.0) : xs[c];
                if (sq) u = cscale(u, R.delta[t]);
            }
            x[0][c] = u;
        }
        f16_pass1_fwd<R1, true>(buf, 0, x[0], tw);
        __syncthreads();
        f16_pass2_fwd(buf, tw);
        __syncwarp();
        f16_pass3_fwd(buf);
        __syncthreads();
        {
            const int j1 = threadIdx.x >> 4, j2 = threadIdx.x & 15;
            const int j1p = (R1 - j1) % R1, j2p = j1 ? 15 - j2 : (16 - j2) & 15;
            const bool shifted = j1 == 0 && j2 == 0;                    // partner of j3 is (16 - j3) % 16, else 15 - j3
            cplx *own = buf + F16_PAD(j1 * 256 + j2 * 16);
            const cplx *prt = buf + F16_PAD(j1p * 256 + j2p * 16);
            const cplx *tg = R.TG16 + (j1 * 256 + j2);                   // [2][M2] in the storage order F16_TPOS
            double sg = par ? -1.0 : 1.0;
            if (!sq) sg = -sg;                                          // u1: T - sigma H, u2: T + sigma H
            cplx v[16];
#pragma unroll
            for (int j3 = 0; j3 < 16; ++j3) {
                const cplx u = own[j3], un = prt[shifted ? (16 - j3) & 15 : 15 - j3];
                const cplx th = __ldg(&tg[16 * j3]), gh = cscale(__ldg(&tg[M + 16 * j3]), sg);
                v[j3] = cadd(cmul(th, u), cmul(gh, un));
            }
            __syncthreads();                                            // every partner value has been read
            bfly16<true>(v);
#pragma unroll
            for (int j3 = 0; j3 < 16; ++j3) own[j3] = v[j3];
        }
        __syncwarp();
        f16_pass2_inv(buf, tw);
        __syncthreads();
        f16_pass1_inv<R1, true>(buf, 0, x[0], tw);
        if (!sq) {
#pragma unroll
            for (int c = 0; c < HR; ++c) sy1[256 * c] = x[0][c];
            __syncthreads();                                            // buf is refilled by the second sequence
        }
    }
    const cplx xpole = s_pole;
#pragma unroll
    for (int c = 0; c < HR; ++c) {
        const int t = threadIdx.x + 256 * c;
        if (t < Lm) {
            const cplx y2 = x[0][c], y1 = sy1[256 * c];
            const double dl = R.delta[t], ds = R.dsum[t], vv = vp[t];
            cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
            if (t & 1) h = cscale(h, -1.0);
            h.x += fma(ds, xs[c].x, vv * xpole.x);
            h.y += fma(ds, xs[c].y, vv * xpole.y);
            colT[t] = h;
        } else if (t == Lm) {
            cplx acc = cmake(0.0, 0.0);
            for (int w = 0; w < 8; ++w) acc = cadd(acc, s_part[w]);
            colT[t] = acc;
        }
    }
    __syncthreads();  // buf, s_part, s_pole are reused by the next column
    }
}

// a2 at Toeplitz length 256 (grids with 65 <= L_j <= 128: the two top angular scales of BASELINE config 5, over all
// stacked shells).  A sequence is one half-warp's 256-point problem, so nothing crosses a warp: warp = column, its two
// half-warps carry u1 = a x and u2 = delta a x; lane l holds the ring values x_t, t = l + 16 k (k < 8), feeds the
// radix-16 pass straight from registers (upper half zero) and gets y(t) back from the last inverse pass -- no pass over
// stride 256, no block barrier, and the partner spectrum U(-k) of the Hankel term lives in the same half-warp.
__global__ void __launch_bounds__(256, 2) reweight16s_kernel(const cplx *__restrict__ F, cplx *__restrict__ Ft, RwArgs A,
                                                            RwTab R, int ncolumns)
{
    extern __shared__ cplx buf[];
    const int L = R.L, Lm = L - 1;
    const int lane = threadIdx.x & 31, l = lane & 15, half = lane >> 4, warp = threadIdx.x >> 5;
    const int colid = blockIdx.x * 8 + warp;
    const bool has = colid < ncolumns;
    const int mi = colid % A.Md, q = (colid / A.Md) % A.nn, b = colid / (A.Md * A.nn);
    const int m = A.isReal ? mi : mi - (L - 1);
    const int nv = has ? A.n_val[q] : 0, row = has ? A.n_row[q] : 0;
    const int par = ((m + nv) & 1) ? 1 : 0;  // 0: sigma = +1, 1: sigma = -1
    const cplx *col = F + ((size_t)(has ? b : 0) * A.nrows + row) * (size_t)L * A.Md + (has ? mi : 0);
    cplx *colT = Ft + (((size_t)(has ? b : 0) * A.nrows + row) * A.Md + (has ? mi : 0)) * (size_t)L;
    const double *rp = R.rpole + par * L, *vp = R.vpole + par * L;
    double s, c;
    sincospi(-2.0 * (double)l / 256.0, &s, &c);
    const cplx w2 = cmake(c, s);

    cplx xs[8];
    cplx dot = cmake(0.0, 0.0), xpole = cmake(0.0, 0.0);
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int t = l + 16 * k;
        cplx xv = cmake(0.0, 0.0);
        if (t < L && has) {
            xv = col[(size_t)t * A.Md];
            const double r = rp[t];
            dot.x = fma(r, xv.x, dot.x);
            dot.y = fma(r, xv.y, dot.y);
        }
        xs[k] = xv;
        if (t == Lm) xpole = xv;
        cplx u = cmake(0.0, 0.0);
        if (t < Lm) {
            u = (t & 1) ? cscale(xv, -1.0) : xv;
            if (half) u = cscale(u, R.delta[t]);
        }
        v[k] = u;
    }
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) {  // over the 16 lanes of the half-warp (both halves hold the same column)
        dot.x += __shfl_xor_sync(0xffffffffu, dot.x, o);
        dot.y += __shfl_xor_sync(0xffffffffu, dot.y, o);
        xpole.x += __shfl_xor_sync(0xffffffffu, xpole.x, o);
        xpole.y += __shfl_xor_sync(0xffffffffu, xpole.y, o);
    }
    cplx *seq = buf + F16_PAD((threadIdx.x >> 4) * 256);      // this half-warp's 256 elements (272 slots)
    {   // radix-16 pass over stride 16 from registers
        bfly16<false, true, false>(v);
        twiddle_apply<16, false>(v, w2);
        cplx *bq = seq + l;
#pragma unroll
        for (int k = 0; k < 16; ++k) bq[17 * k] = v[k];
    }
    __syncwarp();
    {   // innermost forward pass on 16 contiguous elements
        cplx *bq = seq + 17 * l;
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = bq[k];
        bfly16<false>(v);
#pragma unroll
        for (int k = 0; k < 16; ++k) bq[k] = v[k];
    }
    __syncwarp();
    {   // Y(p) = That(p) U(p) -/+ sigma Ghat(p) U(p'), p = 16 j2 + j3 <-> k = j2 + 16 j3; p' = (16 - j2) % 16 * 16 + ...
        const int j2 = l, j2p = (16 - j2) & 15;
        const cplx *prt = seq + 17 * j2p;
        const cplx *tg = R.TG16 + j2;                             // [2][256] in the storage order F16_TPOS
        double sg = par ? -1.0 : 1.0;
        if (!half) sg = -sg;                                      // u1: T - sigma H, u2: T + sigma H
#pragma unroll
        for (int j3 = 0; j3 < 16; ++j3) {
            const cplx un = prt[j2 ? 15 - j3 : (16 - j3) & 15];
            const cplx th = __ldg(&tg[16 * j3]), gh = cscale(__ldg(&tg[256 + 16 * j3]), sg);
            v[j3] = cadd(cmul(th, v[j3]), cmul(gh, un));
        }
        __syncwarp();                                             // every partner value has been read
        bfly16<true>(v);
        cplx *bq = seq + 17 * l;
#pragma unroll
        for (int k = 0; k < 16; ++k) bq[k] = v[k];
    }
    __syncwarp();
    {   // inverse radix-16 pass over stride 16; only y(t), t = l + 16 k < 128, is formed
        const cplx *bq = seq + l;
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = bq[17 * k];
        twiddle_apply<16, true>(v, w2);
        bfly16<true, false, true>(v);
    }
    // half 0 holds y1 = (T - sigma H) u1, half 1 holds y2 = (T + sigma H) u2: half 0 finishes k < 4, half 1 k >= 4
    cplx other[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const cplx snd = half ? v[k] : v[k + 4];
        other[k].x = __shfl_xor_sync(0xffffffffu, snd.x, 16);
        other[k].y = __shfl_xor_sync(0xffffffffu, snd.y, 16);
    }
    if (!has) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int kk = half ? k + 4 : k;
        const int t = l + 16 * kk;
        const cplx mine = half ? v[k + 4] : v[k];
        const cplx y1 = half ? other[k] : mine, y2 = half ? mine : other[k];
        const cplx xv = half ? xs[k + 4] : xs[k];
        if (t < Lm) {
            const double dl = R.delta[t], ds = R.dsum[t], vv = vp[t];
            cplx h = cmake(fma(dl, y1.x, -y2.x), fma(dl, y1.y, -y2.y));
            if (t & 1) h = cscale(h, -1.0);
            h.x += fma(ds, xv.x, vv * xpole.x);
            h.y += fma(ds, xv.y, vv * xpole.y);
            colT[t] = h;
        } else if (t == Lm) {
            colT[t] = dot;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a8 for complex signals (sphere configs 2, the ball), NN <= 3 active rows n, Bluestein lengths 256 ... 1024 (R1 = 1, 2,
// 4): a round holds the NN rows of RB = NB / NN rings, so the gamma DFT of a ring (Eq. 48) is done in registers
// right after / before the transforms -- nothing is parked.  F[b][row][t][m + L-1], W[b][g][t][a] complex.
// ---------------------------------------------------------------------------------------------------------------
template <int R1, int NN>
__global__ void __launch_bounds__(256, 2) so3_inv_c16_kernel(const cplx *__restrict__ F, cplx *__restrict__ W,
                                                            size_t sig_stride, So3Args A, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 >= 2 ? R1 / 2 : 1, RB = NB / NN;
    static_assert(RB >= 1, "more rows than sequences in a round");
    extern __shared__ cplx buf[];
    __shared__ cplx gph[NN * 64];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L, ng = 2 * A.N - 1;
    const cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * n;
    cplx *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    for (int e = threadIdx.x; e < NN * ng; e += 256) gph[e] = cis_2pi(A.n_val[e / ng] * (e % ng), ng);
    cplx x[NB][R1];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int r = q / NN, i = q % NN;
        const int t = blockIdx.x * RB + r;
        const bool on = r < RB && t < L;
        const cplx *Fp = Fb + ((size_t)A.n_row[i] * L + (on ? t : 0)) * n + (L - 1);
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int k = threadIdx.x + 256 * c;
            const int kk = (k < n && on) ? k : 0;
            const cplx v = Fp[kk < L ? kk : kk - n], ch = __ldg(&T.chirp[kk]);
            x[q][c] = (k < n && on) ? cmulc(v, ch) : cmake(0.0, 0.0);
        }
    }
    __syncthreads();  // gph
    f16_convolve_half<R1>(buf, x, T.bhat16_p, tw);
#pragma unroll
    for (int r = 0; r < RB; ++r) {
        const int t = blockIdx.x * RB + r;
        if (t >= L) continue;
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int a = threadIdx.x + 256 * c;
            if (a >= n) continue;
            const cplx ch = __ldg(&T.chirp[a]);
            cplx v[NN];
#pragma unroll
            for (int i = 0; i < NN; ++i) v[i] = cmulc(x[r * NN + i][c], ch);
            cplx *Wr = Wb + (size_t)t * n + a;
            for (int g = 0; g < ng; ++g) {
                cplx o = cmul(gph[g], v[0]);
#pragma unroll
                for (int i = 1; i < NN; ++i) o = cadd(o, cmul(gph[i * ng + g], v[i]));
                Wr[(size_t)g * plane] = o;
            }
        }
    }
}

template <int R1, int NN>
__global__ void __launch_bounds__(256, 2) so3_fwd_c16_kernel(const cplx *__restrict__ W, cplx *__restrict__ F,
                                                            size_t sig_stride, So3Args A, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 >= 2 ? R1 / 2 : 1, RB = NB / NN;
    static_assert(RB >= 1, "more rows than sequences in a round");
    extern __shared__ cplx buf[];
    __shared__ cplx gph[NN * 64];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L, ng = 2 * A.N - 1;
    const double inv_ng = 1.0 / (double)ng, inv_n = 1.0 / (double)n;
    cplx *Fb = F + (size_t)blockIdx.y * A.nrows * L * n;
    const cplx *Wb = W + so3_base(A, blockIdx.y, sig_stride);
    const size_t plane = (size_t)L * n;
    for (int e = threadIdx.x; e < NN * ng; e += 256) gph[e] = cis_2pi(-A.n_val[e / ng] * (e % ng), ng);
    __syncthreads();
    cplx x[NB][R1];
#pragma unroll
    for (int q = 0; q < NB; ++q)
#pragma unroll
        for (int c = 0; c < HR; ++c) x[q][c] = cmake(0.0, 0.0);
#pragma unroll
    for (int r = 0; r < RB; ++r) {
        const int t = blockIdx.x * RB + r;
        if (t >= L) continue;
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int a = threadIdx.x + 256 * c;
            if (a >= n) continue;
            const cplx *Wr = Wb + (size_t)t * n + a;
            cplx y[NN];
#pragma unroll
            for (int i = 0; i < NN; ++i) y[i] = cmake(0.0, 0.0);
            for (int g = 0; g < ng; ++g) {
                const cplx wv = Wr[(size_t)g * plane];
#pragma unroll
                for (int i = 0; i < NN; ++i) y[i] = cadd(y[i], cmul(gph[i * ng + g], wv));
            }
            const cplx ch = cscale(__ldg(&T.chirp[a]), inv_ng);
#pragma unroll
            for (int i = 0; i < NN; ++i) x[r * NN + i][c] = cmul(y[i], ch);
        }
    }
    f16_convolve_half<R1>(buf, x, T.bhat16_m, tw);
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int r = q / NN, i = q % NN;
        const int t = blockIdx.x * RB + r;
        if (r >= RB || t >= L) continue;
        cplx *Fp = Fb + ((size_t)A.n_row[i] * L + t) * n + (L - 1);
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int k = threadIdx.x + 256 * c;
            if (k >= n) continue;
            Fp[k < L ? k : k - n] = cscale(cmul(x[q][c], __ldg(&T.chirp[k])), inv_n);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a1 ring FFTs (Eqs. 2-3) on the radix-16 core: a block works on NB sequences, each a pair of real rings (one
// complex DFT, split by Hermitian symmetry) or one complex ring.  Layouts as in ring_fwd_kernel / ring_inv_kernel.
// ---------------------------------------------------------------------------------------------------------------
template <int R1, bool REAL>
__global__ void __launch_bounds__(256, 2) ring_fwd16_kernel(const void *__restrict__ in, cplx *__restrict__ out, int nrows,
                                                           size_t sig_stride, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 >= 2 ? R1 / 2 : 1, M = R1 * 256;
    extern __shared__ cplx buf[];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L;
    const double inv_n = 1.0 / (double)n;
    cplx x[NB][R1];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int s = blockIdx.x * NB + q;
        const int r0 = REAL ? 2 * s : s, r1 = r0 + 1;
        const bool on0 = r0 < nrows, on1 = REAL && r1 < nrows;
        const size_t o0 = (size_t)((on0 ? r0 : 0) / L) * sig_stride + (size_t)((on0 ? r0 : 0) % L) * n;
        const size_t o1 = (size_t)((on1 ? r1 : 0) / L) * sig_stride + (size_t)((on1 ? r1 : 0) % L) * n;
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int pp = threadIdx.x + 256 * c;
            const int pk = (pp < n && on0) ? pp : 0;
            cplx v;
            if (REAL) {
                const double a = ((const double *)in)[o0 + pk], b = ((const double *)in)[o1 + pk];
                v = cmake(a, on1 ? b : 0.0);
            } else {
                v = ((const cplx *)in)[o0 + pk];
            }
            x[q][c] = (pp < n && on0) ? cmul(v, __ldg(&T.chirp[pk])) : cmake(0.0, 0.0);
        }
    }
    f16_convolve_half<R1>(buf, x, T.bhat16_m, tw);
    if (REAL) {
#pragma unroll
        for (int q = 0; q < NB; ++q)
#pragma unroll
            for (int c = 0; c < HR; ++c) {
                const int k = threadIdx.x + 256 * c;
                buf[F16_PAD(q * M + k)] = cmul(x[q][c], __ldg(&T.chirp[k < n ? k : 0]));
            }
        __syncthreads();
#pragma unroll 1
        for (int q = 0; q < NB; ++q) {
            const int r0 = 2 * (blockIdx.x * NB + q), r1 = r0 + 1;
            if (r0 >= nrows) continue;
            for (int m = threadIdx.x; m < L; m += 256) {
                const cplx a = buf[F16_PAD(q * M + m)], b = cconj(buf[F16_PAD(q * M + (m == 0 ? 0 : n - m))]);
                const cplx sm = cadd(a, b), d = csub(a, b);
                out[(size_t)r0 * L + m] = cscale(sm, 0.5 * inv_n);
                if (r1 < nrows) out[(size_t)r1 * L + m] = cmake(0.5 * inv_n * d.y, -0.5 * inv_n * d.x);
            }
        }
    } else {
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int r0 = blockIdx.x * NB + q;
            if (r0 >= nrows) continue;
#pragma unroll
            for (int c = 0; c < HR; ++c) {
                const int k = threadIdx.x + 256 * c;
                if (k >= n) continue;
                out[(size_t)r0 * n + (k < L ? k : k - n) + (L - 1)] = cscale(cmul(x[q][c], __ldg(&T.chirp[k])), inv_n);
            }
        }
    }
}

template <int R1, bool REAL>
__global__ void __launch_bounds__(256, 2) ring_inv16_kernel(const cplx *__restrict__ in, void *__restrict__ out, int nrows,
                                                           size_t sig_stride, FftTab T)
{
    constexpr int NB = 16 / R1, HR = R1 >= 2 ? R1 / 2 : 1;
    extern __shared__ cplx buf[];
    const F16Tw tw = f16_twiddles<R1>();
    const int n = T.n, L = T.L;
    cplx x[NB][R1];
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int s = blockIdx.x * NB + q;
        const int r0 = REAL ? 2 * s : s, r1 = r0 + 1;
        const bool on0 = r0 < nrows, on1 = REAL && r1 < nrows;
        const cplx *X0 = in + (size_t)(on0 ? r0 : 0) * (REAL ? L : n), *X1 = in + (size_t)(on1 ? r1 : 0) * L;
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int k = threadIdx.x + 256 * c;
            const int kk = (k < n && on0) ? k : 0;
            cplx v;
            if (REAL) {
                const int m = kk < L ? kk : n - kk;
                cplx a = X0[m], b = X1[m];
                if (!on1) b = cmake(0.0, 0.0);
                if (kk >= L) {
                    a = cconj(a);
                    b = cconj(b);
                }
                v = cmake(a.x - b.y, a.y + b.x);  // Z_k = A_k + i B_k
            } else {
                v = X0[(kk < L ? kk : kk - n) + (L - 1)];
            }
            x[q][c] = (k < n && on0) ? cmulc(v, __ldg(&T.chirp[kk])) : cmake(0.0, 0.0);
        }
    }
    f16_convolve_half<R1>(buf, x, T.bhat16_p, tw);
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int s = blockIdx.x * NB + q;
        const int r0 = REAL ? 2 * s : s, r1 = r0 + 1;
        if (r0 >= nrows) continue;
        const size_t o0 = (size_t)(r0 / L) * sig_stride + (size_t)(r0 % L) * n;
        const size_t o1 = (size_t)((r1 < nrows ? r1 : r0) / L) * sig_stride + (size_t)((r1 < nrows ? r1 : r0) % L) * n;
#pragma unroll
        for (int c = 0; c < HR; ++c) {
            const int pp = threadIdx.x + 256 * c;
            if (pp >= n) continue;
            const cplx z = cmulc(x[q][c], __ldg(&T.chirp[pp]));
            if (REAL) {
                ((double *)out)[o0 + pp] = z.x;
                if (r1 < nrows) ((double *)out)[o1 + pp] = z.y;
            } else {
                ((cplx *)out)[o0 + pp] = z;
            }
        }
    }
}

// ---- plan time: kernel spectra in the core's own order --------------------------------------------------------------

template <int R1>
__global__ void __launch_bounds__(256) fft16_forward_kernel(cplx *data)
{
    extern __shared__ cplx buf[];
    const F16Tw tw = f16_twiddles<R1>();
    f16_forward_full<R1, true>(buf, data, data, tw);
}

// natural-order Bluestein kernels: kind 0: b[d mod M] = exp(+i pi d^2/n)/M, |d| < n (forward DFT); kind 1: conjugate
__global__ void chirp_wrap_kernel(cplx *khat, int kind, int n, int M)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    int d = e < n ? e : (e > M - n ? e - M : M);  // M: outside the support
    cplx v = cmake(0.0, 0.0);
    if (d != M) {
        const long long r = ((long long)d * d) % (2LL * n);
        double s, c;
        sincospi((double)r / (double)n, &s, &c);
        v = cscale(cmake(c, kind == 0 ? s : -s), 1.0 / (double)M);
    }
    khat[e] = v;
}

}  // namespace

int launch_fft16_forward(cplx *data, int M, cudaStream_t st)
{
    const size_t sm = (size_t)F16_BUF * sizeof(cplx);
    int rc;
    if (M == 4096) {
        if ((rc = set_smem(fft16_forward_kernel<16>, sm))) return rc;
        S2W_LAUNCH(fft16_forward_kernel<16>, 1, 256, sm, st, data);
    } else if (M == 2048) {
        if ((rc = set_smem(fft16_forward_kernel<8>, sm))) return rc;
        S2W_LAUNCH(fft16_forward_kernel<8>, 1, 256, sm, st, data);
    } else if (M == 1024) {
        if ((rc = set_smem(fft16_forward_kernel<4>, sm))) return rc;
        S2W_LAUNCH(fft16_forward_kernel<4>, 1, 256, sm, st, data);
    } else if (M == 512) {
        if ((rc = set_smem(fft16_forward_kernel<2>, sm))) return rc;
        S2W_LAUNCH(fft16_forward_kernel<2>, 1, 256, sm, st, data);
    } else if (M == 256) {
        if ((rc = set_smem(fft16_forward_kernel<1>, sm))) return rc;
        S2W_LAUNCH(fft16_forward_kernel<1>, 1, 256, sm, st, data);
    } else {
        set_error("launch_fft16_forward: unsupported length");
        return S2W_EINVAL;
    }
    return S2W_OK;
}

int launch_fft16_spectrum(cplx *khat, int kind, int n, int M, cudaStream_t st)
{
    S2W_LAUNCH(chirp_wrap_kernel, (M + 255) / 256, 256, 0, st, khat, kind, n, M);
    return launch_fft16_forward(khat, M, st);
}

template <int R1>
static int so3_pair16_t(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch,
                        const FftTab &T, cudaStream_t st)
{
    constexpr int NB = 16 / R1;
    const size_t sm = (size_t)F16_BUF * sizeof(cplx);
    const int npairs = (T.L + 1) / 2;
    dim3 grid((npairs + NB - 1) / NB, batch);
    int rc;
    if (fwd) {
        if ((rc = set_smem(so3_fwd_pair16_kernel<R1>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, so3_fwd_pair16_kernel<R1>, grid, 256, sm, st, (const double *)in, (cplx *)out,
                     sig_stride, A, T);
    } else {
        if ((rc = set_smem(so3_inv_pair16_kernel<R1>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, so3_inv_pair16_kernel<R1>, grid, 256, sm, st, (const cplx *)in, (double *)out,
                     sig_stride, A, T);
    }
    return S2W_OK;
}

// real signals, 2N-1 <= 9, Bluestein length 1024 / 2048 / 4096 (the caller checks)
int launch_so3_pair16(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch,
                      const FftTab &T, cudaStream_t st)
{
    if (T.M == 4096) return so3_pair16_t<16>(fwd, in, out, sig_stride, A, batch, T, st);
    if (T.M == 2048) return so3_pair16_t<8>(fwd, in, out, sig_stride, A, batch, T, st);
    return so3_pair16_t<4>(fwd, in, out, sig_stride, A, batch, T, st);
}

template <int R1, int NN>
static int so3_c16_t(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                     cudaStream_t st)
{
    constexpr int RB = (16 / R1) / NN;
    const size_t sm = (size_t)F16_BUF * sizeof(cplx);
    dim3 grid((T.L + RB - 1) / RB, batch);
    int rc;
    if (fwd) {
        if ((rc = set_smem(so3_fwd_c16_kernel<R1, NN>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_fwd_c16_kernel<R1, NN>), grid, 256, sm, st, (const cplx *)in, (cplx *)out,
                     sig_stride, A, T);
    } else {
        if ((rc = set_smem(so3_inv_c16_kernel<R1, NN>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_SO3_FFT, (so3_inv_c16_kernel<R1, NN>), grid, 256, sm, st, (const cplx *)in, (cplx *)out,
                     sig_stride, A, T);
    }
    return S2W_OK;
}

bool so3_c16_supported(const So3Args &A, const FftTab &T)
{
    return T.bhat16_m && (T.M == 256 || T.M == 512 || T.M == 1024) && A.nn >= 1 && A.nn <= 3;
}

// complex signals; the caller checks so3_c16_supported
int launch_so3_c16(bool fwd, const void *in, void *out, size_t sig_stride, const So3Args &A, int batch, const FftTab &T,
                   cudaStream_t st)
{
#define S2W_C16_CASE(MM, RR)                                                                          \
    if (T.M == MM) {                                                                                  \
        if (A.nn == 1) return so3_c16_t<RR, 1>(fwd, in, out, sig_stride, A, batch, T, st);            \
        if (A.nn == 2) return so3_c16_t<RR, 2>(fwd, in, out, sig_stride, A, batch, T, st);            \
        return so3_c16_t<RR, 3>(fwd, in, out, sig_stride, A, batch, T, st);                           \
    }
    S2W_C16_CASE(256, 1)
    S2W_C16_CASE(512, 2)
    S2W_C16_CASE(1024, 4)
#undef S2W_C16_CASE
    set_error("launch_so3_c16: unsupported length");
    return S2W_EINVAL;
}

template <int R1, bool REAL>
static int ring16_t(bool fwd, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T, cudaStream_t st)
{
    constexpr int NB = 16 / R1;
    const size_t sm = (size_t)F16_BUF * sizeof(cplx);
    const int nseq = REAL ? (nrows + 1) / 2 : nrows;
    const int grid = (nseq + NB - 1) / NB;
    int rc;
    if (fwd) {
        if ((rc = set_smem(ring_fwd16_kernel<R1, REAL>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, (ring_fwd16_kernel<R1, REAL>), grid, 256, sm, st, in, (cplx *)out, nrows, sig_stride, T);
    } else {
        if ((rc = set_smem(ring_inv16_kernel<R1, REAL>, sm))) return rc;
        S2W_LAUNCH_C(S2W_K_RING_FFT, (ring_inv16_kernel<R1, REAL>), grid, 256, sm, st, (const cplx *)in, out, nrows,
                     sig_stride, T);
    }
    return S2W_OK;
}

// a1 on the radix-16 core; the caller checks T.bhat16_m and f16_supported(T.M)
int launch_ring16(bool fwd, bool real, const void *in, void *out, int nrows, size_t sig_stride, const FftTab &T,
                  cudaStream_t st)
{
#define S2W_R16_CASE(MM, RR)                                                                   \
    if (T.M == MM)                                                                             \
        return real ? ring16_t<RR, true>(fwd, in, out, nrows, sig_stride, T, st)               \
                    : ring16_t<RR, false>(fwd, in, out, nrows, sig_stride, T, st);
    S2W_R16_CASE(4096, 16)
    S2W_R16_CASE(2048, 8)
    S2W_R16_CASE(1024, 4)
    S2W_R16_CASE(512, 2)
    S2W_R16_CASE(256, 1)
#undef S2W_R16_CASE
    set_error("launch_ring16: unsupported length");
    return S2W_EINVAL;
}

// Toeplitz length 2048 ... 256 (the caller checks)
template <int R1>
static int reweight16_t(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const RwTab &R, cudaStream_t st)
{
    constexpr int NC = 8 / R1;
    const int ncol = A.Md * A.nn * batch;
    const size_t sm = (size_t)F16_BUF * sizeof(cplx);
    int rc;
    // two blocks per SM, resident for the whole launch (S2W_RW_PERSIST = blocks, 0: one block per column group).  Measured
    // at C3: the class alone takes the same time (2.34 ms), but the step drops from 13.66 to 13.50 ms -- the launch no
    // longer floods the SMs that the other lanes' kernels are running on
    static const int persist = [] {
        const char *e = getenv("S2W_RW_PERSIST");
        if (e) return atoi(e);
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        return 2 * sms;
    }();
    const int ngroups = (ncol + NC - 1) / NC;
    if (persist > 0 && ngroups > persist) {  // persistent blocks with a cp.async staging area for the next column group
        const size_t smp = (size_t)(F16_BUF + 1024) * sizeof(cplx);
        if ((rc = set_smem(reweight16p_kernel<R1>, smp))) return rc;
        S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight16p_kernel<R1>, persist, 256, smp, st, F, Ft, A, R, ncol);
        return S2W_OK;
    }
    if ((rc = set_smem(reweight16_kernel<R1>, sm))) return rc;
    S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight16_kernel<R1>, ngroups, 256, sm, st, F, Ft, A, R, ncol);
    return S2W_OK;
}

int launch_reweight16(const cplx *F, cplx *Ft, const RwArgs &A, int batch, const RwTab &R, cudaStream_t st)
{
    switch (R.fft.M) {
    case 4096: {
        const int ncol = A.Md * A.nn * batch;
        const size_t sm = (size_t)(F16_BUF + 2048) * sizeof(cplx);
        int rc = set_smem(reweight16w_kernel, sm);
        if (rc) return rc;
        static const int persist_w = [] {
            const char *e = getenv("S2W_RW_PERSIST");
            if (e) return atoi(e);
            int dev = 0, sms = 148;
            if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            return 2 * sms;
        }();
        const int nblk = (persist_w > 0 && ncol > persist_w) ? persist_w : ncol;
        S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight16w_kernel, nblk, 256, sm, st, F, Ft, A, R, ncol);
        return S2W_OK;
    }
    case 2048: return reweight16_t<8>(F, Ft, A, batch, R, st);
    case 1024: return reweight16_t<4>(F, Ft, A, batch, R, st);
    case 512: return reweight16_t<2>(F, Ft, A, batch, R, st);
    case 256: {
        const int ncol = A.Md * A.nn * batch;
        const size_t sm = (size_t)F16_BUF * sizeof(cplx);
        int rc = set_smem(reweight16s_kernel, sm);
        if (rc) return rc;
        S2W_LAUNCH_C(S2W_K_REWEIGHT, reweight16s_kernel, (ncol + 7) / 8, 256, sm, st, F, Ft, A, R, ncol);
        return S2W_OK;
    }
    }
    set_error("launch_reweight16: unsupported length");
    return S2W_EINVAL;
}

}  // namespace s2w
