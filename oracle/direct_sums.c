/* oracle/direct_sums.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, direct-summation CPU reference for the heavy inner sums of the
 * scale-discretised wavelet transform of arXiv:2402.01282 (PAPER.md = "P:").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant with paper_2402_01282_b200/csrc (the CUDA path).
 *
 * REAL is chosen at compile time: `long double` (parity reference, 64-bit
 * mantissa) or `double` (the timed CPU baseline).  Complex numbers are stored
 * as interleaved (re, im) pairs of REAL.
 *
 * Every function is the definition written out: a three-term recursion that
 * generates d^l_{mn}(beta) one l at a time, and literal sums over l, t, k, p.
 * There is no blocking, fusion or re-ordering beyond the loop nests shown.
 *
 * Conventions (readings R2, R3, R6):
 *   d^l_{mn}(beta) = <l m| exp(-i beta J_y) |l n>   so d^1_{10} = -sin(beta)/sqrt 2
 *   D^l_{mn}(alpha,beta,gamma) = exp(-i m alpha) d^l_{mn}(beta) exp(-i n gamma)   (Eq. 47)
 *   MW sampling: theta_t = pi (2t+1)/(2L-1), t = 0..L-1; phi_p = 2 pi p/(2L-1)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef REAL
#define REAL long double
#endif

#if defined(ORC_DOUBLE)
#define R_SQRT sqrt
#define R_COS cos
#define R_SIN sin
#define R_ATAN atan
#define R_FABS fabs
#else
#define R_SQRT sqrtl
#define R_COS cosl
#define R_SIN sinl
#define R_ATAN atanl
#define R_FABS fabsl
#endif

static REAL orc_pi(void) { return (REAL)4 * R_ATAN((REAL)1); }

int orc_sizeof_real(void) { return (int)sizeof(REAL); }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* cos and sin of pi * num / den for integers (exact argument reduction). */
static void orc_cis_pi_frac(long long num, long long den, REAL *c, REAL *s)
{
    long long r = num % (2 * den);
    if (r < 0) r += 2 * den;
    REAL a = orc_pi() * (REAL)r / (REAL)den;
    *c = R_COS(a);
    *s = R_SIN(a);
}

/* ------------------------------------------------------------------------
 * Seed of the l-recursion (Varshalovich et al. cited P:434):
 *   S(l0, q) = d^{l0}_{l0,q}(beta) = sqrt((2 l0)! / ((l0+q)! (l0-q)!))
 *                                     cos^{l0+q}(beta/2) (-sin(beta/2))^{l0-q}
 * evaluated as an interleaved product so that no partial product overflows:
 *   binom(a+b, b) = prod_{i=1..b} (a+i)/i  with a = l0+q, b = l0-q.
 * ---------------------------------------------------------------------- */
static REAL orc_seed(int l0, int q, REAL beta)
{
    int a = l0 + q, b = l0 - q;
    REAL c = R_COS(beta / 2), s = R_SIN(beta / 2);
    REAL v = 1;
    int top = a > b ? a : b;
    for (int i = 1; i <= top; ++i) {
        if (i <= b) v *= R_SQRT((REAL)(a + i) / (REAL)i) * (-s);
        if (i <= a) v *= c;
    }
    return v;
}

/* d^l_{mn}(beta) for l = 0 .. L-1 written to d[0..L-1]; zero for l < max(|m|,|n|).
 * Seed at l0 = max(|m|,|n|) from S(l0,.) and the symmetries
 *   d^l_{mn} = (-1)^{m-n} d^l_{nm} = d^l_{-n,-m},
 * then the textbook three-term recursion in l:
 *   d^{l+1} = (l+1)(2l+1)/sqrt(((l+1)^2-m^2)((l+1)^2-n^2))
 *             * [ (cos(beta) - m n/(l(l+1))) d^l - sqrt((l^2-m^2)(l^2-n^2))/(l(2l+1)) d^{l-1} ].
 * For l0 = 0: P_0 = 1, P_1 = cos(beta). */
void orc_wigner_d(int L, int m, int n, REAL beta, REAL *d)
{
    int am = m < 0 ? -m : m, an = n < 0 ? -n : n;
    int l0 = am > an ? am : an;
    for (int l = 0; l < L; ++l) d[l] = 0;
    if (l0 >= L) return;
    REAL seed;
    if (m == l0)
        seed = orc_seed(l0, n, beta);
    else if (m == -l0)
        seed = (((l0 + n) & 1) ? -1 : 1) * orc_seed(l0, -n, beta);
    else if (n == l0)
        seed = (((l0 - m) & 1) ? -1 : 1) * orc_seed(l0, m, beta);
    else /* n == -l0 */
        seed = orc_seed(l0, -m, beta);
    d[l0] = seed;
    REAL x = R_COS(beta);
    REAL dm1 = 0, d0 = seed;
    for (int l = l0; l + 1 < L; ++l) {
        REAL d1;
        if (l == 0) {
            d1 = x * d0; /* P_1 = cos(beta) P_0 */
        } else {
            REAL lp = (REAL)(l + 1);
            REAL A = lp * (REAL)(2 * l + 1) /
                     R_SQRT((lp * lp - (REAL)m * m) * (lp * lp - (REAL)n * n));
            REAL B = (REAL)m * (REAL)n / ((REAL)l * lp);
            REAL C = R_SQRT(((REAL)l * l - (REAL)m * m) * ((REAL)l * l - (REAL)n * n)) /
                     ((REAL)l * (REAL)(2 * l + 1));
            d1 = A * ((x - B) * d0 - C * dm1);
        }
        d[l + 1] = d1;
        dm1 = d0;
        d0 = d1;
    }
}

/* Same, with beta passed by pointer (ctypes cannot pass a long double by value exactly). */
void orc_wigner_d_p(int L, int m, int n, const REAL *beta, REAL *d) { orc_wigner_d(L, m, n, *beta, d); }

/* MW colatitudes theta_t = pi (2t+1)/(2L-1), t = 0..L-1. */
void orc_mw_thetas(int L, REAL *theta)
{
    for (int t = 0; t < L; ++t) theta[t] = orc_pi() * (REAL)(2 * t + 1) / (REAL)(2 * L - 1);
}

/* ------------------------------------------------------------------------
 * Inverse beta-contraction (the l-sum of Eq. 3 / Eq. 5):
 *   F[mi][t] = sum_{l=max(|m|,|n|)}^{L-1} d^l_{mn}(beta_t) X[l][mi],   m = mi-(L-1)
 * X: [L][2L-1] complex, F: [2L-1][nbeta] complex.
 * ---------------------------------------------------------------------- */
void orc_dl_inverse(int L, int n, int nbeta, const REAL *beta, const REAL *X, REAL *F)
{
    int M = 2 * L - 1;
#pragma omp parallel
    {
        REAL *d = (REAL *)malloc(sizeof(REAL) * (size_t)L);
#pragma omp for schedule(dynamic, 1)
        for (int mi = 0; mi < M; ++mi) {
            int m = mi - (L - 1);
            for (int t = 0; t < nbeta; ++t) {
                orc_wigner_d(L, m, n, beta[t], d);
                REAL re = 0, im = 0;
                for (int l = 0; l < L; ++l) {
                    re += d[l] * X[2 * ((size_t)l * M + mi)];
                    im += d[l] * X[2 * ((size_t)l * M + mi) + 1];
                }
                F[2 * ((size_t)mi * nbeta + t)] = re;
                F[2 * ((size_t)mi * nbeta + t) + 1] = im;
            }
        }
        free(d);
    }
}

/* ------------------------------------------------------------------------
 * Forward beta-contraction (the beta-projection of Eq. 48; a3, a6):
 *   W[l][mi] = sum_{t=0}^{nbeta-1} d^l_{mn}(beta_t) H[mi][t]
 * H: [2L-1][nbeta] complex, W: [L][2L-1] complex (zero for l < max(|m|,|n|)).
 * ---------------------------------------------------------------------- */
void orc_dl_forward(int L, int n, int nbeta, const REAL *beta, const REAL *H, REAL *W)
{
    int M = 2 * L - 1;
#pragma omp parallel
    {
        REAL *d = (REAL *)malloc(sizeof(REAL) * (size_t)L);
#pragma omp for schedule(dynamic, 1)
        for (int mi = 0; mi < M; ++mi) {
            int m = mi - (L - 1);
            for (int l = 0; l < L; ++l) {
                W[2 * ((size_t)l * M + mi)] = 0;
                W[2 * ((size_t)l * M + mi) + 1] = 0;
            }
            for (int t = 0; t < nbeta; ++t) {
                orc_wigner_d(L, m, n, beta[t], d);
                REAL hr = H[2 * ((size_t)mi * nbeta + t)], hi = H[2 * ((size_t)mi * nbeta + t) + 1];
                for (int l = 0; l < L; ++l) {
                    W[2 * ((size_t)l * M + mi)] += d[l] * hr;
                    W[2 * ((size_t)l * M + mi) + 1] += d[l] * hi;
                }
            }
        }
        free(d);
    }
}

/* ------------------------------------------------------------------------
 * MW theta-quadrature reweighting (reading R3).
 * For one column F(theta_t), t = 0..L-1, of parity sigma = (-1)^{m+n}:
 *  (ii)  extend to t = L..2L-2:  F(theta_{2L-2-t}) = sigma F(theta_t)
 *  (iii) Fh(k) = 1/(2L-1) sum_{t=0}^{2L-2} F(theta_t) exp(-i k theta_t),  |k| <= L-1
 *  (iv)  G(k') = sum_k Fh(k) w(k+k'),  w(q) = int_0^pi exp(i q theta) sin(theta) dtheta
 *               = 2/(1-q^2) (q even), +-i pi/2 (q = +-1), 0 (other odd q)
 *  (v)   g(theta_t) = sum_{k'} G(k') exp(-i k' theta_t),  t = 0..2L-2
 *  (vi)  h(theta_t) = g(theta_t) + sigma g(theta_{2L-2-t}) (t < L-1),  h(theta_{L-1}) = g(theta_{L-1})
 * so that  int_0^pi F(theta) d(theta) sin(theta) dtheta = 1/(2L-1) sum_{t<L} d(theta_t) h(theta_t)
 * for every trigonometric polynomial d of degree <= L-1 with d(-theta) = sigma d(theta).
 * Fin, Hout: [ncols][L] complex; sigma[ncols] = +1 or -1.
 * ---------------------------------------------------------------------- */
void orc_mw_reweight(int L, int ncols, const int *sigma, const REAL *Fin, REAL *Hout)
{
    int n = 2 * L - 1;
    /* e[(k+L-1)*n + t] = exp(-i k theta_t) */
    REAL *ec = (REAL *)malloc(sizeof(REAL) * (size_t)n * n);
    REAL *es = (REAL *)malloc(sizeof(REAL) * (size_t)n * n);
    for (int k = -(L - 1); k <= L - 1; ++k)
        for (int t = 0; t < n; ++t) {
            REAL c, s;
            orc_cis_pi_frac((long long)k * (2 * t + 1), n, &c, &s);
            ec[(size_t)(k + L - 1) * n + t] = c;
            es[(size_t)(k + L - 1) * n + t] = -s;
        }
#pragma omp parallel
    {
        REAL *ext = (REAL *)malloc(sizeof(REAL) * 2 * (size_t)n);
        REAL *Fh = (REAL *)malloc(sizeof(REAL) * 2 * (size_t)n);
        REAL *G = (REAL *)malloc(sizeof(REAL) * 2 * (size_t)n);
        REAL *g = (REAL *)malloc(sizeof(REAL) * 2 * (size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int c = 0; c < ncols; ++c) {
            const REAL *F = Fin + 2 * (size_t)c * L;
            REAL *H = Hout + 2 * (size_t)c * L;
            REAL sg = (REAL)sigma[c];
            /* (ii) */
            for (int t = 0; t < L; ++t) {
                ext[2 * t] = F[2 * t];
                ext[2 * t + 1] = F[2 * t + 1];
            }
            for (int t = L; t < n; ++t) {
                ext[2 * t] = sg * F[2 * (2 * L - 2 - t)];
                ext[2 * t + 1] = sg * F[2 * (2 * L - 2 - t) + 1];
            }
            /* (iii) */
            for (int ki = 0; ki < n; ++ki) {
                REAL re = 0, im = 0;
                for (int t = 0; t < n; ++t) {
                    REAL cr = ec[(size_t)ki * n + t], ci = es[(size_t)ki * n + t];
                    re += ext[2 * t] * cr - ext[2 * t + 1] * ci;
                    im += ext[2 * t] * ci + ext[2 * t + 1] * cr;
                }
                Fh[2 * ki] = re / (REAL)n;
                Fh[2 * ki + 1] = im / (REAL)n;
            }
            /* (iv) */
            for (int kpi = 0; kpi < n; ++kpi) {
                int kp = kpi - (L - 1);
                REAL re = 0, im = 0;
                for (int ki = 0; ki < n; ++ki) {
                    int q = ki - (L - 1) + kp;
                    REAL wr = 0, wi = 0;
                    if (q % 2 == 0)
                        wr = (REAL)2 / ((REAL)1 - (REAL)q * (REAL)q);
                    else if (q == 1)
                        wi = orc_pi() / 2;
                    else if (q == -1)
                        wi = -orc_pi() / 2;
                    re += Fh[2 * ki] * wr - Fh[2 * ki + 1] * wi;
                    im += Fh[2 * ki] * wi + Fh[2 * ki + 1] * wr;
                }
                G[2 * kpi] = re;
                G[2 * kpi + 1] = im;
            }
            /* (v) */
            for (int t = 0; t < n; ++t) {
                REAL re = 0, im = 0;
                for (int kpi = 0; kpi < n; ++kpi) {
                    REAL cr = ec[(size_t)kpi * n + t], ci = es[(size_t)kpi * n + t];
                    re += G[2 * kpi] * cr - G[2 * kpi + 1] * ci;
                    im += G[2 * kpi] * ci + G[2 * kpi + 1] * cr;
                }
                g[2 * t] = re;
                g[2 * t + 1] = im;
            }
            /* (vi) */
            for (int t = 0; t < L - 1; ++t) {
                H[2 * t] = g[2 * t] + sg * g[2 * (2 * L - 2 - t)];
                H[2 * t + 1] = g[2 * t + 1] + sg * g[2 * (2 * L - 2 - t) + 1];
            }
            H[2 * (L - 1)] = g[2 * (L - 1)];
            H[2 * (L - 1) + 1] = g[2 * (L - 1) + 1];
        }
        free(ext);
        free(Fh);
        free(G);
        free(g);
    }
    free(ec);
    free(es);
}

/* ------------------------------------------------------------------------
 * Plain DFT along the last axis of [nrows][n] complex data on the equispaced
 * grid x_p = 2 pi p / n:
 *   out[r][ki] = scale * sum_{p=0}^{n-1} in[r][p] exp(sign * i * k * x_p),
 *   k = ki + kmin, ki = 0..nk-1.
 * ---------------------------------------------------------------------- */
void orc_dft_rows(int nrows, int n, int kmin, int nk, int sign, const REAL *scale_p, const REAL *in, REAL *out)
{
    REAL scale = *scale_p; /* scalars cross the ctypes boundary by pointer to keep long double exact */
    REAL *cs = (REAL *)malloc(sizeof(REAL) * 2 * (size_t)n);
    for (int r = 0; r < n; ++r) orc_cis_pi_frac(2LL * r, n, &cs[2 * r], &cs[2 * r + 1]);
#pragma omp parallel for schedule(static)
    for (int row = 0; row < nrows; ++row) {
        const REAL *x = in + 2 * (size_t)row * n;
        REAL *y = out + 2 * (size_t)row * nk;
        for (int ki = 0; ki < nk; ++ki) {
            long long k = (long long)ki + kmin;
            REAL re = 0, im = 0;
            for (int p = 0; p < n; ++p) {
                long long r = (k * p) % n;
                if (r < 0) r += n;
                REAL c = cs[2 * r], s = sign * cs[2 * r + 1];
                re += x[2 * p] * c - x[2 * p + 1] * s;
                im += x[2 * p] * s + x[2 * p + 1] * c;
            }
            y[2 * ki] = scale * re;
            y[2 * ki + 1] = scale * im;
        }
    }
    free(cs);
}
