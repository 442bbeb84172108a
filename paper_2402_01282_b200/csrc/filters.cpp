// filters.cpp -- host-side kernel build (Appendix A of arXiv:2402.01282).
// Pure host C++ in long double; results are rounded to double.  No GPU needed.
//
//   s(t)        = exp(-1/(1-t^2)) on (-1,1)                                  (Eq. A3)
//   s_lam(t)    = s(2 lam/(lam-1) (t - 1/lam) - 1)                           (Eq. A2)
//   k_lam(t)    = int_t^1 s_lam^2/t' dt' / int_{1/lam}^1 s_lam^2/t' dt'       (Eq. A4)
//   kappa_lam^2 = k_lam(t/lam) - k_lam(t)  (Eq. A5) = int_{t/lam}^{t} (clipped to [1/lam,1]) / same denominator
//   zeta_{lm}   = xi mu sqrt(2^-q binom(q,(q-m)/2))                          (Eq. A6)
#include "host_math.h"

#include <cmath>
#include <vector>

namespace s2w {

namespace {

typedef long double ld;

const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

// Gauss-Legendre rule on [-1,1] with `n` nodes: Newton iteration on P_n from the Chebyshev-like guess.
void gauss_legendre(int n, std::vector<ld> &x, std::vector<ld> &w)
{
    x.assign(n, 0);
    w.assign(n, 0);
    for (int i = 0; i < n; ++i) {
        ld z = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
        ld dp = 1;
        for (int it = 0; it < 100; ++it) {
            ld p0 = 1, p1 = z;
            for (int k = 1; k < n; ++k) {
                ld p2 = ((2 * k + 1) * z * p1 - k * p0) / (k + 1);
                p0 = p1;
                p1 = p2;
            }
            dp = n * (z * p1 - p0) / (z * z - 1);
            ld dz = p1 / dp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        // recompute derivative at the converged node
        ld p0 = 1, p1 = z;
        for (int k = 1; k < n; ++k) {
            ld p2 = ((2 * k + 1) * z * p1 - k * p0) / (k + 1);
            p0 = p1;
            p1 = p2;
        }
        dp = n * (z * p1 - p0) / (z * z - 1);
        x[i] = z;
        w[i] = 2 / ((1 - z * z) * dp * dp);
    }
}

struct BumpIntegrator {
    ld lam;
    std::vector<ld> gx, gw;
    ld denom;
    explicit BumpIntegrator(ld lam_) : lam(lam_)
    {
        gauss_legendre(96, gx, gw);
        denom = 1;
        denom = integral(1 / lam, 1);
    }
    ld integrand(ld t) const
    {
        ld u = 2 * lam / (lam - 1) * (t - 1 / lam) - 1;
        if (!(fabsl(u) < 1)) return 0;
        ld s = expl(-1 / (1 - u * u));
        return s * s / t;
    }
    // int_a^b s_lam^2(t)/t dt, composite Gauss-Legendre over 16 panels (the integrand is a smooth bump).
    ld integral(ld a, ld b) const
    {
        if (!(b > a)) return 0;
        const int panels = 16;
        ld tot = 0;
        for (int p = 0; p < panels; ++p) {
            ld lo = a + (b - a) * p / panels, hi = a + (b - a) * (p + 1) / panels;
            ld half = (hi - lo) / 2, mid = (hi + lo) / 2, acc = 0;
            for (size_t i = 0; i < gx.size(); ++i) acc += gw[i] * integrand(mid + half * gx[i]);
            tot += half * acc;
        }
        return tot;
    }
    static ld clip(ld t, ld lo, ld hi) { return t < lo ? lo : (t > hi ? hi : t); }
    ld k(ld t) const { return integral(clip(t, 1 / lam, 1), 1) / denom; }
    ld kappa_sq(ld t) const { return integral(clip(t / lam, 1 / lam, 1), clip(t, 1 / lam, 1)) / denom; }
};

ld ipow(ld b, int e)
{
    ld r = 1;
    for (int i = 0; i < e; ++i) r *= b;
    return r;
}

}  // namespace

int scale_count(int L, double lambda)
{
    int J = 0;
    long double p = 1;
    while (p < (long double)L) {
        p *= (long double)lambda;
        ++J;
    }
    return J;
}

int scale_bandlimit(int j, int L, double lambda, bool multires)
{
    if (!multires) return L;
    long double v = ceill(ipow((ld)lambda, j + 1) - 1e-9L);
    return v < (ld)L ? (int)v : L;
}

int scaling_bandlimit(int L, double lambda, int J0, bool multires)
{
    if (!multires) return L;
    long double v = ceill(ipow((ld)lambda, J0) - 1e-9L);
    return v < (ld)L ? (int)v : L;
}

// kappa[j-J0][l] = kappa_lam(l/lam^j), j = J0..J;  ksc[l] = k_lam(l/lam^J0)   (reading R1)
void kappa_profiles(int L, double lambda, int J0, int J, std::vector<double> &kappa, std::vector<double> &ksc)
{
    BumpIntegrator B((ld)lambda);
    kappa.assign((size_t)(J - J0 + 1) * L, 0.0);
    ksc.assign(L, 0.0);
    for (int j = J0; j <= J; ++j) {
        ld sc = ipow((ld)lambda, j);
        for (int l = 0; l < L; ++l) kappa[(size_t)(j - J0) * L + l] = (double)sqrtl(B.kappa_sq((ld)l / sc));
    }
    ld sc0 = ipow((ld)lambda, J0);
    for (int l = 0; l < L; ++l) ksc[l] = (double)B.k((ld)l / sc0);
}

// zeta[l][n+N-1] complex (re, im)   (Eq. A6)
void zeta_tiling(int L, int N, std::vector<double> &zeta)
{
    zeta.assign((size_t)L * (2 * N - 1) * 2, 0.0);
    bool imag = ((N - 1) % 2) != 0;  // xi = 1 for even N-1, i otherwise
    for (int l = 0; l < L; ++l) {
        int par = ((N + l) % 2 == 0) ? 1 : 0;  // [1 + (-1)^{N+l}]/2
        int q = l - par;
        if (q > N - 1) q = N - 1;
        if (q < 0) continue;
        for (int m = -(N - 1); m <= N - 1; ++m) {
            int mu = ((N + m) % 2 == 0) ? 0 : 1;  // [1 - (-1)^{N+m}]/2
            int am = m < 0 ? -m : m;
            if (!mu || am > q || ((q - m) % 2)) continue;
            int kk = (q - m) / 2;
            ld binom = 1;
            for (int i = 1; i <= kk; ++i) binom = binom * (q - kk + i) / i;
            double v = (double)sqrtl(binom / ipow(2, q));
            size_t o = ((size_t)l * (2 * N - 1) + (m + N - 1)) * 2;
            zeta[o + (imag ? 1 : 0)] = v;
        }
    }
}

double pi_d() { return (double)PI_L; }

// Generalised Gauss-Laguerre (alpha = 2) nodes x_i and q_i = w_i e^{x_i} (reading R8):
// x_i are the roots of L_P^(2); w_i = Gamma(P+3) x_i / (P! (P+1)^2 [L_{P+1}^(2)(x_i)]^2), so that
// w_i e^{x_i} = (P+2) x_i / ((P+1) [e^{-x_i/2} L_{P+1}^(2)(x_i)]^2).
// Roots by Newton iteration with deflation-free bracketing: the scaled function e^{-x/2} L_P^(2)(x) is evaluated by
// the three-term recurrence, sign changes are located on a fine grid and refined by bisection + Newton.
namespace {
ld scaled_laguerre2(int n, ld x, ld *prev)
{
    ld l0 = expl(-x / 2), l1 = (3 - x) * l0;
    if (n == 0) {
        if (prev) *prev = 0;
        return l0;
    }
    for (int k = 1; k < n; ++k) {
        ld l2 = ((2 * k + 3 - x) * l1 - (k + 2) * l0) / (k + 1);
        l0 = l1;
        l1 = l2;
    }
    if (prev) *prev = l0;
    return l1;
}
}  // namespace

void gauss_laguerre2(int P, std::vector<double> &x, std::vector<double> &q)
{
    x.assign(P, 0.0);
    q.assign(P, 0.0);
    // roots lie in (0, 4P + 6); oscillation spacing is >= ~ 1/(P+2) near the origin
    std::vector<ld> roots;
    ld hi = 4.0L * P + 10, step = 0.5L / (P + 2);
    ld a = 1e-12L, fa = scaled_laguerre2(P, a, 0);
    while (a < hi && (int)roots.size() < P) {
        // spacing between roots grows with x: use a step proportional to sqrt(x) spacing estimate
        ld h = step * (1 + 2 * sqrtl(a * (P + 2)));
        ld b = a + h, fb = scaled_laguerre2(P, b, 0);
        if ((fa < 0) != (fb < 0)) {
            ld lo = a, up = b, flo = fa;
            for (int it = 0; it < 200; ++it) {
                ld mid = (lo + up) / 2, fm = scaled_laguerre2(P, mid, 0);
                if ((fm < 0) == (flo < 0)) {
                    lo = mid;
                    flo = fm;
                } else
                    up = mid;
                if (up - lo < 1e-18L * (1 + mid)) break;
            }
            ld r = (lo + up) / 2;
            for (int it = 0; it < 4; ++it) {  // Newton polish: x L_n' = n L_n - (n+2) L_{n-1}
                ld pm1, f = scaled_laguerre2(P, r, &pm1);
                ld df = (P * f - (P + 2) * pm1) / r;  // e^{-x/2} L_P'(x)
                // d/dx [e^{-x/2} L] = e^{-x/2} (L' - L/2); at a root L = 0 so the scaled derivative is e^{-x/2} L'
                if (df != 0) r -= f / df;
            }
            roots.push_back(r);
        }
        a = b;
        fa = fb;
    }
    for (int i = 0; i < P && i < (int)roots.size(); ++i) {
        ld r = roots[i];
        ld lp1 = scaled_laguerre2(P + 1, r, 0);
        x[i] = (double)r;
        q[i] = (double)((ld)(P + 2) * r / ((ld)(P + 1) * lp1 * lp1));
    }
    if ((int)roots.size() != P) x.clear();  // signals failure to the caller
}

// K_p(r_i) for p < Pband at nodes x_i = r_i/tau: sqrt(1/((p+1)(p+2))) tau^{-3/2} e^{-x/2} L_p^(2)(x)   (Eq. 6)
void laguerre_basis(int Pband, const std::vector<double> &x, double tau, std::vector<double> &K)
{
    size_t n = x.size();
    K.assign((size_t)Pband * n, 0.0);
    ld t32 = powl((ld)tau, -1.5L);
    for (size_t i = 0; i < n; ++i) {
        ld xi = x[i];
        ld l0 = expl(-xi / 2), l1 = (3 - xi) * l0;
        for (int p = 0; p < Pband; ++p) {
            ld v = (p == 0) ? l0 : l1;
            if (p >= 1 && p + 1 < Pband) {
                ld l2 = ((2 * p + 3 - xi) * l1 - (p + 2) * l0) / (p + 1);
                l0 = l1;
                l1 = l2;
            }
            K[(size_t)p * n + i] = (double)(v * t32 / sqrtl((ld)(p + 1) * (p + 2)));
        }
    }
}

}  // namespace s2w
