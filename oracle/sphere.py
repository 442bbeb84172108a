"""oracle/sphere.py -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py).

Directional scale-discretised wavelet transform on the sphere, written out from
the definitions of arXiv:2402.01282 ("P:n" = /root/reference/PAPER.md line n)
with the readings R1-R17 of DESIGN.md.  The order of operations is that of
Algorithm 1; the heavy sums are the literal loops of
oracle/direct_sums.c.  `prec` selects the arithmetic: "f80" (long double,
the parity reference) or "f64" (double, the timed CPU baseline).

Array conventions (all C-ordered):
  f, W^Phi        [L][2L-1]            pixels on the MW grid theta_t x phi_p
  flm             [L][2L-1]            f_{l m} at [l][m + L-1]
  psi             [J-J0+1][L][2N-1]    Psi^j_{l n} at [j-J0][l][n + N-1]   (complex)
  phi             [L]                  Phi_{l 0}                           (real)
  W^{Psi j}       [2N-1][L_j][2L_j-1]  samples (gamma_g, beta_t, alpha_a)
  Wigner coeffs   [2N-1][L][2L-1]      at [n + N-1][l][m + L-1]
"""
import ctypes

import numpy as np

from . import build as _build

REAL = {"f80": np.longdouble, "f64": np.float64}
CPLX = {"f80": np.clongdouble, "f64": np.complex128}
_LIBS = {}

# DFT sums longer than this use numpy's pocketfft (a library FFT standing in for
# the same DFT sum, SURVEY.md 8(c) Tier 1); shorter ones are literal sums in C.
DIRECT_DFT_MAX = 511


def _lib(prec):
    if prec not in _LIBS:
        _build.build()
        lib = ctypes.CDLL(_build.lib_path(prec))
        assert lib.orc_sizeof_real() == np.dtype(REAL[prec]).itemsize
        _LIBS[prec] = lib
    return _LIBS[prec]


def num_threads(prec="f80"):
    return int(_lib(prec).orc_num_threads())


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _as(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def pi(prec):
    rt = REAL[prec]
    return rt(4) * np.arctan(rt(1))


# --------------------------------------------------------------------------
# sampling (McEwen-Wiaux)
# --------------------------------------------------------------------------
def mw_thetas(L, prec="f80"):
    rt = REAL[prec]
    return pi(prec) * (2 * np.arange(L).astype(rt) + 1) / rt(2 * L - 1)


def mw_phis(L, prec="f80"):
    rt = REAL[prec]
    return 2 * pi(prec) * np.arange(2 * L - 1).astype(rt) / rt(2 * L - 1)


# --------------------------------------------------------------------------
# Driscoll-Healy sampling ("sampling agnostic").  Reading R19: the paper names the sampling
# schemes of S2FFT without formulas; the equiangular Driscoll & Healy (1994) grid with 2L rings is taken,
#   theta_t = pi (2t+1)/(4L), t = 0..2L-1,   phi_p = 2 pi p/(2L-1), p = 0..2L-2,
# with the quadrature weights of their Theorem 3 on it,
#   q_t = (2/L) sin(theta_t) sum_{k<L} sin((2k+1) theta_t)/(2k+1):   sum_t q_t g(theta_t) = int_0^pi g sin(theta) dtheta
# for every g that is a cosine polynomial of degree < 2L (so the product of two band-limited functions is integrated
# exactly and no reweighting operator is needed).
# --------------------------------------------------------------------------
def dh_thetas(L, prec="f80"):
    rt = REAL[prec]
    return pi(prec) * (2 * np.arange(2 * L).astype(rt) + 1) / rt(4 * L)


def dh_weights(L, prec="f80"):
    rt = REAL[prec]
    th = dh_thetas(L, prec)
    k = np.arange(L).astype(rt)
    return (rt(2) / rt(L)) * np.sin(th) * (np.sin((2 * k[None, :] + 1) * th[:, None]) / (2 * k[None, :] + 1)).sum(axis=1)


def thetas_of(L, sampling, prec="f80"):
    if sampling == "mw":
        return mw_thetas(L, prec)
    if sampling == "dh":
        return dh_thetas(L, prec)
    raise ValueError("sampling must be 'mw' or 'dh'")


# --------------------------------------------------------------------------
# O1 filters (Appendix A)
# --------------------------------------------------------------------------
def _gauss_legendre(n, prec):
    """Gauss-Legendre nodes/weights on [-1,1]: numpy's double nodes polished by
    Newton steps on P_n in the working precision."""
    rt = REAL[prec]
    x = np.polynomial.legendre.leggauss(n)[0].astype(rt)
    for _ in range(4):
        p0 = np.ones_like(x)
        p1 = x.copy()
        for k in range(1, n):
            p0, p1 = p1, ((2 * k + 1) * x * p1 - k * p0) / rt(k + 1)
        dp = n * (x * p1 - p0) / (x * x - 1)
        x = x - p1 / dp
    p0 = np.ones_like(x)
    p1 = x.copy()
    for k in range(1, n):
        p0, p1 = p1, ((2 * k + 1) * x * p1 - k * p0) / rt(k + 1)
    dp = n * (x * p1 - p0) / (x * x - 1)
    w = 2 / ((1 - x * x) * dp * dp)
    return x, w


def schwartz_s(t):
    """s(t) = exp(-1/(1-t^2)) on (-1,1), 0 elsewhere (Eq. A3)."""
    t = np.asarray(t)
    out = np.zeros_like(t)
    inside = np.abs(t) < 1
    out[inside] = np.exp(-1 / (1 - t[inside] * t[inside]))
    return out


def s_lambda(t, lam):
    """s_lambda(t) = s(2 lam/(lam-1) (t - 1/lam) - 1) (Eq. A2)."""
    return schwartz_s(2 * lam / (lam - 1) * (t - 1 / lam) - 1)


def _bump_integral(a, b, lam, prec, nodes=400):
    """int_a^b s_lambda^2(t')/t' dt' for arrays a <= b inside [1/lam, 1] (the integrand of Eq. A4):
    converged Gauss-Legendre quadrature (R1d), two panels."""
    x, w = _gauss_legendre(nodes, prec)
    mid = (a + b) / 2
    tot = np.zeros_like(a)
    for lo, hi in ((a, mid), (mid, b)):
        half = (hi - lo) / 2
        tt = lo[:, None] + half[:, None] * (x[None, :] + 1)
        sl = s_lambda(tt, lam)
        tot = tot + half * np.sum(w[None, :] * sl * sl / tt, axis=1)
    return tot


def k_lambda(t, lam, prec="f80"):
    """k_lambda(t) = int_t^1 s_lambda^2(t')/t' dt' / int_{1/lam}^1 (same)  (Eq. A4);
    1 for t <= 1/lam, 0 for t >= 1."""
    rt = REAL[prec]
    t = np.atleast_1d(np.asarray(t, dtype=rt))
    lam = rt(lam)
    one = np.ones(1, dtype=rt)
    den = _bump_integral(one / lam, one, lam, prec)[0]
    lo = np.clip(t, 1 / lam, rt(1))
    return _bump_integral(lo, np.ones_like(lo), lam, prec) / den


def kappa_lambda_sq(t, lam, prec="f80"):
    """kappa_lambda(t)^2 = k_lambda(t/lam) - k_lambda(t) (Eq. A5).  Both terms are integrals of the
    same integrand, so their difference is the single integral over [t/lam, t] clipped to the support
    [1/lam, 1]; written that way the tiny values next to the edges of the support are not lost to
    cancellation (reading R1c)."""
    rt = REAL[prec]
    t = np.atleast_1d(np.asarray(t, dtype=rt))
    lam = rt(lam)
    one = np.ones(1, dtype=rt)
    den = _bump_integral(one / lam, one, lam, prec)[0]
    lo = np.clip(t / lam, 1 / lam, rt(1))
    hi = np.clip(t, 1 / lam, rt(1))
    return _bump_integral(lo, hi, lam, prec) / den


def scale_range(L, lam, J0):
    """J = smallest integer with lam^J >= L (R1b); scales j = J0..J."""
    J = 0
    while float(lam) ** J < L:
        J += 1
    if J0 < 0 or J0 > J:
        raise ValueError("J0 out of range")
    return J


def bandlimit_of_scale(j, L, lam, multires):
    """L_j = min(ceil(lam^{j+1}), L) with multiresolution (Eq. 38; R1c), else L."""
    if not multires:
        return L
    return int(min(int(np.ceil(float(lam) ** (j + 1) - 1e-9)), L))


def bandlimit_of_scaling(L, lam, J0, multires):
    """L_s = min(ceil(lam^{J0}), L) (R1c): Phi_{l0} vanishes for l >= lam^{J0}."""
    if not multires:
        return L
    return int(min(int(np.ceil(float(lam) ** J0 - 1e-9)), L))


def kappa(L, lam, J0, prec="f80"):
    """kappa^j(l) = kappa_lambda(l / lam^j), kappa_lambda(t) = sqrt(k(t/lam) - k(t))
    (Eq. A5; reading R1), j = J0..J, and the scaling profile
    eta(l) = sqrt(k_lambda(l / lam^J0)).  Returns ([J-J0+1][L], [L])."""
    rt = REAL[prec]
    J = scale_range(L, lam, J0)
    ell = np.arange(L).astype(rt)
    lamr = rt(lam)
    kap = np.zeros((J - J0 + 1, L), dtype=rt)
    for j in range(J0, J + 1):
        kap[j - J0] = np.sqrt(kappa_lambda_sq(ell / lamr ** j, lam, prec))
    eta = np.sqrt(k_lambda(ell / lamr ** J0, lam, prec))
    return kap, eta


def _binom(q, k):
    from math import comb
    return comb(q, k)


def zeta(L, N, prec="f80"):
    """zeta_{l m} = xi mu sqrt(2^-q binom(q, (q-m)/2)) (Eq. A6):
    xi = 1 for even N-1 else i; mu = [1-(-1)^{N+m}]/2; q = min(N-1, l-[1+(-1)^{N+l}]/2).
    Returned as complex [L][2N-1] at [l][m+N-1]."""
    rt, ct = REAL[prec], CPLX[prec]
    z = np.zeros((L, 2 * N - 1), dtype=ct)
    xi = ct(1) if (N - 1) % 2 == 0 else ct(1j)
    for l in range(L):
        q = min(N - 1, l - (1 + (-1) ** (N + l)) // 2)
        if q < 0:
            continue
        for m in range(-(N - 1), N):
            mu = (1 - (-1) ** (N + m)) // 2
            if mu == 0 or abs(m) > q or (q - m) % 2:
                continue
            z[l, m + N - 1] = xi * np.sqrt(rt(_binom(q, (q - m) // 2)) / rt(2) ** q)
    return z


def filters(L, N, lam, J0, prec="f80"):
    """Psi^j_{l n} = sqrt((2l+1)/8pi^2) kappa^j(l) zeta_{l n} (Eq. A9 without p);
    Phi_{l 0} = sqrt((2l+1)/4pi) eta(l) (Eq. A10).  Returns (psi, phi, J)."""
    rt = REAL[prec]
    J = scale_range(L, lam, J0)
    kap, eta = kappa(L, lam, J0, prec)
    z = zeta(L, N, prec)
    ell = np.arange(L).astype(rt)
    p = pi(prec)
    psi = np.sqrt((2 * ell + 1) / (8 * p * p))[None, :, None] * kap[:, :, None] * z[None, :, :]
    phi = np.sqrt((2 * ell + 1) / (4 * p)) * eta
    return psi, phi, J


# --------------------------------------------------------------------------
# plain DFT along the last axis (FFT ordering k = 0..n-1, unnormalised)
# --------------------------------------------------------------------------
def dft_last_axis(x, sign, prec):
    ct, rt = CPLX[prec], REAL[prec]
    x = _as(x, ct)
    n = x.shape[-1]
    if n > DIRECT_DFT_MAX:
        return np.fft.fft(x, axis=-1) if sign < 0 else np.fft.ifft(x, axis=-1) * n
    rows = int(np.prod(x.shape[:-1], dtype=np.int64))
    out = np.empty_like(x)
    lib = _lib(prec)
    scale = np.ones(1, dtype=rt)
    lib.orc_dft_rows.argtypes = [ctypes.c_int] * 5 + [ctypes.c_void_p] * 3
    lib.orc_dft_rows(rows, n, 0, n, int(sign), _ptr(scale), _ptr(x), _ptr(out))
    return out


def _centered_to_fft_order(a, L):
    """[..., 2L-1] indexed m+L-1  ->  indexed m mod (2L-1)."""
    return np.roll(a, -(L - 1), axis=-1)


def _fft_order_to_centered(a, L):
    return np.roll(a, L - 1, axis=-1)


# --------------------------------------------------------------------------
# beta-contractions and MW reweighting: thin wrappers over direct_sums.c
# --------------------------------------------------------------------------
def wigner_d(L, m, n, beta, prec="f80"):
    """d^l_{mn}(beta), l = 0..L-1 (O4)."""
    rt = REAL[prec]
    lib = _lib(prec)
    d = np.zeros(L, dtype=rt)
    b = np.array([beta], dtype=rt)
    lib.orc_wigner_d_p.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    lib.orc_wigner_d_p(int(L), int(m), int(n), _ptr(b), _ptr(d))
    return d


def dl_inverse(X, L, n, betas, prec):
    """F[mi][t] = sum_l d^l_{mn}(beta_t) X[l][mi]."""
    rt, ct = REAL[prec], CPLX[prec]
    X = _as(X, ct)
    betas = _as(betas, rt)
    F = np.empty((2 * L - 1, betas.size), dtype=ct)
    lib = _lib(prec)
    lib.orc_dl_inverse.argtypes = [ctypes.c_int] * 3 + [ctypes.c_void_p] * 3
    lib.orc_dl_inverse(int(L), int(n), int(betas.size), _ptr(betas), _ptr(X), _ptr(F))
    return F


def dl_forward(H, L, n, betas, prec):
    """W[l][mi] = sum_t d^l_{mn}(beta_t) H[mi][t]."""
    rt, ct = REAL[prec], CPLX[prec]
    H = _as(H, ct)
    betas = _as(betas, rt)
    W = np.empty((L, 2 * L - 1), dtype=ct)
    lib = _lib(prec)
    lib.orc_dl_forward.argtypes = [ctypes.c_int] * 3 + [ctypes.c_void_p] * 3
    lib.orc_dl_forward(int(L), int(n), int(betas.size), _ptr(betas), _ptr(H), _ptr(W))
    return W


def mw_reweight(F, L, sigma, prec):
    """O3 (ii)-(vi) on columns F[c][t], parity sigma[c] = +-1."""
    ct = CPLX[prec]
    F = _as(F, ct)
    sigma = _as(sigma, np.int32)
    H = np.empty_like(F)
    lib = _lib(prec)
    lib.orc_mw_reweight.argtypes = [ctypes.c_int, ctypes.c_int] + [ctypes.c_void_p] * 3
    lib.orc_mw_reweight(int(L), int(F.shape[0]), _ptr(sigma), _ptr(F), _ptr(H))
    return H


# --------------------------------------------------------------------------
# O2 / O3: spherical harmonic transforms Y^-1, Y (Eqs. 2-3), spin s (sY_lm by reading R2, Goldberg et al. 1967 convention; the paper prints no formula):
#   sY_{lm}(theta, phi) = (-1)^s sqrt((2l+1)/4pi) D^{l*}_{m,-s}(phi, theta, 0)
#                       = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi},      zero for l < |s|.
# --------------------------------------------------------------------------
def sht_inverse(flm, L, prec="f80", thetas=None, spin=0, sampling="mw"):
    """f(theta_t, phi_p) = sum_{l m} f_{lm} sY_{lm}; spin 0: Y_{lm} = sqrt((2l+1)/4pi) d^l_{m0}(theta) e^{i m phi}
    (Eq. 3; R2).  `thetas` overrides the MW rings (used to evaluate single rings)."""
    rt, ct = REAL[prec], CPLX[prec]
    flm = _as(flm, ct)
    ell = np.arange(L).astype(rt)
    c_l = np.sqrt((2 * ell + 1) / (4 * pi(prec))) * (-1 if spin % 2 else 1)
    th = thetas_of(L, sampling, prec) if thetas is None else _as(thetas, rt)
    Fm = dl_inverse(c_l[:, None] * flm, L, -spin, th, prec)      # [mi][t]
    Fm = _centered_to_fft_order(Fm.T, L)                          # [t][m mod n]
    return dft_last_axis(Fm, +1, prec)                            # sum_m F_m e^{+i m phi_p}


def sht_forward(f, L, prec="f80", spin=0, sampling="mw"):
    """f_{lm} = int f sY*_{lm} dOmega, exact on the MW grid for band-limit L (O3, R3); the integrand's theta
    dependence has parity (-1)^{m+s} under the extension of R3 (ii).  sampling="dh": the same integral by the
    Driscoll-Healy quadrature on 2L rings, f_{lm} = 2 pi c_l sum_t q_t d^l_{m,-s}(theta_t) F_m(theta_t)."""
    rt, ct = REAL[prec], CPLX[prec]
    f = _as(f, ct)
    n = 2 * L - 1
    Fm = dft_last_axis(f, -1, prec) / rt(n)                       # (i)  [t][m mod n]
    Fm = _fft_order_to_centered(Fm, L).T                          # [mi][t]
    if sampling == "dh":
        W = dl_forward(Fm * dh_weights(L, prec)[None, :], L, -spin, dh_thetas(L, prec), prec)
        ell = np.arange(L).astype(rt)
        c_l = np.sqrt((2 * ell + 1) / (4 * pi(prec))) * (-1 if spin % 2 else 1)
        return 2 * pi(prec) * c_l[:, None] * W
    m = np.arange(-(L - 1), L)
    H = mw_reweight(Fm, L, np.where((m + spin) % 2 == 0, 1, -1), prec)   # (ii)-(vi), parity (-1)^{m+s}
    W = dl_forward(H, L, -spin, mw_thetas(L, prec), prec)         # (vii)
    ell = np.arange(L).astype(rt)
    c_l = np.sqrt((2 * ell + 1) / (4 * pi(prec))) * (-1 if spin % 2 else 1)
    return (2 * pi(prec) / rt(n)) * c_l[:, None] * W


# --------------------------------------------------------------------------
# Wigner transforms D^-1, D on SO(3) (Eqs. 4-5; Eqs. 47-48)
# --------------------------------------------------------------------------
def _gamma_phases(N, sign, prec):
    """E[g][ni] = exp(sign * i * n * gamma_g), gamma_g = 2 pi g/(2N-1), n = ni-(N-1)."""
    rt, ct = REAL[prec], CPLX[prec]
    ng = 2 * N - 1
    g = np.arange(ng)[:, None]
    n = np.arange(-(N - 1), N)[None, :]
    r = (g * n) % ng
    ang = 2 * pi(prec) * r.astype(rt) / rt(ng)
    return (np.cos(ang) + sign * 1j * np.sin(ang)).astype(ct)


def wigner_inverse(X, L, N, prec="f80", n_list=None, thetas=None, sampling="mw"):
    """W(gamma_g, beta_t, alpha_a) = sum_{l m n} X[n][l][m] d^l_{mn}(beta_t) e^{i(m alpha_a + n gamma_g)}
    i.e. Eq. 5 with f^l_{mn} (2l+1)/(8 pi^2) = X and D^{l*}_{mn} from Eq. 47.
    n outside n_list is treated as identically zero."""
    rt, ct = REAL[prec], CPLX[prec]
    X = _as(X, ct)
    th = thetas_of(L, sampling, prec) if thetas is None else _as(thetas, rt)
    ns = range(-(N - 1), N) if n_list is None else n_list
    Fmn = np.zeros((2 * N - 1, th.size, 2 * L - 1), dtype=ct)     # [ni][t][mi]
    for n in ns:
        Fmn[n + N - 1] = dl_inverse(X[n + N - 1], L, n, th, prec).T
    Eg = _gamma_phases(N, +1, prec)                               # [g][ni]
    A = np.einsum("gn,ntm->gtm", Eg, Fmn)                         # sum over n
    A = _centered_to_fft_order(A, L)
    return dft_last_axis(A, +1, prec)                             # sum over m


def wigner_forward(W, L, N, prec="f80", n_list=None, sampling="mw"):
    """f^l_{mn} = int_{SO(3)} W D^l_{mn} dOmega(rho) (Eq. 4; R6) on the MW x gamma grid:
    2-D DFT over (alpha, gamma) (Eq. 48), MW reweighting in beta, projection on d^l_{mn}."""
    rt, ct = REAL[prec], CPLX[prec]
    W = _as(W, ct)
    n_a, n_g = 2 * L - 1, 2 * N - 1
    A = dft_last_axis(W, -1, prec) / rt(n_a)                      # [g][t][m mod n]
    A = _fft_order_to_centered(A, L)
    Eg = _gamma_phases(N, -1, prec)                               # [g][ni]
    Fmn = np.einsum("gn,gtm->ntm", Eg, A) / rt(n_g)               # [ni][t][mi]
    ns = range(-(N - 1), N) if n_list is None else n_list
    out = np.zeros((2 * N - 1, L, 2 * L - 1), dtype=ct)
    m = np.arange(-(L - 1), L)
    p = pi(prec)
    for n in ns:
        if sampling == "dh":                                      # Driscoll-Healy quadrature in beta, no reweighting
            H = Fmn[n + N - 1].T * dh_weights(L, prec)[None, :]
            out[n + N - 1] = (2 * p) ** 2 * dl_forward(H, L, n, dh_thetas(L, prec), prec)
            continue
        sigma = np.where((m + n) % 2 == 0, 1, -1)
        H = mw_reweight(Fmn[n + N - 1].T, L, sigma, prec)         # [mi][t]
        out[n + N - 1] = ((2 * p) ** 2 / rt(n_a)) * dl_forward(H, L, n, mw_thetas(L, prec), prec)
    return out


# --------------------------------------------------------------------------
# O5 / O6: Algorithm 1
# --------------------------------------------------------------------------
def _active_n(psi_j):
    """n with Psi^j_{. n} not identically zero (the set script-N of DESIGN.md)."""
    N = (psi_j.shape[1] + 1) // 2
    return [ni - (N - 1) for ni in range(2 * N - 1) if np.any(psi_j[:, ni] != 0)]


def _crop_lm(a, L, Lc):
    """[.., L][2L-1] -> [.., Lc][2Lc-1] (l < Lc, |m| < Lc)."""
    return a[..., :Lc, (L - 1) - (Lc - 1):(L - 1) + Lc]


def _pad_lm(a, Lc, L):
    out = np.zeros(a.shape[:-2] + (L, 2 * L - 1), dtype=a.dtype)
    out[..., :Lc, (L - 1) - (Lc - 1):(L - 1) + Lc] = a
    return out


def analysis_from_flm(flm, L, N, lam, J0, multires, prec="f80", filt=None, scales=None, rings=None, spin=0,
                      sampling="mw"):
    """Algorithm 1 'Analysis' after its first line:
    returns (W_phi, {j: W_psi_j}).  `scales` restricts j; `rings` = {j: ring indices}
    evaluates only those beta rings of scale j (same sums, fewer outputs)."""
    rt, ct = REAL[prec], CPLX[prec]
    psi, phi, J = filters(L, N, lam, J0, prec) if filt is None else filt
    flm = _as(flm, ct)
    ell = np.arange(L).astype(rt)
    # W^Phi_hat = Phi f_hat : einsum("lm,l->lm") with entries sqrt(4pi/(2l+1)) Phi*_{l0}  (Eq. 29/41, R5)
    wphi_hat = np.einsum("lm,l->lm", flm, np.sqrt(4 * pi(prec) / (2 * ell + 1)) * phi)
    Ls = bandlimit_of_scaling(L, lam, J0, multires)
    W_phi = sht_inverse(_crop_lm(wphi_hat, L, Ls), Ls, prec, spin=spin, sampling=sampling)   # Y^-1 (Eq. 12)
    W_psi = {}
    for j in (range(J0, J + 1) if scales is None else scales):
        Lj = bandlimit_of_scale(j, L, lam, multires)
        # W_hat^{Psi j} = N Psi^j f_hat: einsum("lm,ln->nlm"); N = 8pi^2/(2l+1) cancels
        # the (2l+1)/(8pi^2) of Eq. 5 inside D^-1
        X = np.einsum("lm,ln->nlm", flm, np.conj(psi[j - J0]))
        th = None
        if rings is not None and j in rings:
            th = thetas_of(Lj, sampling, prec)[np.asarray(rings[j])]
        W_psi[j] = wigner_inverse(_crop_lm(X, L, Lj), Lj, N, prec, _active_n(psi[j - J0]), th, sampling=sampling)  # D^-1
    return W_phi, W_psi


def analysis(f, L, N, lam, J0, multires, prec="f80", filt=None, spin=0, sampling="mw"):
    """Algorithm 1 'Analysis wavelet transform'; `spin`: the signal's spin number (spin fields: Eq. 1; sY_lm: reading R2)."""
    flm = sht_forward(f, L, prec, spin=spin, sampling=sampling)   # f_hat <- Y f
    return analysis_from_flm(flm, L, N, lam, J0, multires, prec, filt, spin=spin, sampling=sampling)


def synthesis_to_flm(W_phi, W_psi, L, N, lam, J0, multires, prec="f80", filt=None, spin=0, sampling="mw"):
    """Algorithm 1 'Synthesis' up to its last line: returns f_hat."""
    rt, ct = REAL[prec], CPLX[prec]
    psi, phi, J = filters(L, N, lam, J0, prec) if filt is None else filt
    ell = np.arange(L).astype(rt)
    Ls = bandlimit_of_scaling(L, lam, J0, multires)
    wphi_hat = _pad_lm(sht_forward(W_phi, Ls, prec, spin=spin, sampling=sampling), Ls, L)    # Y W^Phi
    flm = np.einsum("lm,l->lm", wphi_hat, np.sqrt(4 * pi(prec) / (2 * ell + 1)) * phi)
    for j in range(J0, J + 1):
        Lj = bandlimit_of_scale(j, L, lam, multires)
        what = wigner_forward(W_psi[j], Lj, N, prec, _active_n(psi[j - J0]), sampling=sampling)     # D W^{Psi j}
        # f_hat += Psi^dagger W_hat: einsum("nlm,ln->lm")  (Eq. 42; no extra normalisation)
        flm = flm + np.einsum("nlm,ln->lm", _pad_lm(what, Lj, L), psi[j - J0])
    return flm


def synthesis(W_phi, W_psi, L, N, lam, J0, multires, prec="f80", filt=None, spin=0, sampling="mw"):
    """Algorithm 1 'Synthesis wavelet transform'."""
    flm = synthesis_to_flm(W_phi, W_psi, L, N, lam, J0, multires, prec, filt, spin=spin, sampling=sampling)
    return sht_inverse(flm, L, prec, spin=spin, sampling=sampling)   # f <- Y^-1 f_hat
