"""oracle/ball.py -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py).

Fourier-Laguerre directional wavelet transform on the ball B^3 = R+ x S^2,
written out from arXiv:2402.01282 ("P:n" = PAPER.md line n), Algorithm 2
(P:463-484), with the readings R7-R10, R15 of DESIGN.md.  Angular work is
delegated to oracle/sphere.py; the radial part is the definition below.

Array conventions:
  f, W^Phi          [P][L][2L-1]                 shells r_i = tau x_i (Gauss-Laguerre nodes)
  flmp              [P][L][2L-1]                 f_{l m p} at [p][l][m+L-1]
  W^{Psi jj'}       [P_j'][2N-1][L_j][2L_j-1]    shells of the P_j'-node rule
"""
import numpy as np

from . import sphere as S

REAL, CPLX = S.REAL, S.CPLX


# --------------------------------------------------------------------------
# O8 radial: generalised Gauss-Laguerre (alpha = 2) nodes and the basis K_p (Eq. 6)
# --------------------------------------------------------------------------
def _scaled_laguerre2(nmax, x):
    """lag[n] = exp(-x/2) L_n^{(2)}(x), n = 0..nmax, by the three-term recurrence
    (n+1) L_{n+1} = (2n+3-x) L_n - (n+2) L_{n-1}   (alpha = 2)."""
    x = np.asarray(x)
    out = np.empty((nmax + 1,) + x.shape, dtype=x.dtype)
    out[0] = np.exp(-x / 2)
    if nmax >= 1:
        out[1] = (3 - x) * out[0]
    for n in range(1, nmax):
        out[n + 1] = ((2 * n + 3 - x) * out[n] - (n + 2) * out[n - 1]) / (n + 1)
    return out


def radial_nodes(P, tau, prec="f80"):
    """Nodes x_i = roots of L_P^{(2)} (R8), r_i = tau x_i, and the weights of
    int_0^inf x^2 e^{-x} g(x) dx = sum_i w_i g(x_i):
        w_i = Gamma(P+3) x_i / (P! (P+1)^2 [L_{P+1}^{(2)}(x_i)]^2).
    Returned: r_i, and q_i = tau^3 w_i e^{x_i} (the weight that multiplies f(r_i) K_p(r_i)
    in the quadrature of Eq. 7), computed without ever forming w_i or e^{x_i}."""
    rt = REAL[prec]
    from scipy.special import roots_genlaguerre
    x = roots_genlaguerre(P, 2)[0].astype(rt)
    for _ in range(5):  # Newton polish in working precision: x L_n' = n L_n - (n+2) L_{n-1}
        lag = _scaled_laguerre2(P, x)
        dlag = (P * lag[P] - (P + 2) * lag[P - 1]) / x if P >= 1 else np.zeros_like(x)
        x = x - lag[P] / dlag
    lag = _scaled_laguerre2(P + 1, x)
    # w_i e^{x_i} = (P+2) x_i / ((P+1) [e^{-x_i/2} L_{P+1}(x_i)]^2)   since Gamma(P+3)/P! = (P+1)(P+2)
    q = rt(tau) ** 3 * rt(P + 2) * x / (rt(P + 1) * lag[P + 1] ** 2)
    return rt(tau) * x, q


def laguerre_basis(Pmax, r, tau, prec="f80"):
    """K[p][i] = K_p(r_i) = sqrt(p!/(p+2)!) tau^{-3/2} e^{-r/(2 tau)} L_p^{(2)}(r/tau)  (Eq. 6)."""
    rt = REAL[prec]
    r = np.asarray(r, dtype=rt)
    lag = _scaled_laguerre2(max(Pmax - 1, 0), r / rt(tau))[:Pmax]
    p = np.arange(Pmax).astype(rt)
    norm = 1 / np.sqrt((p + 1) * (p + 2)) / rt(tau) ** rt(1.5)
    return norm[:, None] * lag


def laguerre_forward(fr, P, tau, prec="f80", nodes=None):
    """f_p = int r^2 f(r) K_p(r) dr (Eq. 7) by Gauss-Laguerre quadrature on the P nodes:
    f_p = sum_i q_i K_p(r_i) f(r_i).  fr: [P][...]."""
    r, q = radial_nodes(P, tau, prec) if nodes is None else nodes
    K = laguerre_basis(P, r, tau, prec)
    return np.einsum("pi,i,i...->p...", K, q, fr)


def laguerre_inverse(fp, Pnodes, tau, prec="f80", nodes=None):
    """f(r_i) = sum_p f_p K_p(r_i) (Eq. 8) on the Pnodes-node grid.  fp: [Pband][...]."""
    r, _ = radial_nodes(Pnodes, tau, prec) if nodes is None else nodes
    K = laguerre_basis(fp.shape[0], r, tau, prec)
    return np.einsum("pi,p...->i...", K, fp)


# --------------------------------------------------------------------------
# Z, Z^-1: spherical-Laguerre transforms (Eqs. 10-11)
# --------------------------------------------------------------------------
def z_forward(f, L, P, tau, prec="f80"):
    flm_r = np.stack([S.sht_forward(f[i], L, prec) for i in range(P)])
    return laguerre_forward(flm_r, P, tau, prec)


def z_inverse(flmp, L, P, tau, prec="f80"):
    flm_r = laguerre_inverse(flmp, P, tau, prec)
    return np.stack([S.sht_inverse(flm_r[i], L, prec) for i in range(P)])


# --------------------------------------------------------------------------
# Q, Q^-1: Wigner-Laguerre transforms on H^4 = R+ x SO(3) (Eqs. 24-25): Q = K D, with
# D of Eq. 4 (no conjugate, reading R6) and K of Eq. 7.  Reading R18: Eq. 24 prints Q^* in the analysis integral, which
# contradicts P:424 ("Q = K D", D as in Eq. 4) and Eqs. 4-5; the basis function is Q^l_{mnp}(h) = K_p(r) D^l_{mn}(rho),
# analysis  f^l_{mnp} = int f Q^l_{mnp} r^2 dr dOmega(rho),  synthesis  f = sum (2l+1)/(8 pi^2) f^l_{mnp} K_p D^{l*}_{mn}.
#   f      [P][2N-1][L][2L-1]   samples f(r_i, gamma_g, beta_t, alpha_a) on the Gauss-Laguerre shells x the MW grid
#   fhat   [2N-1][P][L][2L-1]   f^l_{mnp} at [n+N-1][p][l][m+L-1], |n| <= min(N-1, l)
# --------------------------------------------------------------------------
def q_forward(f, L, P, N, tau, prec="f80"):
    ct = CPLX[prec]
    per_shell = np.stack([S.wigner_forward(f[i], L, N, prec) for i in range(P)])      # [i][n][l][m]: D, Eq. 4
    out = np.empty((2 * N - 1, P, L, 2 * L - 1), dtype=ct)
    for ni in range(2 * N - 1):
        out[ni] = laguerre_forward(per_shell[:, ni], P, tau, prec)                   # K, Eq. 7
    return out


def q_inverse(fhat, L, P, N, tau, prec="f80"):
    rt, ct = REAL[prec], CPLX[prec]
    fhat = fhat.astype(ct)
    ell = np.arange(L).astype(rt)
    w = (2 * ell + 1) / (8 * S.pi(prec) ** 2)                                          # Eq. 5 / Eq. 25
    shells = np.stack([laguerre_inverse(fhat[ni], P, tau, prec) for ni in range(2 * N - 1)])   # [n][i][l][m]: K^-1
    out = np.empty((P, 2 * N - 1, L, 2 * L - 1), dtype=ct)
    for i in range(P):
        X = shells[:, i] * w[None, :, None]
        out[i] = S.wigner_inverse(X, L, N, prec)                                      # D^-1, Eq. 5 with Eq. 47
    return out


# --------------------------------------------------------------------------
# filters (Appendix A.3-A.4)
# --------------------------------------------------------------------------
def filters(L, P, N, lam, nu, J0, J0p, prec="f80"):
    """kappa^j(l), kappa^{j'}(p), zeta_{l n} (Eq. A9 stored separably) and
    Phi_{l 0 p} = sqrt((2l+1)/4pi) sqrt(a + b - a b), a = k_lam(l/lam^J0), b = k_nu(p/nu^J0')  (R9).
    Returns dict(kap_l [J-J0+1][L], kap_p [J'-J0'+1][P], zeta [L][2N-1], phi [P][L], J, Jp)."""
    rt = REAL[prec]
    J = S.scale_range(L, lam, J0)
    Jp = S.scale_range(P, nu, J0p)
    kap_l, eta_l = S.kappa(L, lam, J0, prec)
    kap_p, eta_p = S.kappa(P, nu, J0p, prec)
    a = eta_l ** 2
    b = eta_p ** 2
    ell = np.arange(L).astype(rt)
    phi = np.sqrt((2 * ell + 1) / (4 * S.pi(prec)))[None, :] * np.sqrt(
        a[None, :] + b[:, None] - a[None, :] * b[:, None])
    return dict(kap_l=kap_l, kap_p=kap_p, zeta=S.zeta(L, N, prec), phi=phi, J=J, Jp=Jp)


def psi_scale(filt, j, jp, J0, J0p, prec="f80"):
    """Psi^{jj'}_{l n p} = sqrt((2l+1)/8pi^2) kappa^j(l) kappa^{j'}(p) zeta_{l n} as [P][L][2N-1]."""
    rt = REAL[prec]
    L = filt["kap_l"].shape[1]
    ell = np.arange(L).astype(rt)
    pre = np.sqrt((2 * ell + 1) / (8 * S.pi(prec) ** 2))
    return (filt["kap_p"][jp - J0p][:, None, None] * (pre * filt["kap_l"][j - J0])[None, :, None]
            * filt["zeta"][None, :, :])


# --------------------------------------------------------------------------
# O9: Algorithm 2
# --------------------------------------------------------------------------
def analysis_from_flmp(flmp, L, P, N, lam, nu, J0, J0p, tau, prec="f80", filt=None, scales=None):
    """Algorithm 2 'Analysis' after its first line: returns (W_phi [P][L][2L-1], {(j,j'): W})."""
    rt, ct = REAL[prec], CPLX[prec]
    filt = filters(L, P, N, lam, nu, J0, J0p, prec) if filt is None else filt
    flmp = np.asarray(flmp, dtype=ct)
    ell = np.arange(L).astype(rt)
    # W^Phi_hat = Phi f_hat: einsum("plm,pl->plm") with sqrt(4pi/(2l+1)) Phi_{l0p}  (Eq. 35)
    wphi_hat = np.einsum("plm,pl->plm", flmp, np.sqrt(4 * S.pi(prec) / (2 * ell + 1))[None, :] * filt["phi"])
    W_phi = z_inverse(wphi_hat, L, P, tau, prec)
    out = {}
    all_scales = [(j, jp) for j in range(J0, filt["J"] + 1) for jp in range(J0p, filt["Jp"] + 1)]
    for (j, jp) in (all_scales if scales is None else scales):
        Lj = S.bandlimit_of_scale(j, L, lam, True)
        Pj = S.bandlimit_of_scale(jp, P, nu, True)
        psi = psi_scale(filt, j, jp, J0, J0p, prec)                      # [P][L][2N-1]
        X = np.einsum("plm,pln->pnlm", flmp, np.conj(psi))               # N Psi^{jj'} f_hat
        X = S._crop_lm(X, L, Lj)[:Pj]                                     # l < L_j, p < P_j'
        Xr = laguerre_inverse(X, Pj, tau, prec)                          # K^-1 on the P_j' grid
        ns = S._active_n(psi.reshape(-1, psi.shape[-1]))
        out[(j, jp)] = np.stack([S.wigner_inverse(Xr[i], Lj, N, prec, ns) for i in range(Pj)])  # D^-1 per shell
    return W_phi, out


def analysis(f, L, P, N, lam, nu, J0, J0p, tau, prec="f80", filt=None):
    """Algorithm 2 'Analysis wavelet transform': W = Q^-1 N Psi Z f."""
    return analysis_from_flmp(z_forward(f, L, P, tau, prec), L, P, N, lam, nu, J0, J0p, tau, prec, filt)


def synthesis_to_flmp(W_phi, W_psi, L, P, N, lam, nu, J0, J0p, tau, prec="f80", filt=None):
    """Algorithm 2 'Synthesis' up to its last line."""
    rt, ct = REAL[prec], CPLX[prec]
    filt = filters(L, P, N, lam, nu, J0, J0p, prec) if filt is None else filt
    ell = np.arange(L).astype(rt)
    wphi_hat = z_forward(W_phi, L, P, tau, prec)
    flmp = np.einsum("plm,pl->plm", wphi_hat, np.sqrt(4 * S.pi(prec) / (2 * ell + 1))[None, :] * filt["phi"])
    for j in range(J0, filt["J"] + 1):
        for jp in range(J0p, filt["Jp"] + 1):
            Lj = S.bandlimit_of_scale(j, L, lam, True)
            Pj = S.bandlimit_of_scale(jp, P, nu, True)
            psi = psi_scale(filt, j, jp, J0, J0p, prec)
            ns = S._active_n(psi.reshape(-1, psi.shape[-1]))
            W = W_psi[(j, jp)]
            what_r = np.stack([S.wigner_forward(W[i], Lj, N, prec, ns) for i in range(Pj)])  # D per shell
            what = laguerre_forward(what_r, Pj, tau, prec)               # K on the P_j' grid  (Q = K D)
            full = np.zeros((P, 2 * N - 1, L, 2 * L - 1), dtype=ct)
            full[:Pj] = S._pad_lm(what, Lj, L)
            flmp = flmp + np.einsum("pnlm,pln->plm", full, psi)          # Psi^dagger
    return flmp


def synthesis(W_phi, W_psi, L, P, N, lam, nu, J0, J0p, tau, prec="f80", filt=None):
    """Algorithm 2 'Synthesis wavelet transform'."""
    flmp = synthesis_to_flmp(W_phi, W_psi, L, P, N, lam, nu, J0, J0p, tau, prec, filt)
    return z_inverse(flmp, L, P, tau, prec)
