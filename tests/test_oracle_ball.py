"""Pins for oracle/ball.py (CPU only): Gauss-Laguerre moments, closed forms, scipy's Laguerre
polynomials, orthonormality, the (l,p) admissibility identity, reduction to the sphere, round trip."""
import math

import numpy as np
import pytest
import scipy.special as sc

from oracle import ball as B
from oracle import sphere as S
from paper_2402_01282_b200 import inputs as I

LD = np.longdouble


@pytest.mark.parametrize("P", [1, 2, 7, 16, 40])
def test_gauss_laguerre_moments(P):
    """sum_i w_i x_i^k = Gamma(k+3) for k <= 2P-1 (weight x^2 e^-x, R8).  radial_nodes returns
    q_i = tau^3 w_i e^{x_i}, so w_i = q_i e^{-x_i} at tau = 1."""
    r, q = B.radial_nodes(P, 1.0)
    w = q * np.exp(-r)
    for k in range(0, 2 * P):
        got = np.sum(w * r ** k)
        assert abs(float(got) / math.gamma(k + 3) - 1) < 1e-15
    # closed-form weight formula against scipy's eigen-solver weights
    xs, ws = sc.roots_genlaguerre(P, 2)
    assert np.abs(r.astype(float) - xs).max() < 1e-11 * max(1, xs.max())
    assert np.abs(w.astype(float) / ws - 1).max() < 1e-9


@pytest.mark.parametrize("tau", [1.0, 0.5, 2.5])
def test_laguerre_basis_closed_form_scipy_and_orthonormality(tau):
    P = 24
    r, q = B.radial_nodes(P, tau)
    K = B.laguerre_basis(P, r, tau)
    # K_0(r) = e^{-r/2tau} / sqrt(2 tau^3)   (Eq. 6 with L_0 = 1)
    assert np.abs(K[0] - np.exp(-r / (2 * LD(tau))) / np.sqrt(2 * LD(tau) ** 3)).max() < 1e-18
    rf = r.astype(float)
    for p in range(P):
        ref = (math.sqrt(1.0 / ((p + 1) * (p + 2))) * tau ** -1.5 * np.exp(-rf / (2 * tau))
               * sc.eval_genlaguerre(p, 2, rf / tau))
        assert np.abs(K[p].astype(float) - ref).max() < 1e-12 * max(1.0, np.abs(ref).max())
    # int r^2 K_p K_q dr = delta_pq  by the quadrature of Eq. 7
    G = np.einsum("pi,i,qi->pq", K, q, K)
    assert np.abs(G - np.eye(P)).max() < 1e-16


def test_laguerre_round_trip_on_reduced_grid():
    """A radially band-limited function (p < 8) survives K^-1 on an 8-node grid followed by K (Eqs. 7-8)."""
    rng = np.random.default_rng(0)
    fp = rng.standard_normal((8, 3)) + 1j * rng.standard_normal((8, 3))
    fr = B.laguerre_inverse(fp, 8, 1.3)
    assert np.abs(B.laguerre_forward(fr, 8, 1.3) - fp).max() < 1e-17
    # and is the same function as on a 20-node grid: compare through a direct evaluation of Eq. 8
    r20, _ = B.radial_nodes(20, 1.3)
    direct = sum(fp[p][None, :] * B.laguerre_basis(8, r20, 1.3)[p][:, None] for p in range(8))
    assert np.abs(B.laguerre_inverse(fp, 20, 1.3) - direct).max() < 1e-17


@pytest.mark.parametrize("L,P,N,lam,nu,J0,J0p", [(16, 16, 3, 2, 2, 0, 0), (16, 16, 2, 2, 2, 1, 0), (20, 12, 4, 3, 2, 1, 1)])
def test_ball_admissibility(L, P, N, lam, nu, J0, J0p):
    """Eq. 36: 4pi/(2l+1)|Phi_l0p|^2 + 8pi^2/(2l+1) sum_{n,j,j'} |Psi^{jj'}_lnp|^2 = 1 for all l, p."""
    filt = B.filters(L, P, N, lam, nu, J0, J0p)
    ell = np.arange(L).astype(LD)
    pi = S.pi("f80")
    tot = (4 * pi / (2 * ell + 1))[None, :] * filt["phi"] ** 2
    for j in range(J0, filt["J"] + 1):
        for jp in range(J0p, filt["Jp"] + 1):
            psi = B.psi_scale(filt, j, jp, J0, J0p)
            tot = tot + (8 * pi ** 2 / (2 * ell + 1))[None, :] * np.sum(np.abs(psi) ** 2, axis=2)
    assert np.abs(tot - 1).max() < 1e-17


def test_scaling_filter_equals_printed_cases_of_eq_A10():
    """R9: sqrt(a+b-ab) equals eta_nu(p/nu^J0') where a = 0, eta_lam(l/lam^J0) where b = 0 (Eq. A10)."""
    L, P, lam, nu, J0, J0p = 32, 32, 2, 2, 2, 3
    filt = B.filters(L, P, 1, lam, nu, J0, J0p)
    _, eta_l = S.kappa(L, lam, J0)
    _, eta_p = S.kappa(P, nu, J0p)
    ell = np.arange(L).astype(LD)
    c = np.sqrt((2 * ell + 1) / (4 * S.pi("f80")))
    for l in range(L):
        for p in range(P):
            if eta_l[l] == 0:
                assert abs(filt["phi"][p, l] - c[l] * eta_p[p]) < 1e-18
            if eta_p[p] == 0:
                assert abs(filt["phi"][p, l] - c[l] * eta_l[l]) < 1e-18


def test_ball_with_radially_trivial_input_reduces_to_sphere():
    """If f_{lmp} = f_lm delta_{p0} then Z^-1 f = K_0(r) * (Y^-1 f_lm) shell by shell."""
    L, P, tau = 8, 6, 1.0
    flm = I.flm_complex(L, 3, 1, "white")[0]
    flmp = np.zeros((P, L, 2 * L - 1), dtype=complex)
    flmp[0] = flm
    f = B.z_inverse(flmp, L, P, tau)
    r, _ = B.radial_nodes(P, tau)
    fs = S.sht_inverse(flm, L)
    K0 = np.exp(-r / 2) / np.sqrt(LD(2))
    assert np.abs(f - K0[:, None, None] * fs[None]).max() < 1e-17


@pytest.mark.parametrize("L,P,N,J0,J0p", [(8, 8, 2, 0, 0), (8, 4, 3, 1, 0), (6, 9, 1, 0, 1)])
def test_ball_round_trip(L, P, N, J0, J0p):
    flmp = I.flmp_complex(L, P, 5)
    f = B.z_inverse(flmp, L, P, 1.0)
    assert np.abs(B.z_forward(f, L, P, 1.0) - flmp).max() < 1e-16
    W_phi, W_psi = B.analysis(f, L, P, N, 2, 2, J0, J0p, 1.0)
    f2 = B.synthesis(W_phi, W_psi, L, P, N, 2, 2, J0, J0p, 1.0)
    assert np.abs(f2 - f).max() / np.abs(f).max() < 1e-16
    for (j, jp), W in W_psi.items():
        assert W.shape == (S.bandlimit_of_scale(jp, P, 2, True), 2 * N - 1,
                           S.bandlimit_of_scale(j, L, 2, True), 2 * S.bandlimit_of_scale(j, L, 2, True) - 1)


# ---- Wigner-Laguerre transform Q = K D (Eqs. 24-25; reading R18) ----
def _random_fhat(L, P, N, seed):
    """Band-limited coefficients f^l_{mnp}: |m| <= l, |n| <= min(N-1, l)."""
    rng = np.random.default_rng(seed)
    fh = rng.standard_normal((2 * N - 1, P, L, 2 * L - 1)) + 1j * rng.standard_normal((2 * N - 1, P, L, 2 * L - 1))
    ell = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    fh *= (np.abs(m) <= ell)[None, None]
    for ni in range(2 * N - 1):
        fh[ni] *= (abs(ni - (N - 1)) <= np.arange(L))[None, :, None]
    return fh


def test_wigner_laguerre_inverse_is_the_literal_sum_of_eq_25():
    """q_inverse at sampled points h = (r_i, alpha, beta, gamma) against Eq. 25 written out: sum over (l, m, n, p) of
    (2l+1)/(8 pi^2) f^l_{mnp} K_p(r) d^l_{mn}(beta) e^{i(m alpha + n gamma)} (D^* of Eq. 47), with K_p from its own
    closed form (scipy genlaguerre) and d^l_{mn} from the long-double recursion pinned in test_oracle_sphere."""
    from scipy.special import eval_genlaguerre, gammaln
    L, P, N, tau = 5, 4, 3, 1.3
    fh = _random_fhat(L, P, N, 3)
    f = B.q_inverse(fh, L, P, N, tau, "f80")
    r, _ = B.radial_nodes(P, tau, "f80")
    th = S.mw_thetas(L, "f80").astype(float)
    ph = S.mw_phis(L, "f80").astype(float)
    for (i, g, t, a) in [(0, 0, 0, 0), (1, 3, 2, 5), (3, 4, 4, 8), (2, 1, 3, 2)]:
        gam = 2 * np.pi * g / (2 * N - 1)
        tot = 0
        for p in range(P):
            x = float(r[i]) / tau
            Kp = np.exp(0.5 * (gammaln(p + 1) - gammaln(p + 3))) * tau ** -1.5 * np.exp(-x / 2) * eval_genlaguerre(p, 2, x)
            for n in range(-(N - 1), N):
                for m in range(-(L - 1), L):
                    d = S.wigner_d(L, m, n, LD(th[t]), "f80").astype(float)
                    for l in range(max(abs(m), abs(n)), L):
                        tot += (2 * l + 1) / (8 * np.pi ** 2) * fh[n + N - 1, p, l, m + L - 1] * Kp * d[l] \
                            * np.exp(1j * (m * ph[a] + n * gam))
        assert abs(complex(f[i, g, t, a]) - tot) < 1e-12 * max(1.0, abs(tot))


def test_wigner_laguerre_forward_inverts_the_inverse():
    """Q Q^-1 = identity on band-limited coefficients (orthogonality and completeness behind Eq. 25), odd and even N."""
    for (L, P, N, tau) in ((6, 5, 3, 1.0), (5, 3, 2, 0.7), (4, 6, 4, 2.0)):
        fh = _random_fhat(L, P, N, L + P + N)
        back = B.q_forward(B.q_inverse(fh, L, P, N, tau, "f80"), L, P, N, tau, "f80")
        assert np.abs(back - fh).max() < 1e-13 * np.abs(fh).max()


def test_wigner_laguerre_reduces_to_its_factors():
    """N = 1: Q is the spherical-Laguerre transform Z (D with n = 0 is the SHT up to the 2 pi of the gamma integral and
    sqrt(4pi/(2l+1)): D^l_{m0} = sqrt(4pi/(2l+1)) Y*_{lm}); a radially constant-in-p input reduces K to one column."""
    L, P, tau = 6, 4, 1.0
    rng = np.random.default_rng(5)
    flmp = rng.standard_normal((P, L, 2 * L - 1)) + 1j * rng.standard_normal((P, L, 2 * L - 1))
    flmp *= (np.abs(np.arange(-(L - 1), L))[None, :] <= np.arange(L)[:, None])[None]
    f = B.z_inverse(flmp, L, P, tau, "f80")                     # [P][L][2L-1], a function on the ball
    qh = B.q_forward(f[:, None], L, P, 1, tau, "f80")[0]         # the same function, constant in gamma
    ell = np.arange(L)
    expect = 2 * np.pi * np.sqrt(4 * np.pi / (2 * ell + 1))[None, :, None] * flmp
    # int f D^l_{m0} = 2 pi sqrt(4pi/(2l+1)) int f Y*_{lm}: Y*_{lm} = (-1)^m Y_{l,-m} is what D^l_{m0} = d^l_{m0} e^{-i m alpha} gives
    assert np.abs(qh - expect).max() < 1e-12 * np.abs(expect).max()
