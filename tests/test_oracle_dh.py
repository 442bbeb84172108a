"""CPU pins of the oracle's Driscoll-Healy sampling (reading R19): the quadrature is exact on
cosine polynomials of degree < 2L, closed-form Y_lm sampled on the grid project onto single coefficients, forward o inverse
is the identity, the coefficients of a band-limited function do not depend on the sampling it was given in, and the
wavelet transform reconstructs exactly."""
import numpy as np
import pytest
import scipy.special as sc

from oracle import sphere as S
from paper_2402_01282_b200 import inputs

LD = np.longdouble


@pytest.mark.parametrize("L", [1, 2, 5, 16, 33])
def test_dh_quadrature_is_exact_on_cosine_polynomials_below_degree_2L(L):
    """sum_t q_t cos(k theta_t) = int_0^pi cos(k theta) sin(theta) dtheta = 2/(1-k^2) for even k, 0 for odd k, k < 2L;
    and it is NOT exact at k = 4L (the first alias of k = 0 on the grid), so the rule is no finer than claimed."""
    th, q = S.dh_thetas(L, "f80"), S.dh_weights(L, "f80")
    for k in range(2 * L):
        exact = 2.0 / (1.0 - k * k) if k % 2 == 0 else 0.0
        assert abs(float((q * np.cos(k * th)).sum()) - exact) < 1e-15 * max(1, L)
    assert abs(float((q * np.cos(4 * L * th)).sum())) > 1.0
    assert th.size == 2 * L and np.all(np.diff(th.astype(float)) > 0) and 0 < th[0] and th[-1] < np.pi


def test_closed_form_harmonics_sampled_on_the_dh_grid_project_onto_single_coefficients():
    L = 12
    th = S.dh_thetas(L, "f64")
    ph = S.mw_phis(L, "f64")
    T, P = np.meshgrid(th, ph, indexing="ij")
    for (l, m) in ((0, 0), (1, 0), (1, 1), (2, 0), (3, -2), (7, 5), (11, -11)):
        f = sc.sph_harm_y(l, m, T, P)
        flm = S.sht_forward(f, L, "f80", sampling="dh")
        expect = np.zeros((L, 2 * L - 1), dtype=complex)
        expect[l, m + L - 1] = 1.0
        assert np.abs(flm.astype(complex) - expect).max() < 1e-13
    f = np.sqrt(5 / (16 * np.pi)) * (3 * np.cos(T) ** 2 - 1)            # Y_20 in closed form
    assert abs(complex(S.sht_forward(f, L, "f80", sampling="dh")[2, L - 1]) - 1) < 1e-14
    back = S.sht_inverse(expect, L, "f80", sampling="dh")
    assert np.abs(back.astype(complex) - sc.sph_harm_y(11, -11, T, P)).max() < 1e-14


@pytest.mark.parametrize("L", [1, 2, 9, 32])
def test_dh_forward_inverts_inverse_and_agrees_with_the_mw_transform(L):
    flm = inputs.flm_complex(L, 60 + L, 1)[0]
    f_dh = S.sht_inverse(flm, L, "f80", sampling="dh")
    assert f_dh.shape == (2 * L, 2 * L - 1)
    back = S.sht_forward(f_dh, L, "f80", sampling="dh")
    assert np.abs(back - flm).max() < 1e-13 * max(np.abs(flm).max(), 1e-300)
    # the same function sampled on the MW grid has the same coefficients (independent code path: R3 reweighting)
    f_mw = S.sht_inverse(flm, L, "f80")
    assert np.abs(S.sht_forward(f_mw, L, "f80") - back).max() < 1e-13 * max(np.abs(flm).max(), 1e-300)


@pytest.mark.parametrize("L,N,lam,J0,real", [(8, 3, 2.0, 0, False), (12, 2, 2.0, 1, True), (16, 4, 3.0, 1, False)])
def test_dh_wavelet_transform_reconstructs_and_shares_harmonic_content_with_mw(L, N, lam, J0, real):
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, 70 + L, 1)[0]
    f = S.sht_inverse(flm, L, "f80", sampling="dh")
    filt = S.filters(L, N, lam, J0, "f80")
    phi, psi = S.analysis(f, L, N, lam, J0, True, "f80", filt, sampling="dh")
    for j, w in psi.items():
        Lj = S.bandlimit_of_scale(j, L, lam, True)
        assert w.shape == (2 * N - 1, 2 * Lj, 2 * Lj - 1)
        if real:
            assert np.abs(w.imag).max() <= 1e-14 * max(np.abs(w).max(), 1e-300)
    back = S.synthesis(phi, psi, L, N, lam, J0, True, "f80", filt, sampling="dh")
    assert np.abs(back - f).max() < 1e-13 * np.abs(f).max()
    # Wigner coefficients recovered from the DH samples of a scale equal those recovered from its MW samples
    _, psi_mw = S.analysis_from_flm(flm, L, N, lam, J0, True, "f80", filt)
    J = max(psi)
    Lj = S.bandlimit_of_scale(J, L, lam, True)
    a = S.wigner_forward(psi[J], Lj, N, "f80", sampling="dh")
    b = S.wigner_forward(psi_mw[J], Lj, N, "f80")
    assert np.abs(a - b).max() < 1e-13 * max(np.abs(b).max(), 1e-300)
