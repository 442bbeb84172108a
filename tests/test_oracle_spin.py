"""CPU pins of the oracle's spin-s harmonic transforms (reading R2, Goldberg et al. 1967 convention -- the paper prints no formula; its Eq. 1, is the transformation law: sY_lm = (-1)^s sqrt((2l+1)/4pi) D^{l*}_{m,-s}):
textbook closed forms of the spin-weighted harmonics (Goldberg et al. 1967 phase, the one Eq. 1 reproduces), their
orthonormality through the exact MW quadrature, exact forward o inverse on band-limited spin signals, and exact
reconstruction of the spin wavelet transform."""
import numpy as np
import pytest

from oracle import sphere as S


def _grid(L):
    th = np.asarray(S.mw_thetas(L, "f80"), dtype=np.float64)
    ph = np.asarray(S.mw_phis(L, "f80"), dtype=np.float64)
    return th[:, None], ph[None, :]


def _delta(L, l, m):
    flm = np.zeros((L, 2 * L - 1), dtype=np.clongdouble)
    flm[l, m + L - 1] = 1
    return flm


CLOSED = [
    # spin, l, m, function of (theta, phi)
    (1, 1, 0, lambda t, p: np.sqrt(3 / (8 * np.pi)) * np.sin(t) + 0j * p),
    (1, 1, 1, lambda t, p: -np.sqrt(3 / (16 * np.pi)) * (1 - np.cos(t)) * np.exp(1j * p)),
    (1, 1, -1, lambda t, p: -np.sqrt(3 / (16 * np.pi)) * (1 + np.cos(t)) * np.exp(-1j * p)),
    (-1, 1, 0, lambda t, p: -np.sqrt(3 / (8 * np.pi)) * np.sin(t) + 0j * p),
    (2, 2, 0, lambda t, p: np.sqrt(15 / (32 * np.pi)) * np.sin(t) ** 2 + 0j * p),
    (2, 2, 2, lambda t, p: np.sqrt(5 / (64 * np.pi)) * (1 - np.cos(t)) ** 2 * np.exp(2j * p)),
    (2, 2, -2, lambda t, p: np.sqrt(5 / (64 * np.pi)) * (1 + np.cos(t)) ** 2 * np.exp(-2j * p)),
]


@pytest.mark.parametrize("spin,l,m,fn", CLOSED)
def test_spin_weighted_harmonics_closed_forms(spin, l, m, fn):
    L = 5
    t, p = _grid(L)
    got = np.asarray(S.sht_inverse(_delta(L, l, m), L, "f80", spin=spin), dtype=np.complex128)
    assert np.abs(got - fn(t, p)).max() < 1e-15


@pytest.mark.parametrize("spin", [1, -1, 2, -2, 3])
def test_spin_forward_inverts_inverse_and_harmonics_are_orthonormal(spin):
    L = 9
    rng = np.random.default_rng(spin + 10)
    flm = (rng.standard_normal((L, 2 * L - 1)) + 1j * rng.standard_normal((L, 2 * L - 1))).astype(np.clongdouble)
    for l in range(L):
        for m in range(-(L - 1), L):
            if abs(m) > l or l < abs(spin):
                flm[l, m + L - 1] = 0
    f = S.sht_inverse(flm, L, "f80", spin=spin)
    back = S.sht_forward(f, L, "f80", spin=spin)
    assert np.abs(back - flm).max() < 1e-16 * 50
    # a single harmonic projects onto itself only
    one = S.sht_forward(S.sht_inverse(_delta(L, 4, -2), L, "f80", spin=spin), L, "f80", spin=spin)
    assert abs(one[4, -2 + L - 1] - 1) < 1e-17 * 100
    one[4, -2 + L - 1] = 0
    assert np.abs(one).max() < 1e-17 * 100
    # below l = |s| there are no spin-s harmonics
    assert np.abs(S.sht_inverse(_delta(L, abs(spin) - 1, 0), L, "f80", spin=spin)).max() == 0


@pytest.mark.parametrize("L,N,lam,J0,mr,spin", [(8, 2, 2.0, 0, True, 2), (9, 3, 2.0, 1, True, -1), (8, 1, 2.0, 0, False, 1)])
def test_spin_wavelet_transform_reconstructs_exactly(L, N, lam, J0, mr, spin):
    rng = np.random.default_rng(L + spin)
    flm = (rng.standard_normal((L, 2 * L - 1)) + 1j * rng.standard_normal((L, 2 * L - 1))).astype(np.clongdouble)
    for l in range(L):
        for m in range(-(L - 1), L):
            if abs(m) > l or l < abs(spin):
                flm[l, m + L - 1] = 0
    f = S.sht_inverse(flm, L, "f80", spin=spin)
    W_phi, W_psi = S.analysis(f, L, N, lam, J0, mr, "f80", spin=spin)
    back = S.synthesis(W_phi, W_psi, L, N, lam, J0, mr, "f80", spin=spin)
    assert np.abs(back - f).max() < 1e-15 * np.abs(f).max()
