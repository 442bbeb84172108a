"""CPU pins of oracle/adjoint.py: the adjoint of the oracle's analysis A and synthesis S is the
conjugate transpose of the matrix of the map.  Pinned by what defines an adjoint and by what the paper's transform
fixes: <A x, y> = <x, A^H y> with A x computed by applying the oracle directly (a transposed or unconjugated matrix, or
a block packed in the wrong order, fails it), exact reconstruction S A = I on band-limited signals carried over to the
adjoints (A^H S^H g = g for band-limited g's pixel-space dual), and the explicit 1 x 1 case L = 1."""
import numpy as np
import pytest

from oracle import adjoint as ADJ
from oracle import sphere as S
from paper_2402_01282_b200 import inputs

CASES = [(8, 2, 2.0, 0, True), (6, 3, 2.0, 1, True), (7, 1, 3.0, 0, False)]


def _rand_c(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _rand_coeffs(rng, L, N, lam, J0, mr):
    Y_phi, Y_psi = None, {}
    for key, shp in ADJ.shapes(L, N, lam, J0, mr):
        a = _rand_c(rng, shp)
        if key < 0:
            Y_phi = a
        else:
            Y_psi[key] = a
    return Y_phi, Y_psi


@pytest.mark.parametrize("L,N,lam,J0,mr", CASES)
def test_analysis_adjoint_inner_product_identity(L, N, lam, J0, mr):
    rng = np.random.default_rng(10 + L)
    x = _rand_c(rng, (L, 2 * L - 1))          # any pixel array, band-limited or not: A is linear on all of them
    Y_phi, Y_psi = _rand_coeffs(rng, L, N, lam, J0, mr)
    W_phi, W_psi = S.analysis(x, L, N, lam, J0, mr, "f80")
    lhs = np.vdot(ADJ.pack(W_phi, W_psi, L, N, lam, J0, mr), ADJ.pack(Y_phi, Y_psi, L, N, lam, J0, mr))
    rhs = np.vdot(x, ADJ.analysis_adjoint(Y_phi, Y_psi, L, N, lam, J0, mr, "f80"))
    assert abs(lhs - rhs) < 1e-15 * abs(lhs) * 50


@pytest.mark.parametrize("L,N,lam,J0,mr", CASES)
def test_synthesis_adjoint_inner_product_identity(L, N, lam, J0, mr):
    rng = np.random.default_rng(20 + L)
    g = _rand_c(rng, (L, 2 * L - 1))
    Y_phi, Y_psi = _rand_coeffs(rng, L, N, lam, J0, mr)
    f = S.synthesis(Y_phi, Y_psi, L, N, lam, J0, mr, "f80")
    lhs = np.vdot(f, g)
    Z_phi, Z_psi = ADJ.synthesis_adjoint(g, L, N, lam, J0, mr, "f80")
    rhs = np.vdot(ADJ.pack(Y_phi, Y_psi, L, N, lam, J0, mr), ADJ.pack(Z_phi, Z_psi, L, N, lam, J0, mr))
    assert abs(lhs - rhs) < 1e-15 * abs(lhs) * 50


def test_adjoints_inherit_exact_reconstruction():
    """S A f = f for band-limited f (Eq. 30), so <S A f, g> = <f, g> = <f, A^H S^H g> for every g: the
    component of A^H S^H g - g along any band-limited pixel array vanishes."""
    L, N, lam, J0, mr = 8, 2, 2.0, 0, True
    rng = np.random.default_rng(5)
    g = _rand_c(rng, (L, 2 * L - 1))
    Z_phi, Z_psi = ADJ.synthesis_adjoint(g, L, N, lam, J0, mr, "f80")
    h = ADJ.analysis_adjoint(Z_phi, Z_psi, L, N, lam, J0, mr, "f80")
    for seed in range(3):
        f = S.sht_inverse(inputs.flm_complex(L, 300 + seed, 1)[0], L, "f80")
        assert abs(np.vdot(f, h - g)) < 1e-14 * np.linalg.norm(f) * np.linalg.norm(g)
    assert np.linalg.norm(h - g) > 1e-3 * np.linalg.norm(g)   # but A^H S^H is not the identity off the band-limit


def test_one_pixel_case_is_complex_conjugation():
    """L = 1: one pixel, every block one sample; A is a column of numbers a_c and A^H y = sum conj(a_c) y_c."""
    L, N, lam, J0, mr = 1, 1, 2.0, 0, True
    one = np.ones((1, 1), dtype=np.clongdouble)
    W_phi, W_psi = S.analysis(one * (0.3 + 0.7j), L, N, lam, J0, mr, "f80")
    a = ADJ.pack(W_phi, W_psi, L, N, lam, J0, mr) / (0.3 + 0.7j)
    rng = np.random.default_rng(1)
    Y_phi, Y_psi = _rand_coeffs(rng, L, N, lam, J0, mr)
    y = ADJ.pack(Y_phi, Y_psi, L, N, lam, J0, mr)
    got = ADJ.analysis_adjoint(Y_phi, Y_psi, L, N, lam, J0, mr, "f80")
    assert abs(got[0, 0] - np.sum(np.conj(a) * y)) < 1e-17 * (1 + abs(got[0, 0])) * 100
