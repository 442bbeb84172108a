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


def test_ball_adjoint_entries_inner_product_identity():
    """Ball: sampled entries of A^H y and S^H g against <A x, y> and <S w, g> with x / w supported on the sampled
    entries and A x, S w computed by applying the oracle directly."""
    from oracle import ball as OB
    L, P, N, lam, nu, J0, tau = 5, 3, 2, 2.0, 2.0, 0, 1.0
    rng = np.random.default_rng(3)
    nvox = P * L * (2 * L - 1)
    T_phi, T_psi = OB.analysis(np.zeros((P, L, 2 * L - 1), dtype=np.clongdouble), L, P, N, lam, nu, J0, J0, tau, "f80")
    Y_phi = _rand_c(rng, T_phi.shape)
    Y_psi = {k: _rand_c(rng, v.shape) for k, v in T_psi.items()}
    vox = sorted(rng.choice(nvox, size=6, replace=False).tolist())
    x = np.zeros(nvox, dtype=np.clongdouble)
    x[vox] = _rand_c(rng, len(vox))
    W_phi, W_psi = OB.analysis(x.reshape(P, L, 2 * L - 1), L, P, N, lam, nu, J0, J0, tau, "f80")
    lhs = np.vdot(ADJ.ball_pack(W_phi, W_psi), ADJ.ball_pack(Y_phi, Y_psi))
    rhs = np.vdot(x[vox], ADJ.ball_analysis_adjoint_entries(Y_phi, Y_psi, vox, L, P, N, lam, nu, J0, J0, tau, "f80"))
    assert abs(lhs - rhs) < 1e-15 * abs(lhs) * 50
    ncoef = ADJ.ball_pack(T_phi, T_psi).size
    cs = sorted(rng.choice(ncoef, size=8, replace=False).tolist())
    w = np.zeros(ncoef, dtype=np.clongdouble)
    w[cs] = _rand_c(rng, len(cs))
    o = T_phi.size
    V_phi, V_psi = w[:o].reshape(T_phi.shape), {}
    for k in sorted(T_psi):
        V_psi[k] = w[o:o + T_psi[k].size].reshape(T_psi[k].shape)
        o += T_psi[k].size
    g = _rand_c(rng, (P, L, 2 * L - 1))
    lhs = np.vdot(OB.synthesis(V_phi, V_psi, L, P, N, lam, nu, J0, J0, tau, "f80"), g)
    rhs = np.vdot(w[cs], ADJ.ball_synthesis_adjoint_entries(g, (T_phi, T_psi), cs, L, P, N, lam, nu, J0, J0, tau, "f80"))
    assert abs(lhs - rhs) < 1e-15 * abs(lhs) * 50
