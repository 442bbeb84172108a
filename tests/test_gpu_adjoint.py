"""GPU parity tests of the adjoint transforms: s2w_plan_forward_adjoint / s2w_plan_inverse_adjoint
through the C ABI against oracle/adjoint.py (the conjugate transpose of the oracle's own analysis / synthesis matrix)
element by element on the same seeded inputs, and the defining identity <A x, y> = <x, A^H y> at sizes the oracle's
matrix cannot reach.  Tolerance as for the forward transforms: 1e-11 relative max per block."""
import numpy as np
import pytest

from oracle import adjoint as ADJ

pytestmark = pytest.mark.gpu

TOL = 1e-11


def _api():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2402_01282_b200 import api
    return torch, api


def _relmax(a, b):
    den = np.abs(b).max()
    num = np.abs(a - b).max()
    return num if den == 0 else num / den


def _rand_c(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _pack_for_plan(plan, Y_phi, Y_psi):
    packed = np.zeros((1, plan.coeff_elems), dtype=np.complex128)
    nr, ng, nt, npx, off = plan.scale_shape(-1)
    packed[0, off:off + nt * npx] = np.asarray(Y_phi, dtype=np.complex128).ravel()
    for j, a in Y_psi.items():
        nr, ng, nt, npx, off = plan.scale_shape(j)
        packed[0, off:off + ng * nt * npx] = np.asarray(a, dtype=np.complex128).ravel()
    return packed


CASES = [(8, 2, 2.0, 0, True), (6, 3, 2.0, 1, True), (7, 1, 3.0, 0, False), (10, 4, 2.0, 0, True)]


@pytest.mark.parametrize("L,N,lam,J0,mr", CASES)
def test_adjoints_match_oracle(L, N, lam, J0, mr):
    torch, api = _api()
    rng = np.random.default_rng(700 + L)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, False, 1)
    # A^H
    Y_phi, Y_psi = None, {}
    for key, shp in ADJ.shapes(L, N, lam, J0, mr):
        a = _rand_c(rng, shp)
        if key < 0:
            Y_phi = a
        else:
            Y_psi[key] = a
    ref = ADJ.analysis_adjoint(Y_phi, Y_psi, L, N, lam, J0, mr, "f80").astype(np.complex128)
    got = plan.forward_adjoint(torch.from_numpy(_pack_for_plan(plan, Y_phi, Y_psi)).cuda()).cpu().numpy()
    assert _relmax(got.reshape(L, 2 * L - 1), ref) < TOL
    # S^H
    g = _rand_c(rng, (L, 2 * L - 1))
    Z_phi, Z_psi = ADJ.synthesis_adjoint(g, L, N, lam, J0, mr, "f80")
    z = plan.inverse_adjoint(torch.from_numpy(np.ascontiguousarray(g.reshape(1, -1))).cuda())
    scal, scales = plan.split(z)
    assert _relmax(scal[0].cpu().numpy(), Z_phi.astype(np.complex128)) < TOL
    for j, refj in Z_psi.items():
        gotj = scales[(j, 0)][0].cpu().numpy()
        assert gotj.shape == refj.shape
        if np.abs(refj).max() == 0:
            assert np.abs(gotj).max() == 0
        else:
            assert _relmax(gotj, refj.astype(np.complex128)) < TOL, j
    plan.close()


@pytest.mark.parametrize("L,N,lam,J0,mr,batch", [(64, 3, 2.0, 1, True, 2), (300, 3, 2.0, 2, True, 1), (130, 5, 2.0, 3, False, 1),
                                                 (1024, 2, 2.0, 8, True, 1)])
def test_inner_product_identities_at_larger_sizes(L, N, lam, J0, mr, batch):
    """<A x, y> = <x, A^H y> and <S y, x> = <y, S^H x> for random (not band-limited) x and y: several ring groups per
    warp, ragged groups, the Toeplitz/Hankel reweighting and the ring-by-ring kernels of the large grids."""
    torch, api = _api()
    gen = torch.Generator(device="cuda").manual_seed(L + N)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, False, batch)
    x = torch.randn(batch, plan.signal_elems, dtype=torch.complex128, device="cuda", generator=gen)
    y = torch.randn(batch, plan.coeff_elems, dtype=torch.complex128, device="cuda", generator=gen)
    Ax, Ahy = plan.forward(x), plan.forward_adjoint(y)
    lhs, rhs = torch.vdot(Ax.flatten(), y.flatten()), torch.vdot(x.flatten(), Ahy.flatten())
    assert abs(lhs - rhs) < 1e-12 * Ax.norm() * y.norm()
    Sy, Shx = plan.inverse(y), plan.inverse_adjoint(x)
    lhs, rhs = torch.vdot(Sy.flatten(), x.flatten()), torch.vdot(y.flatten(), Shx.flatten())
    assert abs(lhs - rhs) < 1e-12 * Sy.norm() * x.norm()
    # a second call replays the captured graph (the harmonic sums accumulate by atomics: equal up to rounding order)
    assert float((plan.inverse_adjoint(x) - Shx).abs().max()) < 1e-13 * float(Shx.abs().max())
    plan.close()


@pytest.mark.parametrize("L,N,lam,J0,mr", [(8, 2, 2.0, 0, True), (9, 3, 2.0, 1, True), (7, 4, 2.0, 0, False)])
def test_real_plan_adjoints_match_oracle(L, N, lam, J0, mr):
    """Real-signal plans (m >= 0 kernels): the matrix of A is real in the pixel basis, so its adjoint on a real
    cotangent is the oracle's A^H applied to it (imaginary part zero); the same for S."""
    torch, api = _api()
    rng = np.random.default_rng(800 + L)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, True, 1)
    Y_phi, Y_psi = None, {}
    for key, shp in ADJ.shapes(L, N, lam, J0, mr):
        a = rng.standard_normal(shp)
        if key < 0:
            Y_phi = a
        else:
            Y_psi[key] = a
    ref = ADJ.analysis_adjoint(Y_phi, Y_psi, L, N, lam, J0, mr, "f80")
    assert np.abs(ref.imag).max() < 1e-15 * np.abs(ref).max()
    packed = _pack_for_plan(plan, Y_phi, Y_psi).real.copy()
    got = plan.forward_adjoint(torch.from_numpy(packed).cuda()).cpu().numpy()
    assert _relmax(got.reshape(L, 2 * L - 1), ref.real.astype(np.float64)) < TOL
    g = rng.standard_normal((L, 2 * L - 1))
    Z_phi, Z_psi = ADJ.synthesis_adjoint(g, L, N, lam, J0, mr, "f80")
    z = plan.inverse_adjoint(torch.from_numpy(np.ascontiguousarray(g.reshape(1, -1))).cuda())
    scal, scales = plan.split(z)
    assert _relmax(scal[0].cpu().numpy(), Z_phi.real.astype(np.float64)) < TOL
    for j, refj in Z_psi.items():
        assert np.abs(refj.imag).max() <= 1e-15 * max(np.abs(refj).max(), 1e-300)
        gotj = scales[(j, 0)][0].cpu().numpy()
        if np.abs(refj).max() == 0:
            assert np.abs(gotj).max() == 0
        else:
            assert _relmax(gotj, refj.real.astype(np.float64)) < TOL, j
    plan.close()


@pytest.mark.parametrize("L,N,lam,J0,mr,batch", [(96, 6, 2.0, 3, True, 1), (600, 5, 2.0, 6, True, 2), (1024, 5, 2.0, 9, True, 4)])
def test_real_plan_inner_product_identities(L, N, lam, J0, mr, batch):
    """<A x, y> = <x, A^T y>, <S y, x> = <y, S^T x> on real plans: ring-pair (alpha, gamma) kernels, accumulating and
    parked gamma planes, the metric configuration's top scales (L = 1024, N = 5, batch 4, J0 = 9)."""
    torch, api = _api()
    gen = torch.Generator(device="cuda").manual_seed(L + N)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, True, batch)
    x = torch.randn(batch, plan.signal_elems, dtype=torch.float64, device="cuda", generator=gen)
    y = torch.randn(batch, plan.coeff_elems, dtype=torch.float64, device="cuda", generator=gen)
    Ax, Aty = plan.forward(x), plan.forward_adjoint(y)
    assert abs(torch.dot(Ax.flatten(), y.flatten()) - torch.dot(x.flatten(), Aty.flatten())) < 1e-12 * Ax.norm() * y.norm()
    Sy, Stx = plan.inverse(y), plan.inverse_adjoint(x)
    assert abs(torch.dot(Sy.flatten(), x.flatten()) - torch.dot(y.flatten(), Stx.flatten())) < 1e-12 * Sy.norm() * x.norm()
    plan.close()


@pytest.mark.parametrize("L,P,N,lam,nu,J0,tau", [(6, 4, 2, 2.0, 2.0, 0, 1.0), (8, 5, 3, 2.0, 3.0, 1, 0.5)])
def test_ball_adjoints_match_oracle_on_sampled_entries(L, P, N, lam, nu, J0, tau):
    """Ball plans: sampled entries of A^H y and S^H g against the oracle (one oracle transform per entry)."""
    from oracle import ball as OB
    torch, api = _api()
    rng = np.random.default_rng(900 + L)
    plan = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau)
    T_phi, T_psi = OB.analysis(np.zeros((P, L, 2 * L - 1), dtype=np.clongdouble), L, P, N, lam, nu, J0, J0, tau, "f80")
    Y_phi = _rand_c(rng, T_phi.shape)
    Y_psi = {k: _rand_c(rng, v.shape) for k, v in T_psi.items()}
    packed = np.zeros((1, plan.coeff_elems), dtype=np.complex128)
    index_of = {}            # oracle packing index -> plan packing index, block by block
    nr, ng, nt, npx, off = plan.scale_shape(-1)
    packed[0, off:off + nr * nt * npx] = Y_phi.astype(np.complex128).ravel()
    blocks = [(0, off, T_phi.size)]
    o = T_phi.size
    for key in sorted(T_psi):
        nr, ng, nt, npx, off = plan.scale_shape(*key)
        assert (nr, ng, nt, npx) == T_psi[key].shape
        packed[0, off:off + T_psi[key].size] = Y_psi[key].astype(np.complex128).ravel()
        blocks.append((o, off, T_psi[key].size))
        o += T_psi[key].size
    nvox = P * L * (2 * L - 1)
    vox = sorted(rng.choice(nvox, size=24, replace=False).tolist())
    ref = ADJ.ball_analysis_adjoint_entries(Y_phi, Y_psi, vox, L, P, N, lam, nu, J0, J0, tau, "f80")
    got = plan.forward_adjoint(torch.from_numpy(packed).cuda()).cpu().numpy().ravel()
    assert np.abs(got[vox] - ref.astype(np.complex128)).max() < TOL * np.abs(got).max()
    g = _rand_c(rng, (P, L, 2 * L - 1))
    cs = sorted(rng.choice(o, size=40, replace=False).tolist())
    ref = ADJ.ball_synthesis_adjoint_entries(g, (T_phi, T_psi), cs, L, P, N, lam, nu, J0, J0, tau, "f80")
    z = plan.inverse_adjoint(torch.from_numpy(np.ascontiguousarray(g.reshape(1, -1))).cuda()).cpu().numpy().ravel()

    def plan_index(c):
        for o0, off, n in blocks:
            if o0 <= c < o0 + n:
                return off + (c - o0)
        raise AssertionError(c)

    gotc = np.array([z[plan_index(c)] for c in cs])
    assert np.abs(gotc - ref.astype(np.complex128)).max() < TOL * np.abs(z).max()
    plan.close()


@pytest.mark.parametrize("L,P,N,real", [(20, 16, 3, False), (12, 6, 3, True), (128, 128, 3, False)])
def test_ball_inner_product_identities(L, P, N, real):
    """<A x, y> = <x, A^H y>, <S y, x> = <y, S^H x> on ball plans up to BASELINE config 5 (L = P = 128)."""
    torch, api = _api()
    gen = torch.Generator(device="cuda").manual_seed(L + P)
    plan = api.s2ball_plan_create(L, P, N, 2.0, 2.0, 0, 1.0, real=real)
    dt = torch.float64 if real else torch.complex128
    x = torch.randn(1, plan.signal_elems, dtype=dt, device="cuda", generator=gen)
    y = torch.randn(1, plan.coeff_elems, dtype=dt, device="cuda", generator=gen)
    Ax, Ahy = plan.forward(x), plan.forward_adjoint(y)
    assert abs(torch.vdot(Ax.flatten(), y.flatten()) - torch.vdot(x.flatten(), Ahy.flatten())) < 1e-12 * Ax.norm() * y.norm()
    Sy, Shx = plan.inverse(y), plan.inverse_adjoint(x)
    assert abs(torch.vdot(Sy.flatten(), x.flatten()) - torch.vdot(y.flatten(), Shx.flatten())) < 1e-12 * Sy.norm() * x.norm()
    plan.close()


def test_adjoint_argument_errors():
    torch, api = _api()
    plan = api.s2wav_plan_create(8, 2, 2.0, 0, True, False, 1)
    with pytest.raises(ValueError):
        plan.forward_adjoint(torch.zeros(1, plan.coeff_elems - 1, dtype=torch.complex128, device="cuda"))
    assert api.lib().s2w_plan_forward_adjoint(None, None, None, None, None) == -1  # S2W_EINVAL
    plan.close()
