"""GPU parity tests of Driscoll-Healy sampling (S2W_DH, "sampling agnostic"; reading R19):
2L rings per grid, the diagonal Driscoll-Healy quadrature in place of the reweighting operator, the same contraction and
FFT kernels.  Against the oracle's sampling="dh" transforms (pinned in tests/test_oracle_dh.py); tolerances 1e-11 forward,
1e-12 round trip (BASELINE.json)."""
import numpy as np
import pytest

from oracle import sphere as S
from paper_2402_01282_b200 import inputs

pytestmark = pytest.mark.gpu

FWD_TOL = 1e-11
RT_TOL = 1e-12


def _api():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2402_01282_b200 import api
    return torch, api


def _relmax(a, b):
    den = np.abs(b).max()
    num = np.abs(a - b).max()
    return num if den == 0 else num / den


def _signals(L, seed, real, batch):
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, seed, batch)
    f = np.stack([S.sht_inverse(flm[b], L, "f80", sampling="dh") for b in range(batch)])
    if real:
        assert np.abs(f.imag).max() < 1e-14 * max(1.0, np.abs(f).max())
        return flm, np.ascontiguousarray(f.real.astype(np.float64))
    return flm, np.ascontiguousarray(f.astype(np.complex128))


@pytest.mark.parametrize("L,real,batch", [(1, False, 1), (2, True, 1), (5, False, 2), (16, True, 3), (33, False, 1),
                                          (64, True, 2)])
def test_dh_harmonic_transforms_match_oracle(L, real, batch):
    torch, api = _api()
    flm, f = _signals(L, 21 + L, real, batch)
    assert f.shape == (batch, 2 * L, 2 * L - 1)
    plan = api.s2wav_plan_create(L, 1, 2.0, 0, True, real, batch, flags=api.S2W_DH)
    assert plan.signal_elems == 2 * L * (2 * L - 1)
    got = plan.harmonic_forward(torch.from_numpy(f).cuda(), L * (2 * L - 1)).cpu().numpy().reshape(batch, L, 2 * L - 1)
    for b in range(batch):
        ref = S.sht_forward(f[b], L, "f80", sampling="dh").astype(np.complex128)
        assert _relmax(got[b], ref) < FWD_TOL
        assert _relmax(got[b], flm[b]) < FWD_TOL
    back = plan.harmonic_inverse(torch.from_numpy(flm).cuda()).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    plan.close()


DH_CASES = [
    # L, N, lam, J0, multires, real, batch, precompute
    (16, 3, 2.0, 0, True, False, 1, False),
    (24, 4, 2.0, 1, True, True, 2, False),       # even N
    (20, 5, 3.0, 1, True, False, 1, True),       # precomputed-kernel variant on the Driscoll-Healy rings
    (40, 3, 1.7, 2, True, True, 5, False),       # non-integer lambda, two column chunks
    (48, 2, 2.0, 2, False, True, 1, True),       # no multiresolution
    (9, 2, 2.0, 0, True, True, 1, False),        # L_0 = 2 with N = 2
]


@pytest.mark.parametrize("L,N,lam,J0,mr,real,batch,pre", DH_CASES)
def test_dh_wavelet_transform_parity(L, N, lam, J0, mr, real, batch, pre):
    torch, api = _api()
    flm, f = _signals(L, 200 + L + N, real, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, real, batch, flags=api.S2W_DH | (api.S2W_PRECOMPUTE if pre else 0))
    w = plan.forward(torch.from_numpy(f).cuda())
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    cast = (lambda a: a.real.astype(np.float64)) if real else (lambda a: a.astype(np.complex128))
    for b in sorted({0, batch - 1}):
        o_phi, o_psi = S.analysis(f[b], L, N, lam, J0, mr, "f80", filt, sampling="dh")
        assert _relmax(scal[b].cpu().numpy(), cast(o_phi)) < FWD_TOL
        for j in range(plan.J0, plan.J + 1):
            ref = cast(o_psi[j])
            got = scales[(j, 0)][b].cpu().numpy()
            assert got.shape == ref.shape                      # [2N-1][2 L_j][2 L_j - 1]
            if np.abs(ref).max() == 0.0:
                assert np.abs(got).max() == 0.0
            else:
                assert _relmax(got, ref) < FWD_TOL, (b, j)
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    # synthesis parity on the oracle's coefficients
    o_phi, o_psi = S.analysis(f[0], L, N, lam, J0, mr, "f80", filt, sampling="dh")
    o_f = S.synthesis(o_phi, o_psi, L, N, lam, J0, mr, "f80", filt, sampling="dh")
    packed = np.zeros((batch, plan.coeff_elems), dtype=f.dtype)
    nr, ng, nt, npx, off = plan.scale_shape(-1)
    packed[0, off:off + nt * npx] = cast(o_phi).ravel()
    for j in range(plan.J0, plan.J + 1):
        nr, ng, nt, npx, off = plan.scale_shape(j)
        packed[0, off:off + ng * nt * npx] = cast(o_psi[j]).ravel()
    back = plan.inverse(torch.from_numpy(packed).cuda()).cpu().numpy().reshape(f.shape)
    assert _relmax(back[0], cast(o_f)) < FWD_TOL
    plan.close()


@pytest.mark.parametrize("L,N,real,batch", [(512, 3, True, 2), (300, 2, False, 1)])
def test_dh_large_round_trip_and_sampled_rings(L, N, real, batch):
    """Several ring groups per warp on the 2L-ring grids, Bluestein lengths up to 2048: recovered f_lm against the seeded
    truth, sampled rings of the top scale against the oracle, round trip."""
    torch, api = _api()
    lam, J0 = 2.0, 5
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, 80 + L, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, real, batch, flags=api.S2W_DH)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    got = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(batch, L, 2 * L - 1)
    assert _relmax(got, flm) < FWD_TOL
    w = plan.forward(f)
    back = plan.inverse(w)
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    j = plan.J
    Lj = plan.scale_shape(j)[2] // 2
    rings = [0, 1, Lj // 2, Lj, 2 * Lj - 2, 2 * Lj - 1]
    _, o_psi = S.analysis_from_flm(flm[0], L, N, lam, J0, True, "f80", filt, scales=[j], rings={j: np.array(rings)},
                                   sampling="dh")
    ref = o_psi[j]
    ref = ref.real.astype(np.float64) if real else ref.astype(np.complex128)
    blk = scales[(j, 0)][0]
    assert np.abs(blk[:, rings, :].cpu().numpy() - ref).max() / float(blk.abs().max()) < FWD_TOL
    plan.close()


def test_dh_is_rejected_where_it_is_not_built():
    torch, api = _api()
    with pytest.raises(api.S2WError):
        api.s2ball_plan_create(8, 4, 2, 2.0, 2.0, 0, flags=api.S2W_DH)
    with pytest.raises(api.S2WError):
        api.s2wav_plan_create(8, 2, 2.0, 0, True, False, 1, flags=api.S2W_DH, spin=1)
    plan = api.s2wav_plan_create(8, 2, 2.0, 0, True, False, 1, flags=api.S2W_DH)
    y = torch.zeros((1, plan.coeff_elems), dtype=torch.complex128, device="cuda")
    with pytest.raises(api.S2WError):
        plan.forward_adjoint(y)
    plan.close()
