"""GPU parity tests of spin-s plans (spin fields: Eq. 1, Eq. 12; sY_lm by reading R2): s2wav_plan_create_spin through the
C ABI against the oracle's spin transforms on the same seeded inputs -- harmonic transform, wavelet coefficients,
round trip, adjoint identity.  Tolerances as for spin 0."""
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


def _spin_flm(L, seed, spin):
    flm = inputs.flm_complex(L, seed, 1)[0]
    flm[:abs(spin), :] = 0          # no spin-s harmonics below l = |s|
    return flm


@pytest.mark.parametrize("L,N,lam,J0,mr,spin", [(8, 2, 2.0, 0, True, 2), (16, 3, 2.0, 1, True, -1), (20, 4, 2.0, 0, False, 1),
                                                (12, 3, 2.0, 0, True, 3), (33, 5, 2.0, 2, True, -2)])
@pytest.mark.parametrize("pre", [False, True])
def test_spin_transforms_match_oracle(L, N, lam, J0, mr, spin, pre):
    """pre: S2W_PRECOMPUTE -- the table kernels, with the theta quadrature folded into the table of the rows n = -s, +s."""
    torch, api = _api()
    flm = _spin_flm(L, 60 + L, spin)
    f = np.ascontiguousarray(S.sht_inverse(flm, L, "f80", spin=spin).astype(np.complex128))
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, False, 1, spin=spin, flags=api.S2W_PRECOMPUTE if pre else 0)
    fd = torch.from_numpy(f).cuda().reshape(1, -1)
    got = plan.harmonic_forward(fd, L * (2 * L - 1)).cpu().numpy().reshape(L, 2 * L - 1)
    assert _relmax(got, flm) < FWD_TOL
    back = plan.harmonic_inverse(torch.from_numpy(flm).cuda().reshape(1, -1)).cpu().numpy().reshape(L, 2 * L - 1)
    assert _relmax(back, f) < RT_TOL
    w = plan.forward(fd)
    scal, scales = plan.split(w)
    o_phi, o_psi = S.analysis(f, L, N, lam, J0, mr, "f80", spin=spin)
    ref = o_phi.astype(np.complex128)
    gs = scal[0].cpu().numpy()
    if np.abs(ref).max() == 0:
        assert np.abs(gs).max() == 0        # scaling band-limit <= |spin|
    else:
        assert _relmax(gs, ref) < FWD_TOL
    for j in range(plan.J0, plan.J + 1):
        assert _relmax(scales[(j, 0)][0].cpu().numpy(), o_psi[j].astype(np.complex128)) < FWD_TOL, j
    rec = plan.inverse(w).cpu().numpy().reshape(L, 2 * L - 1)
    assert _relmax(rec, f) < RT_TOL
    # adjoint identity on the spin plan
    gen = torch.Generator(device="cuda").manual_seed(L)
    x = torch.randn(1, plan.signal_elems, dtype=torch.complex128, device="cuda", generator=gen)
    y = torch.randn(1, plan.coeff_elems, dtype=torch.complex128, device="cuda", generator=gen)
    Ax, Ahy = plan.forward(x), plan.forward_adjoint(y)
    assert abs(torch.vdot(Ax.flatten(), y.flatten()) - torch.vdot(x.flatten(), Ahy.flatten())) < 1e-12 * Ax.norm() * y.norm()
    Sy, Shx = plan.inverse(y), plan.inverse_adjoint(x)
    assert abs(torch.vdot(Sy.flatten(), x.flatten()) - torch.vdot(y.flatten(), Shx.flatten())) < 1e-12 * Sy.norm() * x.norm()
    plan.close()


def test_spin_round_trip_at_a_large_band_limit():
    """L = 512, spin 2 (polarisation-like), N = 3: recovered f_lm against the seeded truth and the round trip."""
    torch, api = _api()
    L, N, spin = 512, 3, 2
    flm = _spin_flm(L, 61, spin)
    plan = api.s2wav_plan_create(L, N, 2.0, 3, True, False, 1, spin=spin)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda().reshape(1, -1))
    got = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(L, 2 * L - 1)
    assert _relmax(got, flm) < FWD_TOL
    rings = [0, 3, L // 2, L - 1]
    ref = S.sht_inverse(flm, L, "f80", thetas=S.mw_thetas(L, "f80")[rings], spin=spin).astype(np.complex128)
    fn = f.cpu().numpy().reshape(L, 2 * L - 1)
    assert np.abs(fn[rings] - ref).max() / np.abs(fn).max() < RT_TOL
    back = plan.inverse(plan.forward(f))
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    plan.close()


def test_spin_argument_errors():
    torch, api = _api()
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2wav_plan_create(8, 2, 2.0, 0, True, True, 1, spin=1)      # a spin signal is complex
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2wav_plan_create(4, 2, 2.0, 0, True, False, 1, spin=4)     # |spin| >= L
