"""GPU parity tests of the ball (Fourier-Laguerre) wavelet transform: the CUDA path through the C ABI against the CPU
oracle (oracle/ball.py), element by element on the same seeded inputs.  Tolerances: forward coefficients 1e-11
relative max error per scale block, round trip 1e-12 (BASELINE.json, reading R12)."""
import numpy as np
import pytest

from oracle import ball as OB
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


def _voxels(L, P, tau, seed):
    flmp = inputs.flmp_complex(L, P, seed)
    f = OB.z_inverse(flmp, L, P, tau, "f80")
    return flmp, np.ascontiguousarray(f.astype(np.complex128))


@pytest.mark.parametrize("L,P,tau", [(8, 8, 1.0), (12, 5, 2.0), (33, 16, 1.0)])
def test_spherical_laguerre_transform_matches_oracle(L, P, tau):
    """Z and Z^-1 (Eqs. 10-11): per-shell SHT + radial Laguerre contraction (a10)."""
    torch, api = _api()
    flmp, f = _voxels(L, P, tau, 40 + L)
    plan = api.s2ball_plan_create(L, P, 1, 2.0, 2.0, 0, tau)
    got = plan.harmonic_forward(torch.from_numpy(f).cuda().reshape(1, -1), P * L * (2 * L - 1))
    got = got.cpu().numpy().reshape(P, L, 2 * L - 1)
    ref = OB.z_forward(f, L, P, tau, "f80").astype(np.complex128)
    assert _relmax(got, ref) < FWD_TOL
    assert _relmax(got, flmp) < FWD_TOL
    back = plan.harmonic_inverse(torch.from_numpy(flmp).cuda().reshape(1, -1)).cpu().numpy().reshape(P, L, 2 * L - 1)
    assert _relmax(back, f) < RT_TOL
    plan.close()


CASES = [
    # L, P, N, lam_l, lam_p, J0, tau
    (8, 8, 1, 2.0, 2.0, 0, 1.0),
    (12, 8, 3, 2.0, 2.0, 0, 1.0),
    (16, 6, 2, 2.0, 3.0, 1, 0.5),     # even N, P not a power of the dilation, J0 = 1, tau != 1
    (20, 16, 3, 2.0, 2.0, 0, 1.0),
]


@pytest.mark.parametrize("mode", ["default", "recursion"])
@pytest.mark.parametrize("L,P,N,lam,nu,J0,tau", CASES)
def test_ball_forward_inverse_parity(L, P, N, lam, nu, J0, tau, mode):
    """Both modes of a small ball plan against the oracle: the default (L <= 256: precomputed Wigner-d tables with the
    theta quadrature folded in, step a2 a transposing copy) and S2W_RECURSION (on-the-fly recursion, explicit step a2)."""
    torch, api = _api()
    flmp, f = _voxels(L, P, tau, 70 + L + N)
    plan = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, flags=api.S2W_RECURSION if mode == "recursion" else 0)
    fd = torch.from_numpy(f).cuda().reshape(1, -1)
    w = plan.forward(fd)
    scal, scales = plan.split(w)
    filt = OB.filters(L, P, N, lam, nu, J0, J0, "f80")
    o_phi, o_psi = OB.analysis(f, L, P, N, lam, nu, J0, J0, tau, "f80", filt)
    assert _relmax(scal[0].cpu().numpy(), o_phi.astype(np.complex128)) < FWD_TOL
    assert set(scales.keys()) == set(o_psi.keys())
    for key, ref in o_psi.items():
        got = scales[key][0].cpu().numpy()
        assert got.shape == ref.shape, key
        assert _relmax(got, ref.astype(np.complex128)) < FWD_TOL, key
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    # synthesis parity on the oracle's coefficients
    o_f = OB.synthesis(o_phi, o_psi, L, P, N, lam, nu, J0, J0, tau, "f80", filt)
    packed = np.zeros((1, plan.coeff_elems), dtype=np.complex128)
    nr, ng, nt, npx, off = plan.scale_shape(-1)
    packed[0, off:off + nr * nt * npx] = o_phi.astype(np.complex128).ravel()
    for (j, jp), ref in o_psi.items():
        nr, ng, nt, npx, off = plan.scale_shape(j, jp)
        packed[0, off:off + nr * ng * nt * npx] = ref.astype(np.complex128).ravel()
    back2 = plan.inverse(torch.from_numpy(packed).cuda()).cpu().numpy().reshape(f.shape)
    assert _relmax(back2, o_f.astype(np.complex128)) < FWD_TOL
    plan.close()


def test_ball_argument_style_entry_points_and_host_path():
    torch, api = _api()
    L, P, N, lam, nu, J0, tau = 10, 4, 2, 2.0, 2.0, 0, 1.0
    flmp, f = _voxels(L, P, tau, 9)
    fd = torch.from_numpy(f).cuda()
    w = api.s2ball_forward(fd, L, P, N, lam, nu, J0, tau)
    back = api.s2ball_inverse(w, L, P, N, lam, nu, J0, tau)
    assert _relmax(back.cpu().numpy(), f) < RT_TOL
    wh = api.s2ball_forward_host(f, L, P, N, lam, nu, J0, tau)
    assert np.allclose(wh, w.cpu().numpy(), rtol=0, atol=1e-13 * np.abs(wh).max())
    fh = api.s2ball_inverse_host(wh, L, P, N, lam, nu, J0, tau)
    assert _relmax(fh, f) < RT_TOL


def test_ball_real_signal_gives_real_coefficients():
    """A real field on the ball: S2W_REAL path (m >= 0 only) against the complex path."""
    torch, api = _api()
    L, P, N, lam, nu, J0, tau = 12, 6, 3, 2.0, 2.0, 0, 1.0
    flm = np.stack([inputs.flm_real(L, 200 + p, 1)[0] / np.sqrt(p + 1.0) for p in range(P)])
    f = OB.z_inverse(flm, L, P, tau, "f80")
    assert np.abs(f.imag).max() < 1e-14 * np.abs(f).max()
    fr = np.ascontiguousarray(f.real.astype(np.float64))
    pr = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, real=True)
    pc = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, real=False)
    wr = pr.forward(torch.from_numpy(fr).cuda().reshape(1, -1)).cpu().numpy()
    wc = pc.forward(torch.from_numpy(fr.astype(np.complex128)).cuda().reshape(1, -1)).cpu().numpy()
    assert np.abs(wc.imag).max() < 1e-12 * np.abs(wc).max()
    assert _relmax(wr, wc.real) < FWD_TOL
    back = pr.inverse(torch.from_numpy(wr).cuda()).cpu().numpy().reshape(fr.shape)
    assert _relmax(back, fr) < RT_TOL
    pr.close()
    pc.close()


@pytest.mark.parametrize("mode", ["default", "recursion"])
def test_config5_full_size(mode):
    """BASELINE config 5 at full size (L = P = 128, N = 3, complex, 64 (j, j') scales), in the configuration bench.py times
    (default: precomputed tables with the folded quadrature) and with S2W_RECURSION: round trip on all voxels,
    recovered f_lmp against the seeded truth, and two whole (j, j') coefficient blocks against the oracle."""
    torch, api = _api()
    c = inputs.CONFIGS["C5"]
    L, P, N, lam, nu, J0, tau = c["L"], c["P"], c["N"], c["lam"], c["nu"], c["J0"], c["tau"]
    flmp = inputs.config_coefficients("C5")
    plan = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, flags=api.S2W_RECURSION if mode == "recursion" else 0)
    f = plan.harmonic_inverse(torch.from_numpy(flmp).cuda().reshape(1, -1))
    got = plan.harmonic_forward(f, P * L * (2 * L - 1)).cpu().numpy().reshape(P, L, 2 * L - 1)
    assert _relmax(got, flmp) < FWD_TOL
    w = plan.forward(f)
    back = plan.inverse(w)
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    scal, scales = plan.split(w)
    filt = OB.filters(L, P, N, lam, nu, J0, J0, "f80")
    keys = [(4, 5), (6, 3)]
    _, o_psi = OB.analysis_from_flmp(flmp, L, P, N, lam, nu, J0, J0, tau, "f80", filt, scales=keys)
    for key in keys:
        ref = o_psi[key].astype(np.complex128)
        got = scales[key][0].cpu().numpy()
        assert got.shape == ref.shape
        assert _relmax(got, ref) < FWD_TOL, key
    plan.close()


def test_ball_precomputed_kernel_variant_matches_on_the_fly():
    """S2W_PRECOMPUTE on a ball plan: same coefficients as the recursion path, round trip within tolerance."""
    torch, api = _api()
    L, P, N, lam, nu, J0, tau = 20, 8, 3, 2.0, 2.0, 0, 1.0
    flmp, f = _voxels(L, P, tau, 77)
    fd = torch.from_numpy(f).cuda().reshape(1, -1)
    otf = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, flags=api.S2W_RECURSION)
    pre = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, flags=api.S2W_PRECOMPUTE)
    w0, w1 = otf.forward(fd), pre.forward(fd)
    assert float((w0 - w1).abs().max()) < 1e-12 * float(w0.abs().max())
    back = pre.inverse(w1).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    otf.close()
    pre.close()


def test_table2_shape_full_size():
    """The shape of the paper's Table 2 at its largest size (ball, N = 1, L = P = 256): 256 Gauss-
    Laguerre nodes (weights spanning 400 orders of magnitude, built in the log domain), recovered f_lmp against the
    seeded truth, wavelet round trip on all voxels."""
    torch, api = _api()
    c = inputs.CONFIGS["T2"]
    L, P, N, lam, nu, J0, tau = c["L"], c["P"], c["N"], c["lam"], c["nu"], c["J0"], c["tau"]
    flmp = inputs.config_coefficients("T2")
    plan = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau)
    f = plan.harmonic_inverse(torch.from_numpy(flmp).cuda().reshape(1, -1))
    got = plan.harmonic_forward(f, P * L * (2 * L - 1)).cpu().numpy().reshape(P, L, 2 * L - 1)
    assert _relmax(got, flmp) < FWD_TOL
    del got
    w = plan.forward(f)
    back = plan.inverse(w)
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    plan.close()


# ---- stand-alone generalised Fourier transforms on B^3 and H^4 ----
def _band_limited_fhat(L, P, N, seed):
    rng = np.random.default_rng(seed)
    fh = rng.standard_normal((2 * N - 1, P, L, 2 * L - 1)) + 1j * rng.standard_normal((2 * N - 1, P, L, 2 * L - 1))
    ell = np.arange(L)[:, None]
    m = np.arange(-(L - 1), L)[None, :]
    fh *= (np.abs(m) <= ell)[None, None]
    for ni in range(2 * N - 1):
        fh[ni] *= (abs(ni - (N - 1)) <= np.arange(L))[None, :, None]
    return fh


@pytest.mark.parametrize("L,P,N,tau", [(8, 6, 3, 1.0), (12, 5, 2, 0.7), (20, 9, 4, 1.5), (33, 16, 1, 1.0)])
def test_wigner_laguerre_transform_matches_oracle(L, P, N, tau):
    """s2ball_q_inverse / s2ball_q_forward (Q = K D, Eqs. 24-25) element by element against oracle.ball.q_inverse /
    q_forward, odd and even N, and Q Q^-1 = identity on the GPU."""
    import torch
    from paper_2402_01282_b200 import api
    from oracle import ball as B
    fh = _band_limited_fhat(L, P, N, 40 + L)
    f_ref = B.q_inverse(fh, L, P, N, tau, "f80").astype(np.complex128)
    f_gpu = api.s2ball_q_inverse(torch.from_numpy(fh).cuda(), L, P, N, tau)
    assert np.abs(f_gpu.cpu().numpy() - f_ref).max() < 1e-11 * np.abs(f_ref).max()
    fh_ref = B.q_forward(f_ref, L, P, N, tau, "f80").astype(np.complex128)
    fh_gpu = api.s2ball_q_forward(torch.from_numpy(np.ascontiguousarray(f_ref)).cuda(), L, P, N, tau)
    assert np.abs(fh_gpu.cpu().numpy() - fh_ref).max() < 1e-11 * np.abs(fh_ref).max()
    back = api.s2ball_q_forward(f_gpu, L, P, N, tau).cpu().numpy()
    assert np.abs(back - fh).max() < 1e-12 * np.abs(fh).max()


@pytest.mark.parametrize("L,P,tau,real", [(10, 7, 1.0, False), (16, 12, 1.3, True)])
def test_spherical_laguerre_entry_points_match_oracle(L, P, tau, real):
    """s2ball_z_forward / s2ball_z_inverse (Z = K Y, Eqs. 10-11) against oracle.ball.z_forward / z_inverse."""
    import torch
    from paper_2402_01282_b200 import api, inputs
    from oracle import ball as B
    flmp = inputs.flmp_complex(L, P, 77)
    if real:
        m = np.arange(-(L - 1), L)
        flmp = 0.5 * (flmp + ((-1.0) ** np.abs(m))[None, None, :] * np.conj(flmp[:, :, ::-1]))
    f_ref = B.z_inverse(flmp, L, P, tau, "f80")
    if real:
        assert np.abs(f_ref.imag).max() < 1e-14 * np.abs(f_ref).max()
    f_gpu = api.s2ball_z_inverse(torch.from_numpy(flmp).cuda(), L, P, tau, real=real).cpu().numpy()
    ref = f_ref.real.astype(np.float64) if real else f_ref.astype(np.complex128)
    assert np.abs(f_gpu - ref).max() < 1e-11 * np.abs(ref).max()
    back = api.s2ball_z_forward(torch.from_numpy(np.ascontiguousarray(ref)).cuda(), L, P, tau).cpu().numpy()
    assert np.abs(back - flmp).max() < 1e-12 * np.abs(flmp).max()
    z_ref = B.z_forward(f_ref, L, P, tau, "f80").astype(np.complex128)
    assert np.abs(back - z_ref).max() < 1e-11 * np.abs(z_ref).max()
