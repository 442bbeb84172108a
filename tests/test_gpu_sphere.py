"""GPU parity tests: the CUDA path (through the C ABI, via paper_2402_01282_b200.api) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances are BASELINE.json's: forward coefficients within
1e-11 relative max error per scale block, round trip within 1e-12 relative max error (reading R12)."""
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


def _signals(L, seed, real, batch, spectrum="l^-2"):
    """(flm [batch][L][2L-1], pixels [batch][L][2L-1]) -- pixels by the oracle's inverse SHT in long double."""
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, seed, batch, spectrum)
    f = np.stack([S.sht_inverse(flm[b], L, "f80") for b in range(batch)])
    if real:
        assert np.abs(f.imag).max() < 1e-14 * max(1.0, np.abs(f).max())
        return flm, np.ascontiguousarray(f.real.astype(np.float64))
    return flm, np.ascontiguousarray(f.astype(np.complex128))


def _relmax(a, b):
    den = np.abs(b).max()
    num = np.abs(a - b).max()
    return num if den == 0 else num / den


@pytest.mark.parametrize("L,real,batch", [(1, False, 1), (2, True, 1), (5, False, 2), (16, True, 3), (33, False, 1),
                                          (64, True, 1), (100, False, 1)])
def test_harmonic_transforms_match_oracle(L, real, batch):
    torch, api = _api()
    flm, f = _signals(L, 11 + L, real, batch)
    plan = api.s2wav_plan_create(L, 1, 2.0, 0, True, real, batch)
    fd = torch.from_numpy(f).cuda()
    got = plan.harmonic_forward(fd, L * (2 * L - 1)).cpu().numpy().reshape(batch, L, 2 * L - 1)
    for b in range(batch):
        ref = S.sht_forward(f[b], L, "f80").astype(np.complex128)
        assert _relmax(got[b], ref) < FWD_TOL
        assert _relmax(got[b], flm[b]) < FWD_TOL
    back = plan.harmonic_inverse(torch.from_numpy(flm).cuda()).cpu().numpy().reshape(batch, L, 2 * L - 1)
    assert _relmax(back, f) < RT_TOL
    plan.close()


CASES = [
    # L, N, lam, J0, multires, real, batch
    (32, 1, 2.0, 0, False, True, 1),      # BASELINE config 1
    (16, 3, 2.0, 0, True, False, 1),
    (24, 4, 2.0, 1, True, True, 2),       # even N: imaginary zeta
    (20, 5, 3.0, 1, True, False, 1),
    (9, 2, 2.0, 0, True, True, 1),        # L_0 = 2 with N = 2
    (12, 3, 2.0, 0, True, False, 3),      # L_0 = 2 < N
    (40, 3, 1.7, 2, True, True, 5),       # non-integer lambda, batch > 4 (two column chunks)
    (64, 5, 2.0, 2, False, False, 1),     # no multiresolution
    (7, 7, 2.0, 0, True, True, 1),        # N = L
    (1, 1, 2.0, 0, True, False, 1),       # degenerate L = 1
]


@pytest.mark.parametrize("L,N,lam,J0,mr,real,batch", CASES)
def test_forward_inverse_parity_small(L, N, lam, J0, mr, real, batch):
    torch, api = _api()
    spectrum = "white" if L == 32 and N == 1 else "l^-2"
    flm, f = _signals(L, 100 + L + N, real, batch, spectrum)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, real, batch)
    w = plan.forward(torch.from_numpy(f).cuda())
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    worst = 0.0
    for b in range(batch):
        o_phi, o_psi = S.analysis(f[b], L, N, lam, J0, mr, "f80", filt)
        e = _relmax(scal[b].cpu().numpy(), o_phi.astype(np.complex128) if not real else o_phi.real.astype(np.float64))
        worst = max(worst, e)
        for j in range(plan.J0, plan.J + 1):
            ref = o_psi[j]
            if real:
                assert np.abs(ref.imag).max() <= 1e-13 * max(np.abs(ref).max(), 1e-300)
                ref = ref.real.astype(np.float64)
            else:
                ref = ref.astype(np.complex128)
            got = scales[(j, 0)][b].cpu().numpy()
            assert got.shape == ref.shape
            worst = max(worst, _relmax(got, ref))
    assert worst < FWD_TOL, worst
    # round trip on the GPU
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    # synthesis parity: oracle coefficients in, compare with the oracle's synthesis
    o_phi, o_psi = S.analysis(f[0], L, N, lam, J0, mr, "f80", filt)
    o_f = S.synthesis(o_phi, o_psi, L, N, lam, J0, mr, "f80", filt)
    packed = np.zeros((batch, plan.coeff_elems), dtype=f.dtype)
    cast = (lambda a: a.real.astype(np.float64)) if real else (lambda a: a.astype(np.complex128))
    nr, ng, nt, npx, off = plan.scale_shape(-1)
    packed[0, off:off + nt * npx] = cast(o_phi).ravel()
    for j in range(plan.J0, plan.J + 1):
        nr, ng, nt, npx, off = plan.scale_shape(j)
        packed[0, off:off + ng * nt * npx] = cast(o_psi[j]).ravel()
    back = plan.inverse(torch.from_numpy(packed).cuda()).cpu().numpy().reshape(f.shape)
    assert _relmax(back[0], cast(o_f)) < FWD_TOL
    plan.close()


def test_config2_full_parity():
    """BASELINE config 2: L = 256, N = 3, lambda = 2, J0 = 2, multiresolution, complex signal, seed 1."""
    torch, api = _api()
    c = inputs.CONFIGS["C2"]
    L, N, lam, J0 = c["L"], c["N"], c["lam"], c["J0"]
    flm = inputs.config_coefficients("C2")
    f = np.ascontiguousarray(S.sht_inverse(flm[0], L, "f80").astype(np.complex128))[None]
    plan = api.s2wav_plan_create(L, N, lam, J0, True, False, 1)
    w = plan.forward(torch.from_numpy(f).cuda())
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    o_phi, o_psi = S.analysis_from_flm(S.sht_forward(f[0], L, "f80"), L, N, lam, J0, True, "f80", filt)
    assert _relmax(scal[0].cpu().numpy(), o_phi.astype(np.complex128)) < FWD_TOL
    for j in range(plan.J0, plan.J + 1):
        assert _relmax(scales[(j, 0)][0].cpu().numpy(), o_psi[j].astype(np.complex128)) < FWD_TOL, j
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    plan.close()


def test_argument_style_entry_points_and_host_path():
    torch, api = _api()
    L, N, lam, J0 = 16, 3, 2.0, 1
    flm, f = _signals(L, 5, True, 2)
    fd = torch.from_numpy(f).cuda()
    w = api.s2wav_forward(fd, L, N, lam, J0, True)
    back = api.s2wav_inverse(w, L, N, lam, J0, True)
    assert _relmax(back.cpu().numpy(), f) < RT_TOL
    wh = api.s2wav_forward_host(f, L, N, lam, J0, True)
    assert np.array_equal(wh, w.cpu().numpy())
    fh = api.s2wav_inverse_host(wh, L, N, lam, J0, True)
    assert _relmax(fh, f) < RT_TOL
    assert api.launch_count() > 0


def test_error_codes():
    torch, api = _api()
    with pytest.raises(api.S2WError):
        api.s2wav_plan_create(8, 9, 2.0, 0)          # N > L
    with pytest.raises(api.S2WError):
        api.s2wav_plan_create(8, 2, 1.0, 0)          # lambda <= 1
    with pytest.raises(api.S2WError):
        api.s2wav_plan_create(8, 2, 2.0, 7)          # J0 > J


PRE_CASES = [
    # L, N, lam, J0, multires, real, batch
    (24, 4, 2.0, 1, True, True, 2),
    (20, 5, 3.0, 1, True, False, 1),
    (40, 3, 1.7, 2, True, True, 5),
    (64, 5, 2.0, 2, False, False, 1),
    (130, 3, 2.0, 3, True, True, 4),      # several ring groups per hemisphere, ragged last group
]


@pytest.mark.parametrize("L,N,lam,J0,mr,real,batch", PRE_CASES)
def test_precomputed_kernel_variant_parity(L, N, lam, J0, mr, real, batch):
    """S2W_PRECOMPUTE (step a9): the table-streaming DMMA contraction against the oracle and the on-the-fly path."""
    torch, api = _api()
    flm, f = _signals(L, 300 + L + N, real, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, real, batch, flags=api.S2W_PRECOMPUTE)
    otf = api.s2wav_plan_create(L, N, lam, J0, mr, real, batch)
    fd = torch.from_numpy(f).cuda()
    w = plan.forward(fd)
    w2 = otf.forward(fd)
    scale = float(w2.abs().max())
    assert float((w - w2).abs().max()) < 1e-12 * scale
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    cast = (lambda a: a.real.astype(np.float64)) if real else (lambda a: a.astype(np.complex128))
    o_phi, o_psi = S.analysis(f[0], L, N, lam, J0, mr, "f80", filt)
    assert _relmax(scal[0].cpu().numpy(), cast(o_phi)) < FWD_TOL
    for j in range(plan.J0, plan.J + 1):
        assert _relmax(scales[(j, 0)][0].cpu().numpy(), cast(o_psi[j])) < FWD_TOL, j
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    plan.close()
    otf.close()


def test_config3_full_size_sampled_parity():
    """BASELINE config 3 at full size (L = 1024, N = 5, batch 4, real) in the launch configuration bench.py times:
    round trip on all pixels, and forward coefficients of the top scale on sampled beta rings against the oracle
    (which evaluates single rings: oracle.sphere.analysis_from_flm(scales=, rings=))."""
    torch, api = _api()
    c = inputs.CONFIGS["C3"]
    L, N, lam, J0, B = c["L"], c["N"], c["lam"], c["J0"], c["batch"]
    flm = inputs.config_coefficients("C3")
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, B)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    back = plan.inverse(w)
    rt = float((back - f).abs().max() / f.abs().max())
    assert rt < RT_TOL, rt
    # harmonic coefficients recovered from the pixels (forward SHT, steps a1-a3) against the seeded truth
    got_flm = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(B, L, 2 * L - 1)
    assert _relmax(got_flm, flm) < FWD_TOL
    # sampled rings of the two top scales and of a middle scale, signal 1
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    for j, rings in [(plan.J, [0, 1, 357, 1022, 1023]), (plan.J - 1, [3, 511, 1020]), (plan.J - 3, [0, 64, 127])]:
        _, o_psi = S.analysis_from_flm(flm[1], L, N, lam, J0, True, "f80", filt, scales=[j],
                                       rings={j: np.array(rings)})
        ref = o_psi[j].real.astype(np.float64)                      # [2N-1][len(rings)][2L_j-1]
        got = scales[(j, 0)][1][:, rings, :].cpu().numpy()
        den = float(scales[(j, 0)][1].abs().max())
        assert np.abs(got - ref).max() / den < FWD_TOL, j
    plan.close()


def test_config4_band_limit_2048_seeds_and_sampled_rings():
    """BASELINE config 4 grid (L = 2048, real): beyond L ~ 1930 the plain recursion seed underflows fp64,
    so this exercises the range-extended group seeds.  Harmonic transforms: recovered f_lm against the seeded truth,
    pixels of sampled rings (poles, mid-latitudes, the rings whose seeds underflow) against the long-double oracle,
    and the wavelet round trip at N = 3, J0 = 4."""
    torch, api = _api()
    c = inputs.CONFIGS["C4"]
    L, N, lam, J0 = c["L"], c["N"], c["lam"], c["J0"]
    flm = inputs.config_coefficients("C4")
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, 1)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    got_flm = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(1, L, 2 * L - 1)
    assert _relmax(got_flm, flm) < FWD_TOL
    rings = [0, 1, 2, 156, 480, 1023, 1024, 1890, 2045, 2046, 2047]
    th = S.mw_thetas(L, "f80")
    ref = S.sht_inverse(flm[0], L, "f80", thetas=th[rings]).real.astype(np.float64)
    fn = f.cpu().numpy().reshape(L, 2 * L - 1)
    assert np.abs(fn[rings] - ref).max() / np.abs(fn).max() < RT_TOL
    w = plan.forward(f)
    back = plan.inverse(w)
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    plan.close()


EDGE_CASES = [
    # L, N, lam, J0, multires, real, batch
    (2, 1, 2.0, 0, True, True, 1),        # smallest non-trivial grid: 2 rings x 3 samples
    (3, 2, 2.0, 1, True, False, 2),
    (16, 2, 2.0, 4, True, True, 1),       # J0 = J: a single wavelet scale plus the scaling part
    (27, 3, 3.0, 0, True, True, 3),       # lambda = 3, L = lambda^3
    (33, 5, 2.0, 2, False, True, 2),      # no multiresolution, N > 1, real, L = 2^k + 1 (empty top scale)
    (48, 3, 2.0, 1, True, False, 7),      # 14 columns: four column chunks, the last one ragged
    (96, 6, 2.0, 3, True, True, 1),       # even N (imaginary zeta), three ring groups per hemisphere
]


@pytest.mark.parametrize("L,N,lam,J0,mr,real,batch", EDGE_CASES)
def test_forward_inverse_parity_edge_cases(L, N, lam, J0, mr, real, batch):
    torch, api = _api()
    flm, f = _signals(L, 500 + L + N, real, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, real, batch)
    w = plan.forward(torch.from_numpy(f).cuda())
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80")
    cast = (lambda a: a.real.astype(np.float64)) if real else (lambda a: a.astype(np.complex128))
    for b in sorted({0, batch - 1}):
        o_phi, o_psi = S.analysis(f[b], L, N, lam, J0, mr, "f80", filt)
        assert _relmax(scal[b].cpu().numpy(), cast(o_phi)) < FWD_TOL
        for j in range(plan.J0, plan.J + 1):
            ref = cast(o_psi[j])
            got = scales[(j, 0)][b].cpu().numpy()
            assert got.shape == ref.shape
            if np.abs(ref).max() == 0.0:
                assert np.abs(got).max() == 0.0          # empty scale: exactly zero
            else:
                assert _relmax(got, ref) < FWD_TOL, (b, j)
    back = plan.inverse(w).cpu().numpy().reshape(f.shape)
    assert _relmax(back, f) < RT_TOL
    plan.close()


def test_two_plans_and_a_side_stream():
    """Plans are immutable and independent: two plans used alternately, one of them on a non-default stream."""
    torch, api = _api()
    flm_a, f_a = _signals(20, 900, True, 1)
    flm_b, f_b = _signals(28, 901, False, 2)
    pa = api.s2wav_plan_create(20, 3, 2.0, 1, True, True, 1)
    pb = api.s2wav_plan_create(28, 2, 2.0, 0, True, False, 2)
    fa, fb = torch.from_numpy(f_a).cuda(), torch.from_numpy(f_b).cuda()
    ref_a, ref_b = pa.forward(fa).clone(), pb.forward(fb).clone()
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(3):
        with torch.cuda.stream(side):
            wa = pa.forward(fa)
        wb = pb.forward(fb)
        torch.cuda.synchronize()
        # by tolerance, not bitwise: the forward SHT adds eight warps' partial sums with shared-memory atomics, in any
        # order (reading R16)
        assert float((wa - ref_a).abs().max()) <= 1e-12 * float(ref_a.abs().max())
        assert float((wb - ref_b).abs().max()) <= 1e-12 * float(ref_b.abs().max())
    back = pa.inverse(wa).cpu().numpy().reshape(f_a.shape)
    assert _relmax(back, f_a) < RT_TOL
    pa.close()
    pb.close()


@pytest.mark.parametrize("L,N,real", [(600, 3, True), (1100, 2, False)])
def test_large_band_limits_that_are_not_powers_of_two(L, N, real):
    """Ragged ring groups (20 and 36 groups of 32), three groups per warp, Bluestein lengths 4096 and 8192: recovered
    f_lm against the seeded truth, sampled rings against the oracle, wavelet round trip."""
    torch, api = _api()
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, 40 + L, 1)
    plan = api.s2wav_plan_create(L, N, 2.0, 3, True, real, 1)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    got = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(1, L, 2 * L - 1)
    assert _relmax(got, flm) < FWD_TOL
    rings = [0, 1, L // 3, L // 2, L - 2, L - 1]
    ref = S.sht_inverse(flm[0], L, "f80", thetas=S.mw_thetas(L, "f80")[rings])
    fn = f.cpu().numpy().reshape(L, 2 * L - 1)
    ref = ref.real.astype(np.float64) if real else ref.astype(np.complex128)
    assert np.abs(fn[rings] - ref).max() / np.abs(fn).max() < RT_TOL
    w = plan.forward(f)
    back = plan.inverse(w)
    assert float((back - f).abs().max() / f.abs().max()) < RT_TOL
    plan.close()


@pytest.mark.parametrize("N", [1, 2, 4, 5, 6])
def test_real_ring_pair_kernels_agree_with_the_complex_path_on_large_grids(N):
    """Real signals on grids with Bluestein length >= 4096 take the ring-pair (alpha, gamma) kernels (a8): with and
    without a row n = 0 (odd / even N), one or two rows n > 0 (parked in the output planes, no read-modify-write)
    and more than 9 gamma samples (N = 6: accumulating path).  The complex plan, which runs the ring-by-ring kernels
    checked against the oracle at small sizes, must give the same coefficients and the same synthesis."""
    torch, api = _api()
    L = 520
    flm = inputs.flm_real(L, 900 + N, 1)
    pr = api.s2wav_plan_create(L, N, 2.0, 7, True, True, 1)
    pc = api.s2wav_plan_create(L, N, 2.0, 7, True, False, 1)
    f = pr.harmonic_inverse(torch.from_numpy(flm).cuda())
    wr = pr.forward(f)
    wc = pc.forward(f.to(torch.complex128))
    scale = float(wc.abs().max())
    assert float(wc.imag.abs().max()) < 1e-12 * scale
    assert float((wr - wc.real).abs().max()) < 1e-12 * scale
    br = pr.inverse(wr)
    bc = pc.inverse(wc)
    fmax = float(f.abs().max())
    assert float((br - bc.real).abs().max()) < RT_TOL * fmax
    assert float((br - f).abs().max()) < RT_TOL * fmax
    pr.close()
    pc.close()
