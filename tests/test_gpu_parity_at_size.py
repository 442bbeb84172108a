"""GPU parity at the sizes the big configurations run ("Next round" 1).

The Wigner contraction kernels are instantiated per block shape (R ring groups per warp, MAXT threads): grids with
G = 2 ceil(L_j / 64) ring groups run R = ceil(G / W) with W = min(G, 8) warps (G <= 32) or 16 warps (G > 32).  The small
parity cases only reach R = 1; the cases here reach every (R, MAXT) pair of the dispatch tables -- (2, 256) at L = 300,
(3, 256) at L = 600, (4, 256) at L = 1024 (BASELINE config 3), (3, 512) at L = 1100, (4, 512) at L = 1600 and at
L = 2048 (BASELINE config 4) -- for the on-the-fly kernels and for the precomputed-kernel variant (row a9,
S2W_PRECOMPUTE, P:358 / P:434), and compare sampled beta rings of the top scales with the long-double oracle
(oracle.sphere.analysis_from_flm(scales=, rings=) evaluates single rings with the same sums).
Tolerances: BASELINE.json's 1e-11 (forward, per scale block, reading R12) and 1e-12 (round trip)."""
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


def _check_sampled_rings(plan, w, flm_b, b, L, N, lam, J0, real, picks, filt=None):
    """Wavelet coefficients of signal b on the beta rings `picks` = [(j, [ring indices])] against the oracle."""
    scal, scales = plan.split(w)
    filt = S.filters(L, N, lam, J0, "f80") if filt is None else filt
    for j, rings in picks:
        _, o_psi = S.analysis_from_flm(flm_b, L, N, lam, J0, True, "f80", filt, scales=[j],
                                       rings={j: np.array(rings)})
        ref = o_psi[j]                                              # [2N-1][len(rings)][2L_j-1]
        if real:
            assert np.abs(ref.imag).max() <= 1e-13 * np.abs(ref).max()
            ref = ref.real.astype(np.float64)
        else:
            ref = ref.astype(np.complex128)
        blk = scales[(j, 0)][b]
        got = blk[:, rings, :].cpu().numpy()
        den = float(blk.abs().max())
        assert den > 0.0
        err = np.abs(got - ref).max() / den
        assert err < FWD_TOL, (j, err)


def _top_ring_picks(plan, Lj_of):
    out = []
    for j in (plan.J, plan.J - 1, plan.J - 2):
        if j < plan.J0:
            continue
        Lj = Lj_of(j)
        out.append((j, sorted({0, 1, Lj // 3, Lj // 2, Lj - 33, Lj - 2, Lj - 1})))
    return out


PRE_AT_SIZE = [
    # L, N, J0, real, batch      block shape of the top grid (R, MAXT)
    (300, 3, 4, True, 2),      # (2, 256), ragged last ring group
    (600, 2, 6, True, 1),      # (3, 256)
    (1024, 5, 2, True, 4),     # (4, 256): BASELINE config 3 with S2W_PRECOMPUTE, 24.6 GB table
    (1100, 2, 8, False, 1),    # (3, 512), complex: rows n = -1, +1 and the mirrored columns
    (1600, 2, 9, True, 1),     # (4, 512), single real column (half-empty column chunk)
]


@pytest.mark.parametrize("L,N,J0,real,batch", PRE_AT_SIZE)
def test_precomputed_kernel_variant_at_size(L, N, J0, real, batch):
    """Row a9 on the kernel instantiations the large grids dispatch: precomp_inverse_kernel<R, MAXT> and
    wigner_forward_kernel<R, MAXT, PRE> against (i) the oracle on sampled rings, (ii) the on-the-fly plan element by
    element, both directions, (iii) the round trip."""
    torch, api = _api()
    lam = 2.0
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, 700 + L + N, batch)
    otf = api.s2wav_plan_create(L, N, lam, J0, True, real, batch)
    f = otf.harmonic_inverse(torch.from_numpy(flm).cuda())
    w_otf = otf.forward(f)
    back_otf = otf.inverse(w_otf)
    fmax = float(f.abs().max())
    assert float((back_otf - f).abs().max()) < RT_TOL * fmax
    pre = api.s2wav_plan_create(L, N, lam, J0, True, real, batch, flags=api.S2W_PRECOMPUTE)
    w = pre.forward(f)
    scal_o, scales_o = otf.split(w_otf)
    scal_p, scales_p = pre.split(w)
    for key in scales_o:                                            # per scale block, as R12 measures
        den = float(scales_o[key].abs().max())
        assert float((scales_p[key] - scales_o[key]).abs().max()) <= 1e-12 * den, key
    assert float((scal_p - scal_o).abs().max()) <= 1e-12 * float(scal_o.abs().max())
    back = pre.inverse(w)
    assert float((back - f).abs().max()) < RT_TOL * fmax
    assert float((back - back_otf).abs().max()) < RT_TOL * fmax
    Lj_of = lambda j: pre.scale_shape(j)[2]
    b = batch - 1
    _check_sampled_rings(pre, w, flm[b], b, L, N, lam, J0, real, _top_ring_picks(pre, Lj_of))
    pre.close()
    otf.close()


@pytest.mark.parametrize("L,N,J0,real,batch", [(300, 3, 4, True, 2), (600, 2, 6, True, 1), (1100, 2, 8, False, 1),
                                               (1600, 2, 9, True, 1)])
def test_on_the_fly_kernels_at_size_sampled_rings(L, N, J0, real, batch):
    """The on-the-fly instantiations (R, MAXT) = (2, 256), (3, 256), (3, 512), (4, 512) against the oracle on sampled
    rings of the top scales ((4, 256) is test_config3_full_size_sampled_parity)."""
    torch, api = _api()
    lam = 2.0
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, 700 + L + N, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, real, batch)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    Lj_of = lambda j: plan.scale_shape(j)[2]
    _check_sampled_rings(plan, w, flm[0], 0, L, N, lam, J0, real, _top_ring_picks(plan, Lj_of))
    plan.close()


def test_config4_fused_top_scales_against_the_oracle():
    """BASELINE config 4 (L = 2048, N = 3, J0 = 4, real, batch 1), "run twice" (on the fly / precomputed kernels).
    On the fly, the two top scales share one recursion: wigner_inverse_kernel<.., 4, 512, NS = 2> and
    wigner_forward_kernel<4, 512, false, FUSE>.  Sampled rings of scales J and J-1 (poles, mid latitudes, the rings
    whose plain seeds underflow) against the oracle; then the S2W_PRECOMPUTE plan (about 118 GB of table)
    element by element against the on-the-fly coefficients and synthesis."""
    torch, api = _api()
    c = inputs.CONFIGS["C4"]
    L, N, lam, J0 = c["L"], c["N"], c["lam"], c["J0"]
    flm = inputs.config_coefficients("C4")
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, 1)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    back = plan.inverse(w)
    fmax = float(f.abs().max())
    assert float((back - f).abs().max()) < RT_TOL * fmax
    filt = S.filters(L, N, lam, J0, "f80")
    picks = [(plan.J, [0, 1, 156, 480, 1023, 1024, 1890, 2046, 2047]), (plan.J - 1, [0, 2, 157, 700, 1500, 2047]),
             (plan.J - 2, [0, 511, 1023])]
    _check_sampled_rings(plan, w, flm[0], 0, L, N, lam, J0, True, picks, filt)
    plan.close()
    try:
        pre = api.s2wav_plan_create(L, N, lam, J0, True, True, 1, flags=api.S2W_PRECOMPUTE)
    except api.S2WError as e:                                       # S2W_ENOMEM on a device with less HBM
        if "ENOMEM" in str(e):
            pytest.skip("the 118 GB table does not fit on this device")
        raise
    wp = pre.forward(f)
    _, so = pre.split(w)
    _, sp = pre.split(wp)
    for key in so:
        den = float(so[key].abs().max())
        assert float((sp[key] - so[key]).abs().max()) <= 1e-12 * den, key
    bp = pre.inverse(wp)
    assert float((bp - f).abs().max()) < RT_TOL * fmax
    assert float((bp - back).abs().max()) < RT_TOL * fmax
    pre.close()


@pytest.mark.parametrize("N", [1, 2, 4, 5, 6])
def test_real_ring_pair_kernels_against_the_oracle(N):
    """Row a8 for real signals on grids with Bluestein length >= 4096 (so3_*_pair_kernel): with / without a row n = 0
    (odd / even N), parked rows, more than 9 gamma samples (N = 6).  Sampled rings (both rings of a pair, the unpaired
    last ring) of the two top scales against the oracle; synthesis through the round trip."""
    torch, api = _api()
    L, lam, J0 = 520, 2.0, 8
    flm = inputs.flm_real(L, 900 + N, 1)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, 1)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    picks = [(plan.J, [0, 1, 2, 3, 258, 259, 518, 519]), (plan.J - 1, [0, 1, 300, 301, 519])]
    _check_sampled_rings(plan, w, flm[0], 0, L, N, lam, J0, True, picks)
    back = plan.inverse(w)
    assert float((back - f).abs().max()) < RT_TOL * float(f.abs().max())
    plan.close()


@pytest.mark.parametrize("N", [1, 2, 3])
def test_alpha_gamma_prime_factor_255(N):
    """Row a8 on grids with 2 L_j - 1 = 255 = 3 x 5 x 17 alpha samples (complex signals, 1 to 3 rows n): the prime-factor
    kernels of pfa255_kernels.cu.  L = 128, complex, two signals: sampled rings (poles, equator, ragged last block of 15 / nn
    rings) of the two scales with L_j = 128 against the oracle; synthesis through the round trip."""
    torch, api = _api()
    L, lam, J0, batch = 128, 2.0, 5, 2
    flm = inputs.flm_complex(L, 1300 + N, batch)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, False, batch)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    picks = [(plan.J, [0, 1, 4, 5, 63, 64, 120, 124, 125, 126, 127]), (plan.J - 1, [0, 2, 77, 127])]
    for b in range(batch):
        _check_sampled_rings(plan, w, flm[b], b, L, N, lam, J0, False, picks)
    back = plan.inverse(w)
    assert float((back - f).abs().max()) < RT_TOL * float(f.abs().max())
    plan.close()


@pytest.mark.parametrize("N", [1, 2, 4, 5])
def test_alpha_gamma_prime_factor_4095(N):
    """Row a8 for real signals on the grid of L_j = 2048 (4095 = 9 x 5 x 7 x 13 alpha samples): the prime-factor kernels of
    pfa4095_kernels.cu with no row n > 0 (N = 1), without a row n = 0 (even N), with parked rows (N = 4, 5); N = 3 is
    test_config4_fused_top_scales_against_the_oracle.  Sampled rings (both rings of a pair, the last pair) of the top scale
    against the oracle; synthesis through the round trip."""
    torch, api = _api()
    L, lam, J0 = 2048, 2.0, 10
    flm = inputs.flm_real(L, 1400 + N, 1)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, 1)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    w = plan.forward(f)
    picks = [(plan.J, [0, 1, 1026, 1027, 2046, 2047])]
    _check_sampled_rings(plan, w, flm[0], 0, L, N, lam, J0, True, picks)
    back = plan.inverse(w)
    assert float((back - f).abs().max()) < RT_TOL * float(f.abs().max())
    plan.close()


@pytest.mark.parametrize("N", [1, 2, 3, 4])
def test_alpha_gamma_prime_factor_2047(N):
    """Row a8 (and a1) for real signals on the grid of L_j = 1024 (2047 = 23 x 89 alpha samples): the prime-factor kernels with
    the Rader 89-point stage (pfa4095_kernels.cu), with no row n > 0 (N = 1), without a row n = 0 (even N), with a parked
    row (N = 4); N = 5 is test_config3_full_size_sampled_parity.  Recovered f_lm against the seeded truth (ring FFTs),
    sampled rings (both rings of a pair, the last pair) of the top scale against the oracle, synthesis through the round trip."""
    torch, api = _api()
    L, lam, J0 = 1024, 2.0, 9
    flm = inputs.flm_real(L, 1500 + N, 2)
    plan = api.s2wav_plan_create(L, N, lam, J0, True, True, 2)
    f = plan.harmonic_inverse(torch.from_numpy(flm).cuda())
    got = plan.harmonic_forward(f, L * (2 * L - 1)).cpu().numpy().reshape(2, L, 2 * L - 1)
    assert np.abs(got - flm).max() / np.abs(flm).max() < FWD_TOL
    w = plan.forward(f)
    picks = [(plan.J, [0, 1, 514, 515, 1022, 1023])]
    _check_sampled_rings(plan, w, flm[1], 1, L, N, lam, J0, True, picks)
    back = plan.inverse(w)
    assert float((back - f).abs().max()) < RT_TOL * float(f.abs().max())
    plan.close()
