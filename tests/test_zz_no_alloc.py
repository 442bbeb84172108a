"""The allocation-free entry point s2w_plan_harmonic_forward_static (include/s2w.h): the forward spherical harmonic
transform (steps a1-a3; Eq. 2) with its scratch in the library's static device array instead of a caller workspace.

Collected last on purpose (test_zz_*): the suite runs with pytest -x, and a failure here must not hide other tests.
Checks: (i) two (and more) calls in a row, on plans of different shape so that each call finds the previous call's
leftovers in the shared array, against the existing path (s2w_plan_harmonic_forward with a caller workspace) -- the
kernels are the same, so the bar is 1e-12 of the largest coefficient, ten times tighter than the 1e-11 of the forward
parity tests; (ii) against the seeded f_lm the signal was synthesised from and the long-double oracle (1e-11, BASELINE.json);
(iii) plans that need more than S2W_STATIC_SCRATCH_BYTES, and ball plans, are rejected with a clear message;
(iv) the free device memory does not move across calls."""
import numpy as np
import pytest

from oracle import sphere as S
from paper_2402_01282_b200 import inputs

pytestmark = pytest.mark.gpu

FWD_TOL = 1e-11
SAME_KERNELS_TOL = 1e-12


def _api():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2402_01282_b200 import api
    return torch, api


def _relmax(a, b):
    den = float(b.abs().max())
    num = float((a - b).abs().max())
    return num if den == 0 else num / den


def _make(torch, api, L, N, real, batch, seed, flags=0):
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = torch.from_numpy(gen(L, seed, batch)).cuda().reshape(batch, -1)
    plan = api.s2wav_plan_create(L, N, 2.0, 0, True, real, batch, flags=flags)
    f = plan.harmonic_inverse(flm)                                  # pixels with exactly these f_lm (existing path)
    return plan, flm, f, L * (2 * L - 1)


def test_static_scratch_two_calls_in_a_row_match_the_workspace_path():
    torch, api = _api()
    shapes = [(96, 2, False, 2, 0), (64, 1, True, 1, 0), (200, 1, True, 3, 0), (40, 1, True, 2, api.S2W_DH)]
    made = [_make(torch, api, L, N, real, batch, 4100 + L, flags) for (L, N, real, batch, flags) in shapes]
    # the existing path first, for every plan
    want = [plan.harmonic_forward(f, n) for plan, _, f, n in made]
    torch.cuda.synchronize()
    # back-to-back calls on the shared array, no synchronisation in between, shapes alternating; then once more
    order = [0, 1, 0, 2, 3, 1, 2]
    got = [made[i][0].harmonic_forward_static(made[i][2], made[i][3]) for i in order]
    torch.cuda.synchronize()
    for i, g in zip(order, got):
        assert _relmax(g, want[i]) <= SAME_KERNELS_TOL, (shapes[i], _relmax(g, want[i]))
        assert _relmax(g, made[i][1]) < FWD_TOL, shapes[i]
    # the same call twice in a row on one plan gives the same answer twice
    plan, flm, f, n = made[0]
    a = plan.harmonic_forward_static(f, n)
    b = plan.harmonic_forward_static(f, n)
    assert _relmax(a, want[0]) <= SAME_KERNELS_TOL and _relmax(b, want[0]) <= SAME_KERNELS_TOL
    for plan, _, _, _ in made:
        plan.close()


def test_static_scratch_against_the_oracle():
    torch, api = _api()
    L, batch = 48, 2
    flm = inputs.flm_complex(L, 4200, batch)
    f = np.stack([S.sht_inverse(flm[b], L, "f80") for b in range(batch)]).astype(np.complex128)
    plan = api.s2wav_plan_create(L, 1, 2.0, 0, True, False, batch)
    fd = torch.from_numpy(np.ascontiguousarray(f)).cuda().reshape(batch, -1)
    for _ in range(2):                                              # two calls in a row
        got = plan.harmonic_forward_static(fd, L * (2 * L - 1)).cpu().numpy().reshape(batch, L, 2 * L - 1)
        for b in range(batch):
            ref = S.sht_forward(f[b], L, "f80").astype(np.complex128)
            assert np.abs(got[b] - ref).max() / np.abs(ref).max() < FWD_TOL
            assert np.abs(got[b] - flm[b]).max() / np.abs(flm[b]).max() < FWD_TOL
    plan.close()


def test_static_scratch_allocates_nothing():
    torch, api = _api()
    plan, flm, f, n = _make(torch, api, 128, 2, True, 2, 4300)
    out = torch.empty((plan.batch, n), dtype=torch.complex128, device=f.device)
    want = plan.harmonic_forward(f, n)
    plan.harmonic_forward_static(f, n, out=out)                     # first call: kernels loaded, symbol address resolved
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        plan.harmonic_forward_static(f, n, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    assert _relmax(out, want) <= SAME_KERNELS_TOL
    plan.close()


def test_static_scratch_rejects_what_does_not_fit():
    torch, api = _api()
    # complex, N = 1, batch = 1: 16 B * 3 L (2L-1) exceeds 32 MiB from L = 592 on (include/s2w.h)
    L = 640
    need = 16 * 3 * ((L * (2 * L - 1) + 15) // 16 * 16)
    assert need > api.S2W_STATIC_SCRATCH_BYTES
    plan = api.s2wav_plan_create(L, 1, 2.0, 0, True, False, 1)
    f = torch.zeros((1, L * (2 * L - 1)), dtype=torch.complex128, device="cuda")
    with pytest.raises(api.S2WError) as e:
        plan.harmonic_forward_static(f, L * (2 * L - 1))
    assert "S2W_EINVAL" in str(e.value) and "S2W_STATIC_SCRATCH_BYTES" in str(e.value) and str(need) in str(e.value)
    # the caller-workspace path still serves that plan
    assert float(plan.harmonic_forward(f, L * (2 * L - 1)).abs().max()) == 0.0
    plan.close()
    ball = api.s2ball_plan_create(16, 8, 1, 2.0, 2.0, 0, 1.0)
    fb = torch.zeros((1, 8 * 16 * 31), dtype=torch.complex128, device="cuda")
    with pytest.raises(api.S2WError) as e:
        ball.harmonic_forward_static(fb, 8 * 16 * 31)
    assert "S2W_EUNSUPPORTED" in str(e.value)
    ball.close()
