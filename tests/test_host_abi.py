"""CPU tests of the boundary: the C-ABI library builds, loads and exports every symbol include/s2w.h declares; the host
kernel-build calls (filters, Gauss-Laguerre nodes, scale bookkeeping) agree with the oracle; argument errors come back
as codes; and, with no GPU, every transform fails loudly (there is no CPU fallback).  No compute call needs a device."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import ball as OB
from oracle import sphere as S
from paper_2402_01282_b200 import api
from paper_2402_01282_b200 import build as lib_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "s2w.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+)?[A-Za-z_][\w\s\*]*?\b(s2\w+)\s*\(", text, flags=re.M)
    return sorted(set(names))


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = lib_build.build()
    assert os.path.exists(path)
    raw = ctypes.CDLL(path)
    names = _declared_symbols()
    assert len(names) >= 30, names
    for name in names:
        assert hasattr(raw, name), "libs2w.so does not export %s" % name
    # the binding marshals exactly the declared calls
    assert sorted(api.SIGNATURES) == names
    assert api.lib() is not None


def test_binding_constants_match_the_header():
    """The flag bits and the static-scratch capacity of the binding are the header's."""
    text = open(os.path.join(ROOT, "include", "s2w.h")).read()
    enum = re.search(r"enum\s*\{\s*S2W_REAL[^}]*\}", text).group(0)
    flags = {k: int(v) for k, v in re.findall(r"(S2W_[A-Z_]+)\s*=\s*(\d+)", enum)}
    assert flags == {"S2W_REAL": api.S2W_REAL, "S2W_PRECOMPUTE": api.S2W_PRECOMPUTE, "S2W_DH": api.S2W_DH,
                     "S2W_RECURSION": api.S2W_RECURSION}
    assert len(set(flags.values())) == 4 and all(v & (v - 1) == 0 for v in flags.values())   # distinct single bits
    m = re.search(r"#define\s+S2W_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", text)
    assert int(m.group(1)) << int(m.group(2)) == api.S2W_STATIC_SCRATCH_BYTES
    errs = re.search(r"enum\s*\{\s*S2W_OK[^}]*\}", text).group(0)
    codes = {k: int(v) for k, v in re.findall(r"(S2W_E[A-Z]+)\s*=\s*(-?\d+)", errs)}
    assert codes == {v: k for k, v in api._ERRORS.items()}


def test_scale_count_and_error_codes_without_a_device():
    assert api.s2w_scale_count(1024, 2.0) == 10
    assert api.s2w_scale_count(9, 2.0) == 4
    assert api.s2w_scale_count(128, 3.0) == 5
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2wav_kernels(8, 9, 2.0, 0)        # N > L
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2wav_kernels(8, 2, 1.0, 0)        # lambda <= 1
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2wav_kernels(8, 2, 2.0, 9)        # J0 > J
    with pytest.raises(api.S2WError, match="S2W_EINVAL"):
        api.s2ball_radial_nodes(0, 1.0)
    assert isinstance(api.lib().s2w_last_error(), bytes)


@pytest.mark.parametrize("L,N,lam,J0", [(32, 1, 2.0, 0), (64, 5, 2.0, 2), (40, 4, 1.7, 1), (27, 3, 3.0, 0)])
def test_sphere_kernels_match_oracle_filters(L, N, lam, J0):
    """s2wav_kernels (host C++, Gauss-Legendre quadrature of Eq. A4 in long double) against the oracle's Appendix A."""
    psi, phi = api.s2wav_kernels(L, N, lam, J0)
    o_psi, o_phi, J = S.filters(L, N, lam, J0, "f80")
    assert psi.shape == (J - J0 + 1, L, 2 * N - 1)
    assert np.abs(psi - np.asarray(o_psi, dtype=np.complex128)).max() < 1e-14
    assert np.abs(phi - np.asarray(o_phi, dtype=np.float64)).max() < 1e-14
    # admissibility (Eq. 30): 4pi/(2l+1) |Phi_l0|^2 + 8pi^2/(2l+1) sum_j sum_n |Psi^j_ln|^2 = 1
    ell = np.arange(L)
    tot = 4 * np.pi / (2 * ell + 1) * phi ** 2 + 8 * np.pi ** 2 / (2 * ell + 1) * (np.abs(psi) ** 2).sum(axis=(0, 2))
    assert np.abs(tot - 1).max() < 1e-13


def test_ball_kernels_and_radial_nodes_match_oracle():
    L, P, N, lam, nu, J0 = 24, 20, 3, 2.0, 2.0, 0
    k = api.s2ball_kernels(L, P, N, lam, nu, J0)
    o = OB.filters(L, P, N, lam, nu, J0, J0, "f80")
    assert np.abs(k["kappa_l"] - np.asarray(o["kap_l"], dtype=np.float64)).max() < 1e-14
    assert np.abs(k["kappa_p"] - np.asarray(o["kap_p"], dtype=np.float64)).max() < 1e-14
    assert np.abs(k["zeta"] - np.asarray(o["zeta"], dtype=np.complex128)).max() < 1e-14
    assert np.abs(k["phi"] - np.asarray(o["phi"], dtype=np.float64)).max() < 1e-14
    for Pn, tau in [(1, 1.0), (7, 0.5), (64, 1.0), (128, 2.0)]:
        r, q = api.s2ball_radial_nodes(Pn, tau)
        o_r, o_q = OB.radial_nodes(Pn, tau, "f80")
        assert np.abs(r / np.asarray(o_r, dtype=np.float64) - 1).max() < 1e-14
        assert np.abs(q / np.asarray(o_q, dtype=np.float64) - 1).max() < 1e-12


def test_no_cpu_fallback():
    """Without a CUDA device every plan creation / transform returns S2W_ECUDA; nothing is computed on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(api.S2WError, match="S2W_ECUDA"):
        api.s2wav_plan_create(8, 2, 2.0, 0)
    with pytest.raises(api.S2WError, match="S2W_ECUDA"):
        api.s2ball_plan_create(8, 4, 2, 2.0, 2.0, 0)
    f = np.zeros((1, 8, 15))
    with pytest.raises(api.S2WError, match="S2W_ECUDA"):
        api.s2wav_forward_host(f, 8, 2, 2.0, 0)


def test_binding_rejects_dtypes_and_sizes_the_library_would_read_out_of_bounds():
    """the argument-style wrappers inferred `real` from dtype == float64 and took anything else as
    complex128; a float32 / complex64 array was then read out of bounds.  The marshalling layer now refuses."""
    import numpy as np
    import pytest
    from paper_2402_01282_b200 import api
    assert api._dtype_real(np.dtype("float64")) is True and api._dtype_real(np.dtype("complex128")) is False
    for bad in ("float32", "complex64", "int64"):
        with pytest.raises(ValueError):
            api._dtype_real(np.dtype(bad))
    with pytest.raises(ValueError):
        api.s2wav_forward_host(np.zeros((1, 8, 15), dtype=np.float32), 8, 2, 2.0, 0)
    with pytest.raises(ValueError):
        api.s2wav_forward_host(np.zeros((8, 14)), 8, 2, 2.0, 0)          # not a whole number of L x (2L-1) signals
    with pytest.raises(ValueError):
        api.s2wav_inverse_host(np.zeros(17), 8, 2, 2.0, 0)
