"""Thin ctypes binding over the C ABI of include/s2w.h -- argument marshalling only.

Every step of the transforms runs in the CUDA kernels of libs2w.so; PyTorch supplies device memory and streams.
The library must have been built (python -m paper_2402_01282_b200.build, or __graft_entry__.build()); importing
this module without it raises, and transforms fail with S2W_ECUDA when no GPU is present -- there is no CPU fallback.
"""
import ctypes
import os

import numpy as np

from . import build as _build

S2W_REAL = 1
S2W_PRECOMPUTE = 2
S2W_DH = 4
S2W_RECURSION = 8
S2W_STATIC_SCRATCH_BYTES = 32 << 20   # include/s2w.h: capacity of the static device scratch array
_ERRORS = {-1: "S2W_EINVAL", -2: "S2W_ENOMEM", -3: "S2W_ECUDA", -4: "S2W_EUNSUPPORTED"}

_c_int, _c_dbl, _c_vp, _c_sz = ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t
_pi = ctypes.POINTER(ctypes.c_int)

# name -> (restype, argtypes); the full export list of include/s2w.h
SIGNATURES = {
    "s2w_scale_count": (_c_int, [_c_int, _c_dbl, _pi]),
    "s2wav_kernels": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int]),
    "s2ball_kernels": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int]),
    "s2ball_radial_nodes": (_c_int, [_c_vp, _c_vp, _c_int, _c_dbl]),
    "s2wav_plan_create": (_c_int, [ctypes.POINTER(_c_vp), _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int,
                                   _c_int]),
    "s2wav_plan_create_spin": (_c_int, [ctypes.POINTER(_c_vp), _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int,
                                        _c_int, _c_int]),
    "s2ball_plan_create": (_c_int, [ctypes.POINTER(_c_vp), _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int, _c_dbl,
                                    _c_int, _c_int]),
    "s2w_plan_destroy": (_c_int, [_c_vp]),
    "s2w_plan_scales": (_c_int, [_c_vp, _pi, _pi, _pi, _pi]),
    "s2w_plan_scale_shape": (_c_int, [_c_vp, _c_int, _c_int, _pi, _pi, _pi, _pi, ctypes.POINTER(_c_sz)]),
    "s2w_plan_coeff_elems": (_c_sz, [_c_vp]),
    "s2w_plan_signal_elems": (_c_sz, [_c_vp]),
    "s2w_plan_workspace_bytes": (_c_sz, [_c_vp]),
    "s2w_plan_forward": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_inverse": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_forward_adjoint": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_inverse_adjoint": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_harmonic_forward": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_harmonic_inverse": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_vp]),
    "s2w_plan_harmonic_forward_static": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp]),
    "s2wav_forward": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int, _c_vp]),
    "s2wav_inverse": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int, _c_vp]),
    "s2ball_forward": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int, _c_dbl, _c_int, _c_vp]),
    "s2ball_inverse": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int, _c_dbl, _c_int, _c_vp]),
    "s2wav_forward_host": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int]),
    "s2wav_inverse_host": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_int, _c_int, _c_int]),
    "s2ball_forward_host": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int, _c_dbl, _c_int]),
    "s2ball_inverse_host": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_dbl, _c_int, _c_dbl, _c_int]),
    "s2ball_z_forward": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_vp]),
    "s2ball_z_inverse": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_vp]),
    "s2ball_q_forward": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_vp]),
    "s2ball_q_inverse": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_int, _c_dbl, _c_vp]),
    "s2w_cache_clear": (_c_int, []),
    "s2w_probe_fp64": (_c_int, [_c_int, _c_int, ctypes.POINTER(_c_dbl)]),
    "s2w_timing_enable": (_c_int, [_c_int]),
    "s2w_timing_read": (_c_int, [_c_vp, _c_vp, _c_int]),
    "s2w_launch_count": (ctypes.c_ulonglong, []),
    "s2w_last_error": (ctypes.c_char_p, []),
}

_LIB = None


def lib():
    """The loaded libs2w.so (raises if it has not been built)."""
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if not os.path.exists(path):
            raise RuntimeError("libs2w.so is missing: run `python -m paper_2402_01282_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _LIB = L
    return _LIB


class S2WError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        msg = lib().s2w_last_error()
        raise S2WError("%s: %s" % (_ERRORS.get(rc, rc), msg.decode() if msg else ""))


def _np_ptr(a):
    return a.ctypes.data_as(_c_vp)


# ------------------------------------------------------------------------------------------------
# kernel-build calls (host)
# ------------------------------------------------------------------------------------------------
def s2w_scale_count(L, lam):
    J = _c_int(0)
    _check(lib().s2w_scale_count(int(L), float(lam), ctypes.byref(J)))
    return J.value


def s2wav_kernels(L, N, lam, J0):
    """(psi [J-J0+1][L][2N-1] complex128, phi [L] float64)."""
    J = s2w_scale_count(L, lam)
    psi = np.zeros((max(J - J0 + 1, 0), L, 2 * N - 1), dtype=np.complex128)
    phi = np.zeros(L, dtype=np.float64)
    _check(lib().s2wav_kernels(_np_ptr(psi), _np_ptr(phi), int(L), int(N), float(lam), int(J0)))
    return psi, phi


def s2ball_kernels(L, P, N, lam_l, lam_p, J0):
    """dict(kappa_l [J-J0+1][L], kappa_p [J'-J0+1][P], zeta [L][2N-1] complex, phi [P][L])."""
    J, Jp = s2w_scale_count(L, lam_l), s2w_scale_count(P, lam_p)
    kl = np.zeros((max(J - J0 + 1, 0), L))
    kp = np.zeros((max(Jp - J0 + 1, 0), P))
    zeta = np.zeros((L, 2 * N - 1), dtype=np.complex128)
    phi = np.zeros((P, L))
    _check(lib().s2ball_kernels(_np_ptr(kl), _np_ptr(kp), _np_ptr(zeta), _np_ptr(phi), int(L), int(P), int(N),
                                float(lam_l), float(lam_p), int(J0)))
    return dict(kappa_l=kl, kappa_p=kp, zeta=zeta, phi=phi, J=J, Jp=Jp)


def s2ball_radial_nodes(P, tau):
    r = np.zeros(P)
    q = np.zeros(P)
    _check(lib().s2ball_radial_nodes(_np_ptr(r), _np_ptr(q), int(P), float(tau)))
    return r, q


# ------------------------------------------------------------------------------------------------
# plans
# ------------------------------------------------------------------------------------------------
def _torch():
    import torch
    return torch


def _stream_ptr(device=None):
    """The current stream of `device` (a tensor's device; default: the current device)."""
    torch = _torch()
    return _c_vp(torch.cuda.current_stream(device).cuda_stream)


def _dtype_real(dt):
    """True for float64 (S2W_REAL), False for complex128; any other dtype would be read out of bounds by the library."""
    name = str(dt).replace("torch.", "")
    if name == "float64":
        return True
    if name == "complex128":
        return False
    raise ValueError("expected float64 (real signals) or complex128, got %s" % dt)


def _whole(n, unit, what):
    if unit <= 0 or n == 0 or n % unit:
        raise ValueError("%s: %d elements is not a whole number of blocks of %d" % (what, n, unit))
    return n // unit


def _check_tensor(t, dtype, elems, what):
    """Argument marshalling guard: the library reads / writes `elems` elements of `dtype` behind the pointer."""
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype and t.numel() == elems):
        raise ValueError("%s: expected a contiguous CUDA tensor of dtype %s with %d elements, got %s %s with %d"
                         % (what, dtype, elems, "cuda" if t.is_cuda else "cpu", t.dtype, t.numel()))


class Plan:
    """Owner of a s2w_plan handle plus a torch workspace tensor.  Tensors in and out are torch CUDA tensors."""

    def __init__(self, handle, real, batch, kind):
        self._h = handle
        self.real = real
        self.batch = batch
        self.kind = kind
        L = lib()
        self.coeff_elems = int(L.s2w_plan_coeff_elems(self._h))
        self.signal_elems = int(L.s2w_plan_signal_elems(self._h))
        self.workspace_bytes = int(L.s2w_plan_workspace_bytes(self._h))
        j0, j, j0p, jp = _c_int(), _c_int(), _c_int(), _c_int()
        _check(L.s2w_plan_scales(self._h, ctypes.byref(j0), ctypes.byref(j), ctypes.byref(j0p), ctypes.byref(jp)))
        self.J0, self.J, self.J0p, self.Jp = j0.value, j.value, j0p.value, jp.value
        self._work = None

    @property
    def dtype(self):
        torch = _torch()
        return torch.float64 if self.real else torch.complex128

    def close(self):
        if self._h is not None:
            lib().s2w_plan_destroy(self._h)
            self._h = None
            self._work = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _workspace(self, device):
        torch = _torch()
        if self._work is None:
            self._work = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=device)
        return self._work

    def scale_shape(self, j, jp=0):
        """(n_r, n_gamma, n_theta, n_phi, offset_elems); j = -1 is the scaling block."""
        a, b, c, d, off = _c_int(), _c_int(), _c_int(), _c_int(), _c_sz()
        _check(lib().s2w_plan_scale_shape(self._h, int(j), int(jp), ctypes.byref(a), ctypes.byref(b),
                                          ctypes.byref(c), ctypes.byref(d), ctypes.byref(off)))
        return a.value, b.value, c.value, d.value, int(off.value)

    def scale_keys(self):
        if self.kind == "sphere":
            return [(j, 0) for j in range(self.J0, self.J + 1)]
        return [(j, jp) for jp in range(self.J0p, self.Jp + 1) for j in range(self.J0, self.J + 1)]

    def _check_in(self, t, elems, what="input"):
        _check_tensor(t, self.dtype, elems * self.batch, what)

    def _out(self, out, elems, like):
        torch = _torch()
        if out is None:
            return torch.empty((self.batch, elems), dtype=self.dtype, device=like.device)
        self._check_in(out, elems, "out")
        if out.device != like.device:
            raise ValueError("out: on %s, the input is on %s" % (out.device, like.device))
        return out

    def forward(self, f, out=None):
        """Analysis: signal(s) -> packed coefficient tensor [batch][coeff_elems]."""
        torch = _torch()
        self._check_in(f, self.signal_elems)
        out = self._out(out, self.coeff_elems, f)
        _check(lib().s2w_plan_forward(self._h, f.data_ptr(), out.data_ptr(), self._workspace(f.device).data_ptr(),
                                      _stream_ptr(f.device)))
        return out

    def inverse(self, w, out=None, shape=None):
        """Synthesis: packed coefficients -> signal(s)."""
        torch = _torch()
        self._check_in(w, self.coeff_elems)
        out = self._out(out, self.signal_elems, w)
        _check(lib().s2w_plan_inverse(self._h, w.data_ptr(), out.data_ptr(), self._workspace(w.device).data_ptr(),
                                      _stream_ptr(w.device)))
        return out if shape is None else out.view(shape)

    def forward_adjoint(self, y, out=None):
        """Adjoint of the analysis: coefficient-shaped y -> signal-shaped A^H y (s2w_plan_forward_adjoint)."""
        torch = _torch()
        self._check_in(y, self.coeff_elems)
        out = self._out(out, self.signal_elems, y)
        _check(lib().s2w_plan_forward_adjoint(self._h, y.data_ptr(), out.data_ptr(),
                                              self._workspace(y.device).data_ptr(), _stream_ptr(y.device)))
        return out

    def inverse_adjoint(self, g, out=None):
        """Adjoint of the synthesis: signal-shaped g -> coefficient-shaped S^H g (s2w_plan_inverse_adjoint)."""
        torch = _torch()
        self._check_in(g, self.signal_elems)
        out = self._out(out, self.coeff_elems, g)
        _check(lib().s2w_plan_inverse_adjoint(self._h, g.data_ptr(), out.data_ptr(),
                                              self._workspace(g.device).data_ptr(), _stream_ptr(g.device)))
        return out

    def harmonic_forward(self, f, flm_elems):
        torch = _torch()
        self._check_in(f, self.signal_elems)
        out = torch.empty((self.batch, flm_elems), dtype=torch.complex128, device=f.device)
        _check(lib().s2w_plan_harmonic_forward(self._h, f.data_ptr(), out.data_ptr(),
                                               self._workspace(f.device).data_ptr(), _stream_ptr(f.device)))
        return out

    def harmonic_forward_static(self, f, flm_elems, out=None):
        """s2w_plan_harmonic_forward_static: harmonic_forward with the scratch in the library's static device array
        (S2W_STATIC_SCRATCH_BYTES); `out` lets the caller pass the result buffer, so that nothing is allocated here."""
        torch = _torch()
        self._check_in(f, self.signal_elems)
        if out is None:
            out = torch.empty((self.batch, flm_elems), dtype=torch.complex128, device=f.device)
        elif not (out.is_cuda and out.is_contiguous() and out.dtype == torch.complex128
                  and out.numel() == self.batch * flm_elems and out.device == f.device):
            raise ValueError("out: expected a contiguous complex128 CUDA tensor of %d elements" % (self.batch * flm_elems))
        _check(lib().s2w_plan_harmonic_forward_static(self._h, f.data_ptr(), out.data_ptr(), _stream_ptr(f.device)))
        return out

    def harmonic_inverse(self, flm):
        torch = _torch()
        if flm.numel() % self.batch or not (flm.is_cuda and flm.is_contiguous() and flm.dtype == torch.complex128):
            raise ValueError("flm: expected a contiguous complex128 CUDA tensor [batch, ...]")
        out = torch.empty((self.batch, self.signal_elems), dtype=self.dtype, device=flm.device)
        _check(lib().s2w_plan_harmonic_inverse(self._h, flm.data_ptr(), out.data_ptr(),
                                               self._workspace(flm.device).data_ptr(), _stream_ptr(flm.device)))
        return out

    def split(self, w):
        """Views of a packed coefficient tensor: (scaling [batch, (P,) L_s, 2L_s-1], {(j, jp): [batch, (P_j',) 2N-1, L_j, 2L_j-1]})."""
        nr, ng, nt, npx, off = self.scale_shape(-1)
        shp = (self.batch, nt, npx) if self.kind == "sphere" else (self.batch, nr, nt, npx)
        scal = w[:, off:off + nr * nt * npx].reshape(shp)
        out = {}
        for (j, jp) in self.scale_keys():
            nr, ng, nt, npx, off = self.scale_shape(j, jp)
            shp = (self.batch, ng, nt, npx) if self.kind == "sphere" else (self.batch, nr, ng, nt, npx)
            out[(j, jp)] = w[:, off:off + nr * ng * nt * npx].reshape(shp)
        return scal, out


def s2wav_plan_create(L, N, lam, J0, multiresolution=True, real=False, batch=1, device=0, flags=0, spin=0):
    h = _c_vp()
    fl = int(flags) | (S2W_REAL if real else 0)
    if spin:
        _check(lib().s2wav_plan_create_spin(ctypes.byref(h), int(L), int(N), float(lam), int(J0),
                                            int(bool(multiresolution)), fl, int(batch), int(device), int(spin)))
    else:
        _check(lib().s2wav_plan_create(ctypes.byref(h), int(L), int(N), float(lam), int(J0),
                                       int(bool(multiresolution)), fl, int(batch), int(device)))
    return Plan(h, bool(real), int(batch), "sphere")


def s2ball_plan_create(L, P, N, lam_l, lam_p, J0, tau=1.0, real=False, device=0, flags=0):
    h = _c_vp()
    fl = int(flags) | (S2W_REAL if real else 0)
    _check(lib().s2ball_plan_create(ctypes.byref(h), int(L), int(P), int(N), float(lam_l), float(lam_p), int(J0),
                                    float(tau), fl, int(device)))
    return Plan(h, bool(real), 1, "ball")


# ------------------------------------------------------------------------------------------------
# the transforms named by the problem statement (device tensors in, device tensors out)
# ------------------------------------------------------------------------------------------------
_SIZE_CACHE = {}


def _coeff_elems_sphere(L, N, lam, J0, multires):
    key = (L, N, float(lam), J0, bool(multires))
    if key not in _SIZE_CACHE:
        J = s2w_scale_count(L, lam)

        def bl(e):
            if not multires:
                return L
            return int(min(int(np.ceil(float(lam) ** e - 1e-9)), L))
        Ls = bl(J0)
        tot = Ls * (2 * Ls - 1)
        for j in range(J0, J + 1):
            Lj = bl(j + 1)
            tot += (2 * N - 1) * Lj * (2 * Lj - 1)
        _SIZE_CACHE[key] = tot
    return _SIZE_CACHE[key]


def s2wav_forward(f, L, N, lam, J0, multiresolution=True):
    """f: CUDA tensor [batch, L, 2L-1] (float64 -> S2W_REAL, complex128 otherwise) -> packed coefficients [batch, K]."""
    torch = _torch()
    f = f.contiguous()
    batch = _whole(f.numel(), L * (2 * L - 1), "f")
    real = _dtype_real(f.dtype)
    K = _coeff_elems_sphere(L, N, lam, J0, multiresolution)
    w = torch.empty((batch, K), dtype=f.dtype, device=f.device)
    _check(lib().s2wav_forward(f.data_ptr(), w.data_ptr(), int(L), int(N), float(lam), int(J0),
                               int(bool(multiresolution)), S2W_REAL if real else 0, batch, _stream_ptr(f.device)))
    return w


def s2wav_inverse(w, L, N, lam, J0, multiresolution=True):
    """packed coefficients [batch, K] -> f [batch, L, 2L-1]."""
    torch = _torch()
    w = w.contiguous()
    K = _coeff_elems_sphere(L, N, lam, J0, multiresolution)
    batch = _whole(w.numel(), K, "w")
    real = _dtype_real(w.dtype)
    f = torch.empty((batch, L, 2 * L - 1), dtype=w.dtype, device=w.device)
    _check(lib().s2wav_inverse(w.data_ptr(), f.data_ptr(), int(L), int(N), float(lam), int(J0),
                               int(bool(multiresolution)), S2W_REAL if real else 0, batch, _stream_ptr(w.device)))
    return f


def _host_out(out, shape, dtype):
    """Caller-provided output (e.g. a view of pinned memory: copies are then asynchronous DMA) or a fresh array."""
    if out is None:
        return np.empty(shape, dtype=dtype)
    if out.dtype != dtype or out.size != int(np.prod(shape)) or not out.flags["C_CONTIGUOUS"]:
        raise ValueError("out must be a C-contiguous %s array of %d elements" % (dtype, int(np.prod(shape))))
    return out.reshape(shape)


def s2wav_forward_host(f, L, N, lam, J0, multiresolution=True, out=None):
    """numpy in, numpy out; host<->device copies happen inside the library call."""
    f = np.ascontiguousarray(f)
    real = _dtype_real(f.dtype)
    batch = _whole(f.size, L * (2 * L - 1), "f")
    K = _coeff_elems_sphere(L, N, lam, J0, multiresolution)
    w = _host_out(out, (batch, K), f.dtype)
    _check(lib().s2wav_forward_host(_np_ptr(f), _np_ptr(w), int(L), int(N), float(lam), int(J0),
                                    int(bool(multiresolution)), S2W_REAL if real else 0, batch))
    return w


def s2wav_inverse_host(w, L, N, lam, J0, multiresolution=True, out=None):
    w = np.ascontiguousarray(w)
    real = _dtype_real(w.dtype)
    K = _coeff_elems_sphere(L, N, lam, J0, multiresolution)
    batch = _whole(w.size, K, "w")
    f = _host_out(out, (batch, L, 2 * L - 1), w.dtype)
    _check(lib().s2wav_inverse_host(_np_ptr(w), _np_ptr(f), int(L), int(N), float(lam), int(J0),
                                    int(bool(multiresolution)), S2W_REAL if real else 0, batch))
    return f


def _coeff_elems_ball(L, P, N, lam_l, lam_p, J0):
    key = ("ball", L, P, N, float(lam_l), float(lam_p), J0)
    if key not in _SIZE_CACHE:
        J, Jp = s2w_scale_count(L, lam_l), s2w_scale_count(P, lam_p)

        def bl(lam, e, cap):
            return int(min(int(np.ceil(float(lam) ** e - 1e-9)), cap))
        tot = P * L * (2 * L - 1)
        for jp in range(J0, Jp + 1):
            Pj = bl(lam_p, jp + 1, P)
            for j in range(J0, J + 1):
                Lj = bl(lam_l, j + 1, L)
                tot += Pj * (2 * N - 1) * Lj * (2 * Lj - 1)
        _SIZE_CACHE[key] = tot
    return _SIZE_CACHE[key]


def s2ball_forward(f, L, P, N, lam_l, lam_p, J0, tau=1.0):
    """f: CUDA tensor [P, L, 2L-1] on the Gauss-Laguerre shells -> packed coefficients [K]."""
    torch = _torch()
    f = f.contiguous()
    real = _dtype_real(f.dtype)
    if not f.is_cuda or f.numel() != P * L * (2 * L - 1):
        raise ValueError("f: expected a CUDA tensor of %d elements [P, L, 2L-1]" % (P * L * (2 * L - 1)))
    w = torch.empty(_coeff_elems_ball(L, P, N, lam_l, lam_p, J0), dtype=f.dtype, device=f.device)
    _check(lib().s2ball_forward(f.data_ptr(), w.data_ptr(), int(L), int(P), int(N), float(lam_l), float(lam_p),
                                int(J0), float(tau), S2W_REAL if real else 0, _stream_ptr(f.device)))
    return w


def s2ball_inverse(w, L, P, N, lam_l, lam_p, J0, tau=1.0):
    torch = _torch()
    w = w.contiguous()
    real = _dtype_real(w.dtype)
    if not w.is_cuda or w.numel() != _coeff_elems_ball(L, P, N, lam_l, lam_p, J0):
        raise ValueError("w: expected a CUDA tensor of %d elements" % _coeff_elems_ball(L, P, N, lam_l, lam_p, J0))
    f = torch.empty((P, L, 2 * L - 1), dtype=w.dtype, device=w.device)
    _check(lib().s2ball_inverse(w.data_ptr(), f.data_ptr(), int(L), int(P), int(N), float(lam_l), float(lam_p),
                                int(J0), float(tau), S2W_REAL if real else 0, _stream_ptr(w.device)))
    return f


def s2ball_forward_host(f, L, P, N, lam_l, lam_p, J0, tau=1.0, out=None):
    f = np.ascontiguousarray(f)
    real = _dtype_real(f.dtype)
    w = _host_out(out, (_coeff_elems_ball(L, P, N, lam_l, lam_p, J0),), f.dtype)
    _check(lib().s2ball_forward_host(_np_ptr(f), _np_ptr(w), int(L), int(P), int(N), float(lam_l), float(lam_p),
                                     int(J0), float(tau), S2W_REAL if real else 0))
    return w


def s2ball_inverse_host(w, L, P, N, lam_l, lam_p, J0, tau=1.0, out=None):
    w = np.ascontiguousarray(w)
    real = _dtype_real(w.dtype)
    f = _host_out(out, (P, L, 2 * L - 1), w.dtype)
    _check(lib().s2ball_inverse_host(_np_ptr(w), _np_ptr(f), int(L), int(P), int(N), float(lam_l), float(lam_p),
                                     int(J0), float(tau), S2W_REAL if real else 0))
    return f


# ------------------------------------------------------------------------------------------------
# the generalised Fourier transforms on B^3 and H^4 as stand-alone calls (include/s2w.h)
# ------------------------------------------------------------------------------------------------
def s2ball_z_forward(f, L, P, tau=1.0):
    """Spherical-Laguerre transform Z (Eq. 10): f CUDA tensor [P, L, 2L-1] (float64 or complex128) -> f_lmp [P, L, 2L-1]."""
    torch = _torch()
    f = f.contiguous()
    real = _dtype_real(f.dtype)
    if not f.is_cuda or f.numel() != P * L * (2 * L - 1):
        raise ValueError("f: expected a CUDA tensor of %d elements [P, L, 2L-1]" % (P * L * (2 * L - 1)))
    out = torch.empty((P, L, 2 * L - 1), dtype=torch.complex128, device=f.device)
    _check(lib().s2ball_z_forward(f.data_ptr(), out.data_ptr(), int(L), int(P), float(tau), S2W_REAL if real else 0,
                                  _stream_ptr(f.device)))
    return out


def s2ball_z_inverse(flmp, L, P, tau=1.0, real=False):
    """Z^-1 (Eq. 11): f_lmp [P, L, 2L-1] complex128 -> f [P, L, 2L-1] (float64 if real)."""
    torch = _torch()
    flmp = flmp.contiguous()
    _check_tensor(flmp, torch.complex128, P * L * (2 * L - 1), "flmp")
    out = torch.empty((P, L, 2 * L - 1), dtype=torch.float64 if real else torch.complex128, device=flmp.device)
    _check(lib().s2ball_z_inverse(flmp.data_ptr(), out.data_ptr(), int(L), int(P), float(tau), S2W_REAL if real else 0,
                                  _stream_ptr(flmp.device)))
    return out


def s2ball_q_forward(f, L, P, N, tau=1.0):
    """Wigner-Laguerre transform Q = K D (Eq. 24): f [P, 2N-1, L, 2L-1] complex128 -> fhat [2N-1, P, L, 2L-1]."""
    torch = _torch()
    f = f.contiguous()
    _check_tensor(f, torch.complex128, P * (2 * N - 1) * L * (2 * L - 1), "f")
    out = torch.empty((2 * N - 1, P, L, 2 * L - 1), dtype=torch.complex128, device=f.device)
    _check(lib().s2ball_q_forward(f.data_ptr(), out.data_ptr(), int(L), int(P), int(N), float(tau),
                                  _stream_ptr(f.device)))
    return out


def s2ball_q_inverse(fhat, L, P, N, tau=1.0):
    """Q^-1 (Eq. 25): fhat [2N-1, P, L, 2L-1] complex128 -> f [P, 2N-1, L, 2L-1]."""
    torch = _torch()
    fhat = fhat.contiguous()
    _check_tensor(fhat, torch.complex128, P * (2 * N - 1) * L * (2 * L - 1), "fhat")
    out = torch.empty((P, 2 * N - 1, L, 2 * L - 1), dtype=torch.complex128, device=fhat.device)
    _check(lib().s2ball_q_inverse(fhat.data_ptr(), out.data_ptr(), int(L), int(P), int(N), float(tau),
                                  _stream_ptr(fhat.device)))
    return out


def probe_fp64(kind, device=0):
    """Measured TFLOP/s of a DFMA chain (kind 0) or an fp64 mma.sync chain (kind 1)."""
    v = _c_dbl(0.0)
    _check(lib().s2w_probe_fp64(int(kind), int(device), ctypes.byref(v)))
    return v.value


TIMING_CLASSES = ("wigner_inverse", "wigner_forward", "ring_fft", "so3_fft", "reweight", "radial", "other")


def timing_enable(on):
    _check(lib().s2w_timing_enable(int(bool(on))))


def timing_read():
    """{class name: (device ms, launches)} since the previous read (synchronises on the recorded events)."""
    ms = np.zeros(len(TIMING_CLASSES))
    cnt = np.zeros(len(TIMING_CLASSES), dtype=np.uint64)
    _check(lib().s2w_timing_read(_np_ptr(ms), _np_ptr(cnt), len(TIMING_CLASSES)))
    return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(TIMING_CLASSES)}


def launch_count():
    return int(lib().s2w_launch_count())
