"""Seeded synthetic inputs for the configurations of BASELINE.json (recipe: DESIGN.md "Inputs").

This module holds random-number draws and their shaping only -- none of the
transform arithmetic -- so that tests can hand the same arrays to the CUDA path
and to the oracle.  The paper benchmarks on random band-limited signals
(PAPER.md:370); these arrays are the harmonic coefficients of such signals.

Layouts: flm[(batch,) l, m + L-1]; flmp[p, l, m + L-1]; complex128.
"""
import hashlib

import numpy as np

# name -> parameters of BASELINE.json:configs[i]
CONFIGS = {
    "C1": dict(kind="sphere", L=32, N=1, lam=2.0, J0=0, multires=False, real=True, seed=0, batch=1,
               spectrum="white"),
    "C2": dict(kind="sphere", L=256, N=3, lam=2.0, J0=2, multires=True, real=False, seed=1, batch=1,
               spectrum="l^-2"),
    "C3": dict(kind="sphere", L=1024, N=5, lam=2.0, J0=2, multires=True, real=True, seed=2, batch=4,
               spectrum="l^-2"),
    "C4": dict(kind="sphere", L=2048, N=3, lam=2.0, J0=4, multires=True, real=True, seed=3, batch=1,
               spectrum="l^-2"),
    "C5": dict(kind="ball", L=128, P=128, N=3, lam=2.0, nu=2.0, J0=0, J0p=0, tau=1.0, real=False, seed=4,
               spectrum="l^-2 p^-1"),
    # not a BASELINE.json configuration: the shape of the paper's Table 2 (ball, N = 1, P = L) at its largest size
    "T2": dict(kind="ball", L=256, P=256, N=1, lam=2.0, nu=2.0, J0=0, J0p=0, tau=1.0, real=False, seed=5,
               spectrum="l^-2 p^-1"),
}


def flm_real(L, seed, batch=1, spectrum="l^-2"):
    """Coefficients of `batch` real band-limited fields: draws g[b][l][m>=0][re,im] from
    default_rng(seed).standard_normal; f_{l0} = g0 (real), f_{lm} = (g0 + i g1)/sqrt 2 for 0 < m <= l,
    f_{l,-m} = (-1)^m conj f_{lm}; amplitude 1/(l+1) for spectrum "l^-2" (C_l ~ (l+1)^-2), 1 for "white"."""
    g = np.random.default_rng(seed).standard_normal((batch, L, L, 2))
    amp = 1.0 / (np.arange(L) + 1.0) if spectrum == "l^-2" else np.ones(L)
    flm = np.zeros((batch, L, 2 * L - 1), dtype=np.complex128)
    for m in range(L):
        col = (g[:, :, m, 0] + 1j * g[:, :, m, 1]) / np.sqrt(2.0) if m > 0 else g[:, :, 0, 0].astype(np.complex128)
        col = col * amp[None, :]
        col[:, :m] = 0
        flm[:, :, L - 1 + m] = col
        if m > 0:
            flm[:, :, L - 1 - m] = (-1) ** m * np.conj(col)
    return flm


def flm_complex(L, seed, batch=1, spectrum="l^-2"):
    """Coefficients of complex fields: g[b][l][m+L-1][re,im] i.i.d. normal, f_{lm} = (g0 + i g1)/sqrt 2,
    |m| <= l, amplitude as in flm_real."""
    g = np.random.default_rng(seed).standard_normal((batch, L, 2 * L - 1, 2))
    amp = 1.0 / (np.arange(L) + 1.0) if spectrum == "l^-2" else np.ones(L)
    flm = (g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0) * amp[None, :, None]
    m = np.arange(-(L - 1), L)
    flm[:, np.abs(m)[None, :] > np.arange(L)[:, None]] = 0
    return flm


def flmp_complex(L, P, seed):
    """Ball coefficients: g[p][l][m+L-1][re,im] i.i.d. normal, amplitude 1/((l+1) sqrt(p+1))."""
    g = np.random.default_rng(seed).standard_normal((P, L, 2 * L - 1, 2))
    amp = 1.0 / ((np.arange(L) + 1.0)[None, :, None] * np.sqrt(np.arange(P) + 1.0)[:, None, None])
    flmp = (g[..., 0] + 1j * g[..., 1]) / np.sqrt(2.0) * amp
    m = np.arange(-(L - 1), L)
    flmp[:, np.abs(m)[None, :] > np.arange(L)[:, None]] = 0
    return flmp


def config_coefficients(name):
    """The harmonic coefficients of configuration `name` (C1..C5)."""
    c = CONFIGS[name]
    if c["kind"] == "ball":
        return flmp_complex(c["L"], c["P"], c["seed"])
    gen = flm_real if c["real"] else flm_complex
    return gen(c["L"], c["seed"], c["batch"], c["spectrum"])


def sha256(a):
    """Digest of an array's bytes (detects a change of numpy's random stream)."""
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
