"""oracle/adjoint.py -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py).

Adjoints of the sphere wavelet analysis A and synthesis S of oracle/sphere.py (the
"differentiable" half of arXiv:2402.01282: P:9, P:364, P:440 -- the transforms are linear,
so a vector-Jacobian product is the adjoint map).

The definition written out: with <u, v> = sum_i conj(u_i) v_i over the stored samples
(pixels of the MW grid / samples of every coefficient block, no quadrature weights), the
adjoint of a linear map with matrix M is the map with matrix M^H.  M is built column by
column by applying the oracle's own analysis / synthesis to the unit vectors -- no formula
for the adjoint is typed here, so there is nothing to get wrong but the packing and the
conjugation, which tests/test_oracle_adjoint.py pins through <A x, y> = <x, A^H y> with
A x computed directly.  Small band-limits only (one oracle transform per column).

Packing of a coefficient set into one vector: W^Phi, then W^{Psi j} for j = J0..J, each
C-ordered ([L_s][2L_s-1], [2N-1][L_j][2L_j-1]).
"""
import numpy as np

from . import sphere as S


def shapes(L, N, lam, J0, multires):
    """[(key, shape)] of the coefficient blocks in packing order; key -1 is the scaling block."""
    J = S.scale_range(L, lam, J0)
    Ls = S.bandlimit_of_scaling(L, lam, J0, multires)
    out = [(-1, (Ls, 2 * Ls - 1))]
    for j in range(J0, J + 1):
        Lj = S.bandlimit_of_scale(j, L, lam, multires)
        out.append((j, (2 * N - 1, Lj, 2 * Lj - 1)))
    return out


def pack(W_phi, W_psi, L, N, lam, J0, multires):
    parts = []
    for key, shp in shapes(L, N, lam, J0, multires):
        a = np.asarray(W_phi if key < 0 else W_psi[key])
        assert a.shape == shp, (key, a.shape, shp)
        parts.append(a.reshape(-1))
    return np.concatenate(parts)


def unpack(v, L, N, lam, J0, multires):
    W_phi, W_psi, o = None, {}, 0
    for key, shp in shapes(L, N, lam, J0, multires):
        n = int(np.prod(shp))
        a = v[o:o + n].reshape(shp)
        o += n
        if key < 0:
            W_phi = a
        else:
            W_psi[key] = a
    assert o == v.size
    return W_phi, W_psi


def analysis_matrix(L, N, lam, J0, multires, prec="f80"):
    """M[c][k] = (A e_k)_c: column k is the packed analysis of the k-th pixel unit vector."""
    filt = S.filters(L, N, lam, J0, prec)
    npix = L * (2 * L - 1)
    cols = []
    for k in range(npix):
        e = np.zeros(npix, dtype=S.CPLX[prec])
        e[k] = 1
        W_phi, W_psi = S.analysis(e.reshape(L, 2 * L - 1), L, N, lam, J0, multires, prec, filt)
        cols.append(pack(W_phi, W_psi, L, N, lam, J0, multires))
    return np.stack(cols, axis=1)


def synthesis_matrix(L, N, lam, J0, multires, prec="f80"):
    """M[k][c] = (S e_c)_k: column c is the synthesis of the c-th coefficient unit vector."""
    filt = S.filters(L, N, lam, J0, prec)
    ncoef = sum(int(np.prod(shp)) for _, shp in shapes(L, N, lam, J0, multires))
    cols = []
    for c in range(ncoef):
        e = np.zeros(ncoef, dtype=S.CPLX[prec])
        e[c] = 1
        W_phi, W_psi = unpack(e, L, N, lam, J0, multires)
        cols.append(np.asarray(S.synthesis(W_phi, W_psi, L, N, lam, J0, multires, prec, filt)).reshape(-1))
    return np.stack(cols, axis=1)


def analysis_adjoint(Y_phi, Y_psi, L, N, lam, J0, multires, prec="f80", matrix=None):
    """A^H y: coefficient-shaped (Y_phi, {j: Y_psi_j}) -> pixels [L][2L-1]."""
    M = analysis_matrix(L, N, lam, J0, multires, prec) if matrix is None else matrix
    y = pack(Y_phi, Y_psi, L, N, lam, J0, multires).astype(M.dtype)
    return (np.conj(M).T @ y).reshape(L, 2 * L - 1)


def synthesis_adjoint(g, L, N, lam, J0, multires, prec="f80", matrix=None):
    """S^H g: pixels [L][2L-1] -> coefficient-shaped (W_phi, {j: W_psi_j})."""
    M = synthesis_matrix(L, N, lam, J0, multires, prec) if matrix is None else matrix
    v = np.conj(M).T @ np.asarray(g).reshape(-1).astype(M.dtype)
    return unpack(v, L, N, lam, J0, multires)


# --------------------------------------------------------------------------
# ball (oracle/ball.py): the same definition.  A coefficient set is (W_phi [P][L][2L-1],
# {(j, j'): [P_j'][2N-1][L_j][2L_j-1]}), packed W_phi first, then the blocks in sorted key order.
# --------------------------------------------------------------------------
def ball_pack(W_phi, W_psi):
    return np.concatenate([np.asarray(W_phi).reshape(-1)] + [np.asarray(W_psi[k]).reshape(-1) for k in sorted(W_psi)])


def ball_analysis_adjoint_entries(Y_phi, Y_psi, entries, L, P, N, lam, nu, J0, J0p, tau, prec="f80"):
    """Sampled entries of A^H y on the ball: for each voxel index k (C order of [P][L][2L-1]) in `entries`,
    <A e_k, y> -- one oracle analysis each."""
    from . import ball as OB
    filt = OB.filters(L, P, N, lam, nu, J0, J0p, prec)
    y = ball_pack(Y_phi, Y_psi).astype(S.CPLX[prec])
    nvox = P * L * (2 * L - 1)
    out = []
    for k in entries:
        e = np.zeros(nvox, dtype=S.CPLX[prec])
        e[k] = 1
        W_phi, W_psi = OB.analysis(e.reshape(P, L, 2 * L - 1), L, P, N, lam, nu, J0, J0p, tau, prec, filt)
        out.append(np.vdot(ball_pack(W_phi, W_psi), y))
    return np.array(out)


def ball_synthesis_adjoint_entries(g, template, entries, L, P, N, lam, nu, J0, J0p, tau, prec="f80"):
    """Sampled entries of S^H g on the ball: for each packed coefficient index c in `entries`, <S e_c, g> (one oracle
    synthesis each).  `template` = (W_phi, W_psi) of the right shapes (values ignored)."""
    from . import ball as OB
    filt = OB.filters(L, P, N, lam, nu, J0, J0p, prec)
    T_phi, T_psi = template
    keys = sorted(T_psi)
    sizes = [int(np.asarray(T_phi).size)] + [int(np.asarray(T_psi[k]).size) for k in keys]
    ncoef = sum(sizes)
    gv = np.asarray(g).reshape(-1).astype(S.CPLX[prec])
    out = []
    for c in entries:
        e = np.zeros(ncoef, dtype=S.CPLX[prec])
        e[c] = 1
        o = sizes[0]
        W_phi = e[:o].reshape(np.asarray(T_phi).shape)
        W_psi = {}
        for k, n in zip(keys, sizes[1:]):
            W_psi[k] = e[o:o + n].reshape(np.asarray(T_psi[k]).shape)
            o += n
        f = OB.synthesis(W_phi, W_psi, L, P, N, lam, nu, J0, J0p, tau, prec, filt)
        out.append(np.vdot(np.asarray(f).reshape(-1), gv))
    return np.array(out)
