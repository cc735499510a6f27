"""Pins of the oracle's wall-normal diffusion solve for the FACE-centred velocity component w
(Eq. 11, on the staggered grid of PAPER.md:49; reading R16): closed-form
eigenpairs on a uniform grid, the operator as gradient-of-divergence of the MAC grid (independent
code: oracle/projection.py), an independently assembled dense matrix, the maximum principle and
the a -> 0 limit.  No code is shared with the CUDA path."""
import numpy as np
import pytest

import oracle
from oracle import projection as proj
from paper_2502_06296_b200 import workloads as wl


def grid(nz, beta):
    zf = wl.z_faces(nz, 2.0, beta)
    return wl.z_centres(zf), zf


def dense_w_matrix(zc, zf, a):
    """I - a L_z^w assembled from the definition, independently of oracle.c: second difference of
    the face values, faces zf[1..nz-1] unknown, both wall faces 0; last row = identity."""
    nz = zc.size
    T = np.eye(nz)
    zface = zf[1:]                        # position of w_k
    for k in range(nz - 1):
        hm = zface[k] - (zface[k - 1] if k >= 1 else zf[0])     # distance to the face below = dzf_k
        hp = zface[k + 1] - zface[k]                               # to the face above = dzf_{k+1}
        hc = zc[k + 1] - zc[k]                                     # distance between the two cell centres
        T[k, k] += a * (1.0 / (hc * hm) + 1.0 / (hc * hp))
        if k >= 1:
            T[k, k - 1] -= a / (hc * hm)
        if k + 1 <= nz - 2:
            T[k, k + 1] -= a / (hc * hp)
    return T


@pytest.mark.parametrize("nz", [4, 9, 32])
def test_uniform_grid_eigenfunctions(nz):
    """Uniform grid, walls at the faces: w_k = sin(pi q (k+1)/nz) is an eigenvector of the second
    difference with eigenvalue -4 sin^2(pi q / (2 nz)) / dz^2."""
    zc, zf = grid(nz, 0.0)
    dz = 2.0 / nz
    a = 0.37
    for q in (1, 2, nz - 1):
        prof = np.sin(np.pi * q * (np.arange(nz) + 1) / nz)
        prof[-1] = 0.0                    # the top wall face
        r = np.tile(prof[:, None, None], (1, 3, 4))
        w = oracle.helmholtz_w_solve(zc, zf, a, r)
        expect = prof / (1.0 + a * 4.0 * np.sin(np.pi * q / (2 * nz)) ** 2 / dz ** 2)
        assert np.abs(w - expect[:, None, None]).max() <= 1e-14


@pytest.mark.parametrize("nz,beta", [(6, 0.0), (11, 1.8), (40, 2.0)])
def test_matrix_is_gradient_of_divergence_and_matches_dense_assembly(nz, beta):
    zc, zf = grid(nz, beta)
    a = 2.5e-3
    lo, di, up = oracle.helmholtz_w_matrix(zc, zf, a)
    T = np.diag(di) + np.diag(lo[1:], -1) + np.diag(up[:-1], 1)
    assert np.abs(T - dense_w_matrix(zc, zf, a)).max() <= 1e-12 * np.abs(T).max()
    # L_z^w = G_z D_z of the MAC grid: divergence of (0, 0, w) at the cell centres, then its z gradient
    rng = np.random.default_rng(nz)
    w = rng.standard_normal((nz, 2, 2))
    w[-1] = 0.0
    zero = np.zeros_like(w)
    d = proj.divergence(1.0, 1.0, zf, zero, zero, w)
    _, _, gz = proj.gradient(1.0, 1.0, zc, d)
    lw = (w - np.einsum("kl,lji->kji", T, w)) / a          # L_z^w w from the matrix
    assert np.abs(lw[:-1] - gz[:-1]).max() <= 1e-11 * np.abs(gz).max()


@pytest.mark.parametrize("nz,beta,a", [(7, 1.8, 1e-3), (33, 2.0, 5e-5), (64, 1.8, 10.0)])
def test_solve_matches_dense_lu_maximum_principle_and_small_a(nz, beta, a):
    zc, zf = grid(nz, beta)
    rng = np.random.default_rng(7 * nz)
    r = rng.standard_normal((nz, 3, 5))
    w = oracle.helmholtz_w_solve(zc, zf, a, r)
    T = dense_w_matrix(zc, zf, a)
    ref = np.linalg.solve(T, r.reshape(nz, -1)).reshape(r.shape)
    assert np.abs(w - ref).max() <= 1e-12 * np.abs(ref).max()
    assert np.array_equal(w[-1], r[-1])                    # the top wall face keeps its value
    assert np.abs(w).max() <= np.abs(r).max() * (1 + 1e-14)
    w0 = oracle.helmholtz_w_solve(zc, zf, 0.0, r)
    assert np.array_equal(w0, r)
