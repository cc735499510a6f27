"""Pins of oracle/bc.py (Poisson solve with Fourier / cosine / sine expansions and Neumann /
Dirichlet walls; reading R17): the bases are eigenvectors of the stencil
with the closed-form eigenvalues and are orthogonal; the periodic / Neumann case equals oracle.c
(complex DFTs, a different program); every combination round-trips through the operator applied
from the stencil with ghost values; tiny grids against dense LU of that operator; closed-form
eigenfunctions; zero volume mean where the problem is singular."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import bc
from paper_2502_06296_b200 import workloads as wl


def grid(nz, beta):
    zf = wl.z_faces(nz, 2.0, beta)
    return wl.z_centres(zf), zf


@pytest.mark.parametrize("n", [4, 7, 12, 30])
@pytest.mark.parametrize("kind", ["P", "N", "D"])
def test_bases_are_orthogonal_eigenvectors_of_the_stencil(n, kind):
    T, n2, lam = bc.basis(n, kind)
    assert T.shape == (n, n)
    G = T @ T.T
    assert np.abs(G - np.diag(n2)).max() <= 1e-12 * n
    for q in range(n):
        v = T[q]
        lo, hi = np.roll(v, 1), np.roll(v, -1)
        if kind != "P":
            s = 1.0 if kind == "N" else -1.0
            lo[0], hi[-1] = s * v[0], s * v[-1]
        assert np.abs(lo - 2 * v + hi - lam[q] * v).max() <= 1e-12
    assert (lam <= 1e-15).all() and ((lam == 0).sum() == (0 if kind == "D" else 1))


@pytest.mark.parametrize("nx,ny,nz,beta", [(8, 6, 5, 0.0), (12, 16, 9, 1.8), (32, 16, 24, 2.0)])
def test_periodic_neumann_case_equals_oracle_c(nx, ny, nz, beta):
    zc, zf = grid(nz, beta)
    f = wl.remove_weighted_mean(np.random.default_rng(nx + nz).standard_normal((nz, ny, nx)), zf)
    a = bc.poisson_solve(2.0, 3.0, zc, zf, f, "P", "P", "NN")
    b = oracle.poisson_solve(2.0, 3.0, zc, zf, f, 0)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(b).max()
    assert np.abs(bc.apply_operator(2.0, 3.0, zc, zf, b) - oracle.apply_poisson_operator(2.0, 3.0, zc, zf, b)).max() <= 1e-11 * np.abs(f).max()


COMBOS = [c for c in itertools.product("PND", "PND", ["NN", "DD", "ND", "DN"])]


@pytest.mark.parametrize("bcx,bcy,bcz", COMBOS)
def test_apply_then_solve_round_trip_on_a_stretched_grid(bcx, bcy, bcz):
    nx, ny, nz = 10, 8, 11
    zc, zf = grid(nz, 1.8)
    rng = np.random.default_rng(sum(map(ord, bcx + bcy + bcz)))
    phi = rng.standard_normal((nz, ny, nx))
    singular = "D" not in (bcx + bcy + bcz)
    if singular:
        phi = wl.remove_weighted_mean(phi, zf)
    f = bc.apply_operator(1.7, 2.3, zc, zf, phi, bcx, bcy, bcz)
    got = bc.poisson_solve(1.7, 2.3, zc, zf, f, bcx, bcy, bcz)
    assert np.abs(got - phi).max() <= 1e-11 * np.abs(phi).max()
    if singular:
        dzf = np.diff(zf)
        assert abs(np.dot(dzf, got.mean(axis=(1, 2)))) <= 1e-13 * np.abs(got).max()


@pytest.mark.parametrize("bcx,bcy,bcz", [("N", "P", "DD"), ("D", "N", "ND"), ("P", "D", "NN"), ("D", "D", "DN")])
def test_tiny_grid_against_dense_lu_of_the_stencil(bcx, bcy, bcz):
    nx, ny, nz = 4, 3, 5
    zc, zf = grid(nz, 2.0)
    n = nx * ny * nz
    L = np.empty((n, n))
    for c in range(n):
        e = np.zeros(n)
        e[c] = 1.0
        L[:, c] = bc.apply_operator(1.0, 0.8, zc, zf, e.reshape(nz, ny, nx), bcx, bcy, bcz).ravel()
    f = np.random.default_rng(1).standard_normal((nz, ny, nx))
    ref = np.linalg.solve(L, f.ravel()).reshape(f.shape)
    got = bc.poisson_solve(1.0, 0.8, zc, zf, f, bcx, bcy, bcz)
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()


def test_uniform_grid_closed_form_eigenfunction():
    """cos in x (Neumann), sin in y (Dirichlet), sin in z (Dirichlet walls): eigenvalue in closed form."""
    nx, ny, nz, lx, ly = 12, 10, 8, 3.0, 2.0
    zc, zf = grid(nz, 0.0)
    i, j, k = np.arange(nx) + 0.5, np.arange(ny) + 0.5, np.arange(nz) + 0.5
    p, q, r = 3, 2, 4
    mode = (np.sin(np.pi * r * k / nz)[:, None, None] * np.sin(np.pi * q * j / ny)[None, :, None]
            * np.cos(np.pi * p * i / nx)[None, None, :])
    mu = (-4 * np.sin(np.pi * p / (2 * nx)) ** 2 / (lx / nx) ** 2 - 4 * np.sin(np.pi * q / (2 * ny)) ** 2 / (ly / ny) ** 2
          - 4 * np.sin(np.pi * r / (2 * nz)) ** 2 / (2.0 / nz) ** 2)
    got = bc.poisson_solve(lx, ly, zc, zf, mu * mode, "N", "D", "DD")
    assert np.abs(got - mode).max() <= 1e-13
