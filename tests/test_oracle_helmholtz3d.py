"""Pins for the oracle's fully implicit (3-D) Helmholtz solve, definition O-H3 (
Eq. 8): (I - a L_h) u = r, periodic x, y, Dirichlet walls in z."""
import numpy as np
import pytest

import oracle
from paper_2502_06296_b200 import workloads as wl

LD = np.longdouble


def apply_longdouble(u, lx, ly, zc, zf, a):
    """(I - a L_h) u in long double from the definition (independent of oracle.c)."""
    p = u.astype(LD)
    nz, ny, nx = p.shape
    zc, zf = np.asarray(zc, LD), np.asarray(zf, LD)
    dzf = zf[1:] - zf[:-1]
    dzc = zc[1:] - zc[:-1]
    dx, dy = LD(lx) / nx, LD(ly) / ny
    lap = (np.roll(p, -1, 2) - 2 * p + np.roll(p, 1, 2)) / dx ** 2
    lap += (np.roll(p, -1, 1) - 2 * p + np.roll(p, 1, 1)) / dy ** 2
    lap[1:] += (1 / (dzf[1:] * dzc))[:, None, None] * (p[:-1] - p[1:])
    lap[:-1] += (1 / (dzf[:-1] * dzc))[:, None, None] * (p[1:] - p[:-1])
    # Dirichlet walls: ghost value = -interior value, wall on the face
    lap[0] -= 2 / (dzf[0] * 2 * (zc[0] - zf[0])) * p[0]
    lap[-1] -= 2 / (dzf[-1] * 2 * (zf[-1] - zc[-1])) * p[-1]
    return p - LD(a) * lap


def dense_matrix(nx, ny, nz, lx, ly, zc, zf, a):
    n = nx * ny * nz
    M = np.zeros((n, n))
    e = np.zeros((nz, ny, nx))
    for r in range(n):
        e.flat[r] = 1.0
        M[:, r] = apply_longdouble(e, lx, ly, zc, zf, a).astype(np.float64).ravel()
        e.flat[r] = 0.0
    return M


@pytest.mark.parametrize("modes", [(0, 0, 1), (1, 0, 1), (0, 3, 2), (5, 7, 9), (8, 8, 16)])
@pytest.mark.parametrize("a", [5e-5, 0.2])
def test_uniform_grid_eigenfunctions(modes, a):
    """cos(2 pi p i/nx) cos(2 pi r j/ny) sin(pi q (k+1/2)/nz) is an eigenfunction of L_h with
    mu = -4 sin^2(pi p/nx)/dx^2 - 4 sin^2(pi r/ny)/dy^2 - 4 sin^2(pi q/(2 nz))/dz^2."""
    nx = ny = nz = 16
    lx, ly, lz = 2.0, 3.0, 1.5
    p, r, q = modes
    zf = wl.z_faces(nz, lz, 0.0)
    zc = wl.z_centres(zf)
    i, j, k = np.arange(nx), np.arange(ny), np.arange(nz)
    phi = (np.sin(np.pi * q * (k + 0.5) / nz)[:, None, None] * np.cos(2 * np.pi * r * j / ny + 0.3)[None, :, None]
           * np.cos(2 * np.pi * p * i / nx + 0.1)[None, None, :])
    mu = (-4 * np.sin(np.pi * p / nx) ** 2 / (lx / nx) ** 2 - 4 * np.sin(np.pi * r / ny) ** 2 / (ly / ny) ** 2
          - 4 * np.sin(np.pi * q / (2 * nz)) ** 2 / (lz / nz) ** 2)
    for variant in (0, 1):
        got = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, phi, variant)
        assert np.abs(got - phi / (1 - a * mu)).max() <= 1e-13 * np.abs(phi).max()


@pytest.mark.parametrize("shape,beta", [((4, 4, 5), 0.0), ((8, 4, 6), 1.8), ((4, 8, 7), 2.0)])
@pytest.mark.parametrize("a", [1e-3, 0.5])
def test_dense_lu(shape, beta, a):
    nx, ny, nz = shape
    lx, ly = 1.0, 2.0
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    r = np.random.default_rng(nx * 7 + nz).standard_normal((nz, ny, nx))
    M = dense_matrix(nx, ny, nz, lx, ly, zc, zf, a)
    ref = np.linalg.solve(M, r.ravel()).reshape(r.shape)
    for variant in (0, 1):
        got = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, r, variant)
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


def test_apply_then_solve_and_operator_against_longdouble():
    nx, ny, nz, a = 16, 8, 24, 3e-3
    lx, ly = 4 * np.pi, 2 * np.pi
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    u = np.random.default_rng(5).standard_normal((nz, ny, nx))
    r_ld = apply_longdouble(u, lx, ly, zc, zf, a)
    r = oracle.apply_helmholtz3d_operator(lx, ly, zc, zf, a, u)
    assert np.abs(r - r_ld.astype(np.float64)).max() <= 1e-13 * np.abs(r).max()
    got = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, r_ld.astype(np.float64), 1)
    assert np.abs(got - u).max() <= 1e-12 * np.abs(u).max()


def test_special_cases_identity_zonly_maximum_principle_linearity():
    nx, ny, nz = 8, 16, 20
    lx, ly = 2.0, 1.0
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    rng = np.random.default_rng(9)
    r = rng.standard_normal((nz, ny, nx))
    # a = 0: identity
    assert np.abs(oracle.helmholtz3d_solve(lx, ly, zc, zf, 0.0, r, 1) - r).max() <= 1e-14 * np.abs(r).max()
    # right-hand side constant in x, y: reduces to the wall-normal Helmholtz solve (Eq. 11)
    col = rng.standard_normal(nz)
    rz = np.broadcast_to(col[:, None, None], (nz, ny, nx)).copy()
    a = 0.01
    got = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, rz, 1)
    ref = oracle.helmholtz_z_solve(zc, zf, a, rz)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    # maximum principle (M-matrix with row sums >= 1) and linearity
    u = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, r, 1)
    assert np.abs(u).max() <= np.abs(r).max() * (1 + 1e-14)
    r2 = rng.standard_normal((nz, ny, nx))
    u2 = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, r2, 1)
    u12 = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, r + 2 * r2, 1)
    assert np.abs(u12 - (u + 2 * u2)).max() <= 1e-13 * np.abs(u12).max()
    # x / y shift equivariance
    us = oracle.helmholtz3d_solve(lx, ly, zc, zf, a, np.roll(r, (3, 2), (1, 2)), 1)
    assert np.abs(us - np.roll(u, (3, 2), (1, 2))).max() <= 1e-13 * np.abs(u).max()
