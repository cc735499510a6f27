"""Pins for the oracle's divergence / gradient / projection (oracle/projection.py; Eqs. 4-6,
PAPER.md:53-57; reading R15)."""
import numpy as np
import pytest

import oracle
from oracle import projection as proj
from paper_2502_06296_b200 import workloads as wl


def grid(nz, beta):
    zf = wl.z_faces(nz, 2.0, beta)
    return wl.z_centres(zf), zf


def random_velocity(rng, nz, ny, nx):
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    w[-1] = 0.0                                    # no penetration through the top wall
    return u, v, w


@pytest.mark.parametrize("beta", [0.0, 1.8])
def test_divergence_of_gradient_is_the_poisson_operator(beta):
    """D G = L_h exactly: the identity the pressure correction rests on."""
    nx, ny, nz, lx, ly = 16, 8, 12, 3.0, 2.0
    zc, zf = grid(nz, beta)
    phi = np.random.default_rng(1).standard_normal((nz, ny, nx))
    gx, gy, gz = proj.gradient(lx, ly, zc, phi)
    dg = proj.divergence(lx, ly, zf, gx, gy, gz)
    lap = oracle.apply_poisson_operator(lx, ly, zc, zf, phi)
    assert np.abs(dg - lap).max() <= 1e-13 * np.abs(lap).max()


def test_closed_forms():
    nx, ny, nz, lx, ly = 8, 8, 6, 2.0, 4.0
    zc, zf = grid(nz, 1.8)
    one = np.ones((nz, ny, nx))
    # a uniform horizontal flow is divergence free; the gradient of a constant is zero
    assert np.abs(proj.divergence(lx, ly, zf, 3 * one, -2 * one, 0 * one)).max() == 0.0
    assert all(np.abs(g).max() == 0.0 for g in proj.gradient(lx, ly, zc, 5 * one))
    # u = x_face: du/dx = 1 everywhere except across the periodic seam
    xf = (np.arange(nx) + 1.0) * (lx / nx)
    d = proj.divergence(lx, ly, zf, np.broadcast_to(xf, (nz, ny, nx)).copy(), 0 * one, 0 * one)
    assert np.abs(d[:, :, 1:] - 1.0).max() <= 1e-14 and np.abs(d[:, :, 0] - (1.0 - nx)).max() <= 1e-13
    # w = z_face (top faces): dw/dz = 1 in every cell, including the one on the bottom wall (w = 0 there)
    wz = np.broadcast_to(zf[1:, None, None], (nz, ny, nx)).copy()
    assert np.abs(proj.divergence(lx, ly, zf, 0 * one, 0 * one, wz) - 1.0).max() <= 1e-13
    # Phi = zc: dPhi/dz = 1 on interior faces, 0 on the top wall face
    gz = proj.gradient(lx, ly, zc, np.broadcast_to(zc[:, None, None], (nz, ny, nx)).copy())[2]
    assert np.abs(gz[:-1] - 1.0).max() <= 1e-13 and np.abs(gz[-1]).max() == 0.0
    # discrete stream function psi at the cell corners (i+1/2, j+1/2): u = d_y psi on the x-faces,
    # v = -d_x psi on the y-faces is divergence free to rounding
    psi = np.random.default_rng(2).standard_normal((nz, ny, nx))
    u = (psi - np.roll(psi, 1, axis=1)) / (ly / ny)
    v = -(psi - np.roll(psi, 1, axis=2)) / (lx / nx)
    d = proj.divergence(lx, ly, zf, u, v, 0 * one)
    assert np.abs(d).max() <= 1e-12 * np.abs(u).max() / min(lx / nx, ly / ny)

@pytest.mark.parametrize("shape,beta", [((16, 8, 12), 0.0), ((8, 16, 20), 1.8), ((32, 8, 9), 2.0)])
def test_projection_step_makes_the_field_divergence_free(shape, beta):
    """Eq. (4) + Eqs. (5)-(6) with the oracle's Poisson solve: D u^{k+1} = 0 to rounding."""
    nx, ny, nz = shape
    lx, ly, gdt = 4 * np.pi, 2 * np.pi, 0.37e-2
    zc, zf = grid(nz, beta)
    rng = np.random.default_rng(nx + nz)
    u, v, w = random_velocity(rng, nz, ny, nx)
    p = rng.standard_normal((nz, ny, nx))
    rhs = proj.divergence_rhs(lx, ly, zf, u, v, w, 1.0 / gdt)
    dzf = np.diff(zf)
    assert abs(np.einsum("k,kji->", dzf, rhs)) <= 1e-10 * np.abs(rhs).max() * nx * ny   # compatible
    phi = oracle.poisson_solve(lx, ly, zc, zf, rhs, 0)
    un, vn, wn, pn = proj.project(lx, ly, zc, u, v, w, p, phi, gdt)
    div0 = np.abs(proj.divergence(lx, ly, zf, u, v, w)).max()
    assert np.abs(proj.divergence(lx, ly, zf, un, vn, wn)).max() <= 1e-11 * div0
    assert np.abs(wn[-1]).max() == 0.0                       # the wall face is not touched
    assert np.array_equal(pn, p + phi)


@pytest.mark.parametrize("beta", [0.0, 1.8])
def test_helmholtz_z_rhs_against_the_helmholtz_matrix_and_eigenfunctions(beta):
    """u** - a L_z u^k = u** - u^k + (I - a L_z) u^k, with (I - a L_z) the tridiagonal matrix of the
    oracle's Helmholtz solve (oracle.c); on a uniform grid sin(pi q (k+1/2)/nz) is an eigenfunction of
    L_z with eigenvalue mu, so the right-hand side of u** = u^k = f is (1 - a mu) f and Eq. (11) returns
    f itself (the implicit and the explicit half of the wall-normal diffusion cancel)."""
    nx, ny, nz, a = 4, 6, 24, 3e-3
    zc, zf = grid(nz, beta)
    rng = np.random.default_rng(3)
    u2, uk = rng.standard_normal((nz, ny, nx)), rng.standard_normal((nz, ny, nx))
    lo, di, up = oracle.helmholtz_matrix(zc, zf, a)
    muk = di[:, None, None] * uk
    muk[1:] += lo[1:, None, None] * uk[:-1]
    muk[:-1] += up[:-1, None, None] * uk[1:]
    ref = u2 - uk + muk
    got = proj.helmholtz_z_rhs(zc, zf, a, u2, uk)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    if beta == 0.0:
        q = 5
        mode = np.sin(np.pi * q * (np.arange(nz) + 0.5) / nz)
        f = np.broadcast_to(mode[:, None, None], (nz, ny, nx)).copy()
        mu = -4 * np.sin(np.pi * q / (2 * nz)) ** 2 / (2.0 / nz) ** 2
        r = proj.helmholtz_z_rhs(zc, zf, a, f, f)
        assert np.abs(r - (1 - a * mu) * f).max() <= 1e-13
        unew = oracle.helmholtz_z_solve(zc, zf, a, r)
        assert np.abs(unew - f).max() <= 1e-13
