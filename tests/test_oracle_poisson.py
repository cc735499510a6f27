"""Pins for the oracle's Poisson solve (definition O-P).

P2  closed-form discrete eigenfunctions (uniform z, Neumann walls)
P4  bordered dense LU on grids <= 8^3, stretched z, built here from the stencil definition
P5  apply-then-solve round trip on stretched grids
P6  invariants: residual, weighted mean, linearity, shift equivariance, z-flip symmetry
plus the (0,0) closed form, the pivot recurrence against long-double elimination, and the
definition-level DFT variant against the FFT variant.
"""
import numpy as np
import pytest

import oracle
from paper_2502_06296_b200 import workloads as wl

LD = np.longdouble


def stretched(nz, beta=1.8, lz=2.0):
    zf = wl.z_faces(nz, lz, beta)
    return wl.z_centres(zf), zf


def dense_poisson_matrix(nx, ny, nz, lx, ly, zc, zf, dtype=np.float64):
    """The stencil of O-P assembled entry by entry (independent of oracle.c)."""
    zc, zf = np.asarray(zc, dtype), np.asarray(zf, dtype)
    dzf = zf[1:] - zf[:-1]
    dzc = zc[1:] - zc[:-1]
    dx, dy = dtype(lx) / nx, dtype(ly) / ny
    N = nx * ny * nz
    M = np.zeros((N, N), dtype)

    def idx(i, j, k):
        return (k * ny + j % ny) * nx + i % nx

    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                r = idx(i, j, k)
                for (di, dj, w) in ((1, 0, 1 / dx ** 2), (-1, 0, 1 / dx ** 2),
                                    (0, 1, 1 / dy ** 2), (0, -1, 1 / dy ** 2)):
                    M[r, idx(i + di, j + dj, k)] += w
                    M[r, r] -= w
                if k > 0:
                    w = 1 / (dzf[k] * dzc[k - 1])
                    M[r, idx(i, j, k - 1)] += w
                    M[r, r] -= w
                if k < nz - 1:
                    w = 1 / (dzf[k] * dzc[k])
                    M[r, idx(i, j, k + 1)] += w
                    M[r, r] -= w
    return M, dzf


def apply_stencil_longdouble(phi, lx, ly, zc, zf):
    """L_h phi in long double, difference form (independent of oracle.c)."""
    p = phi.astype(LD)
    nz, ny, nx = p.shape
    zc, zf = np.asarray(zc, LD), np.asarray(zf, LD)
    dzf = zf[1:] - zf[:-1]
    dzc = zc[1:] - zc[:-1]
    dx, dy = LD(lx) / nx, LD(ly) / ny
    out = (np.roll(p, -1, 2) - 2 * p + np.roll(p, 1, 2)) / dx ** 2
    out += (np.roll(p, -1, 1) - 2 * p + np.roll(p, 1, 1)) / dy ** 2
    A = 1 / (dzf[1:] * dzc)           # k = 1..nz-1
    C = 1 / (dzf[:-1] * dzc)          # k = 0..nz-2
    out[1:] += A[:, None, None] * (p[:-1] - p[1:])
    out[:-1] += C[:, None, None] * (p[1:] - p[:-1])
    return out


# ----------------------------------------------------------------------------- P2

@pytest.mark.parametrize("modes", [(1, 0, 0), (0, 2, 0), (0, 0, 1), (3, 5, 7), (8, 8, 15), (2, 1, 4)])
def test_uniform_neumann_eigenfunctions(modes):
    """cos(2 pi p i/nx) cos(2 pi r j/ny) cos(pi q (k+1/2)/nz) is an eigenvector of L_h with
    mu = -4 sin^2(pi p/nx)/dx^2 - 4 sin^2(pi r/ny)/dy^2 - 4 sin^2(pi q/(2 nz))/dz^2."""
    nx, ny, nz = 16, 16, 16
    lx, ly, lz = 2 * np.pi, 3.0, 2.0
    p, r, q = modes
    zf = wl.z_faces(nz, lz, 0.0)
    zc = wl.z_centres(zf)
    i, j, k = np.arange(nx), np.arange(ny), np.arange(nz)
    phi = (np.cos(2 * np.pi * q * 0 + np.pi * q * (k + 0.5) / nz)[:, None, None]
           * np.cos(2 * np.pi * r * j / ny)[None, :, None]
           * np.cos(2 * np.pi * p * i / nx)[None, None, :])
    dx, dy, dz = lx / nx, ly / ny, lz / nz
    mu = (-4 * np.sin(np.pi * p / nx) ** 2 / dx ** 2 - 4 * np.sin(np.pi * r / ny) ** 2 / dy ** 2
          - 4 * np.sin(np.pi * q / (2 * nz)) ** 2 / dz ** 2)
    for variant in (0, 1):
        got = oracle.poisson_solve(lx, ly, zc, zf, mu * phi, variant)
        assert np.abs(got - phi).max() <= 1e-13 * np.abs(phi).max()
    # and the operator routine maps phi to mu*phi
    lap = oracle.apply_poisson_operator(lx, ly, zc, zf, phi)
    assert np.abs(lap - mu * phi).max() <= 1e-12 * abs(mu)


# ----------------------------------------------------------------------------- P4

@pytest.mark.parametrize("shape,beta", [((4, 4, 4), 0.0), ((8, 4, 6), 1.8), ((4, 8, 8), 2.0), ((8, 8, 8), 1.8)])
def test_bordered_dense_lu(shape, beta):
    nx, ny, nz = shape
    lx, ly = 4 * np.pi, 2 * np.pi
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    M, dzf = dense_poisson_matrix(nx, ny, nz, lx, ly, zc, zf)
    rng = np.random.default_rng(nx * 100 + nz)
    f = wl.remove_weighted_mean(rng.standard_normal((nz, ny, nx)), zf)
    N = nx * ny * nz
    w = np.repeat(dzf, nx * ny)                   # gauge row: sum dzf_k phi = 0
    B = np.zeros((N + 1, N + 1))
    B[:N, :N] = M
    B[:N, N] = 1.0                                # Lagrange multiplier absorbs incompatibility
    B[N, :N] = w
    sol = np.linalg.solve(B, np.concatenate([f.ravel(), [0.0]]))
    ref = sol[:N].reshape(nz, ny, nx)
    assert abs(sol[N]) <= 1e-12 * np.abs(f).max()  # compatible rhs -> multiplier ~ 0
    for variant in (0, 1):
        got = oracle.poisson_solve(lx, ly, zc, zf, f, variant)
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


def test_left_null_vector_is_dzf():
    """sum_k dzf_k (L_h phi)_k = 0 for any phi: why the rhs mean must be dzf-weighted (R3)."""
    nx, ny, nz = 4, 4, 12
    zc, zf = stretched(nz)
    rng = np.random.default_rng(3)
    phi = rng.standard_normal((nz, ny, nx))
    lap = oracle.apply_poisson_operator(2.0, 2.0, zc, zf, phi)
    dzf = np.diff(zf)
    assert abs(np.einsum("k,kji->", dzf, lap)) <= 1e-10 * np.abs(lap).max()
    assert abs(lap.sum()) > 1e-6 * np.abs(lap).max()   # the arithmetic mean does NOT vanish


# ----------------------------------------------------------------------------- P5 / P6

@pytest.mark.parametrize("shape,beta,lx,ly", [((16, 8, 12), 1.8, 4 * np.pi, 2 * np.pi),
                                              ((32, 16, 48), 2.0, 8 * np.pi, 3 * np.pi)])
def test_apply_then_solve_roundtrip_stretched(shape, beta, lx, ly):
    nx, ny, nz = shape
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    x = (np.arange(nx) + 0.5) * lx / nx
    y = (np.arange(ny) + 0.5) * ly / ny
    phi = (np.cos(np.pi * zc)[:, None, None] * (1 + 0.5 * np.sin(2 * np.pi * y / ly))[None, :, None]
           * (1 + 0.3 * np.cos(4 * np.pi * x / lx))[None, None, :]
           + (zc ** 2 * (3 - zc))[:, None, None] * np.sin(2 * np.pi * x / lx)[None, None, :])
    dzf = np.diff(zf)
    phi = phi - np.einsum("k,kji->", dzf, phi) / (dzf.sum() * nx * ny)
    f = apply_stencil_longdouble(phi, lx, ly, zc, zf).astype(np.float64)
    got = oracle.poisson_solve(lx, ly, zc, zf, f, 1)
    assert np.abs(got - phi).max() <= 1e-12 * np.abs(phi).max()


@pytest.mark.parametrize("cfg", ["uniform", "stretched"])
def test_residual_and_weighted_mean_invariants(cfg):
    if cfg == "uniform":
        w = wl.scaled(wl.CONFIGS["c0"], 32, 32, 32)
    else:
        w = wl.scaled(wl.CONFIGS["c1"], 32, 16, 64)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    phi = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    res = (f.astype(LD) - apply_stencil_longdouble(phi, w.lx, w.ly, zc, zf)).astype(np.float64)
    if cfg == "uniform":
        assert np.abs(res).max() <= 1e-12 * np.abs(f).max()
    # normwise backward error (reading R11): ||r|| / (||L_h|| ||phi|| + ||f||)
    dzf, dzc = np.diff(zf), np.diff(zc)
    normL = 4 / (w.lx / w.nx) ** 2 + 4 / (w.ly / w.ny) ** 2 + 4 / (dzf.min() * dzc.min())
    assert np.abs(res).max() <= 1e-14 * (normL * np.abs(phi).max() + np.abs(f).max())
    # zero volume mean of the solution
    wm = np.einsum("k,kji->", dzf, phi) / (dzf.sum() * w.nx * w.ny)
    assert abs(wm) <= 1e-15 * np.abs(phi).max() * 10


def test_linearity_shift_equivariance_and_zflip():
    w = wl.scaled(wl.CONFIGS["c1"], 16, 16, 24)
    zc, zf = wl.grid(w)
    rng = np.random.default_rng(11)
    f1 = wl.remove_weighted_mean(rng.standard_normal((w.nz, w.ny, w.nx)), zf)
    f2 = wl.remove_weighted_mean(rng.standard_normal((w.nz, w.ny, w.nx)), zf)
    s = lambda f: oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)  # noqa: E731
    p1, p2 = s(f1), s(f2)
    scale = np.abs(p1).max() + np.abs(p2).max()
    assert np.abs(s(2.5 * f1 - 0.75 * f2) - (2.5 * p1 - 0.75 * p2)).max() <= 1e-12 * scale
    assert np.abs(s(np.roll(f1, (3, 5), (1, 2))) - np.roll(p1, (3, 5), (1, 2))).max() <= 1e-12 * scale
    # the tanh grid is symmetric about the centre plane: flipping z commutes with the solve
    assert np.abs(np.diff(zf) - np.diff(zf)[::-1]).max() <= 1e-15
    assert np.abs(s(f1[::-1].copy()) - p1[::-1]).max() <= 1e-11 * scale


def test_definition_dft_variant_equals_fft_variant_c0_shape():
    w = wl.scaled(wl.CONFIGS["c0"], 32, 32, 16)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    a = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 0)
    b = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()


# ------------------------------------------------------------------- column solvers

@pytest.mark.parametrize("nz,beta,sigma", [(16, 0.0, 1.0), (64, 1.8, 0.25), (256, 1.8, 0.25),
                                           (512, 2.0, 0.0625), (512, 2.0, 3.0e4)])
def test_pivot_recurrence_matches_longdouble_elimination(nz, beta, sigma):
    """orc_thomas_poisson uses the exact diagonal -(A+C)-sigma of the double tables (R5):
    compare with Gaussian elimination of that very system carried out in long double."""
    zc, zf = stretched(nz, beta) if beta else (wl.z_centres(wl.z_faces(nz)), wl.z_faces(nz))
    dzf, dzc, A, C = oracle.z_tables(zc, zf)
    rng = np.random.default_rng(nz)
    d = rng.standard_normal(nz)
    got = oracle.thomas_poisson(A, C, sigma, d)
    Al, Cl, dl = A.astype(LD), C.astype(LD), d.astype(LD)
    diag = -(Al + Cl) - LD(sigma)
    cp, dp = np.zeros(nz, LD), np.zeros(nz, LD)
    cp[0], dp[0] = Cl[0] / diag[0], dl[0] / diag[0]
    for k in range(1, nz):
        m = diag[k] - Al[k] * cp[k - 1]
        cp[k], dp[k] = Cl[k] / m, (dl[k] - Al[k] * dp[k - 1]) / m
    x = np.zeros(nz, LD)
    x[-1] = dp[-1]
    for k in range(nz - 2, -1, -1):
        x[k] = dp[k] - cp[k] * x[k + 1]
    assert np.abs(got - x.astype(np.float64)).max() <= 1e-13 * np.abs(x).max()


@pytest.mark.parametrize("nz,beta", [(8, 0.0), (12, 1.8), (128, 2.0)])
def test_zero_mode_closed_form(nz, beta):
    """(0,0) column: pseudo-inverse solution with zero dzf-weighted mean, vs dense bordered LU."""
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    dzf, dzc, A, C = oracle.z_tables(zc, zf)
    rng = np.random.default_rng(nz)
    d = rng.standard_normal(nz)
    d -= np.dot(dzf, d) / dzf.sum()
    T = np.diag(-(A + C)) + np.diag(A[1:], -1) + np.diag(C[:-1], 1)
    B = np.zeros((nz + 1, nz + 1))
    B[:nz, :nz], B[:nz, nz], B[nz, :nz] = T, 1.0, dzf
    ref = np.linalg.solve(B, np.concatenate([d, [0.0]]))[:nz]
    got = oracle.zero_mode_column(dzf, dzc, d)
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
    assert abs(np.dot(dzf, got)) <= 1e-14 * np.abs(got).max() * dzf.sum()
    assert np.abs(T @ got - d).max() <= 1e-12 * np.abs(T).max() * np.abs(got).max()


def test_z_tables_uniform_reduce_to_textbook():
    nz, lz = 10, 2.0
    zf = wl.z_faces(nz, lz)
    dzf, dzc, A, C = oracle.z_tables(wl.z_centres(zf), zf)
    dz = lz / nz
    assert np.allclose(dzf, dz, rtol=0, atol=1e-15) and np.allclose(dzc, dz, rtol=0, atol=1e-15)
    assert A[0] == 0.0 and C[-1] == 0.0
    assert np.allclose(A[1:], 1 / dz ** 2, rtol=1e-13) and np.allclose(C[:-1], 1 / dz ** 2, rtol=1e-13)


@pytest.mark.parametrize("shape,beta", [((8, 4, 6), 1.8), ((4, 8, 7), 2.0), ((6, 4, 5), 0.0)])
def test_apply_operator_matches_independent_stencil_on_stretched_grid(shape, beta):
    """oracle.apply_poisson_operator (the checker of the full-size c3 GPU test) against the two
    independent statements of O-P in this file: the dense matrix assembled entry by entry and
    the long-double difference-form stencil (Eq. 12)."""
    nx, ny, nz = shape
    lx, ly = 8 * np.pi, 3 * np.pi
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    M, _ = dense_poisson_matrix(nx, ny, nz, lx, ly, zc, zf)
    phi = np.random.default_rng(91 + nz).standard_normal((nz, ny, nx))
    got = oracle.apply_poisson_operator(lx, ly, zc, zf, phi)
    scale = np.abs(M).sum(axis=1).max() * np.abs(phi).max()
    assert np.abs(got.reshape(-1) - M @ phi.reshape(-1)).max() <= 1e-14 * scale
    ref_ld = apply_stencil_longdouble(phi, lx, ly, zc, zf)
    assert np.abs(got - ref_ld.astype(np.float64)).max() <= 1e-14 * scale
