"""Pins for the oracle's wall-normal Helmholtz solve (definition O-H) and for the
transcriptions of the paper's Algorithm 1 / Algorithm 2 / PCR (P3, P4, P6, P7)."""
import numpy as np
import pytest

import oracle
from oracle import algorithms as alg
from paper_2502_06296_b200 import workloads as wl


def dense_helmholtz_matrix(zc, zf, a):
    """I - a L_z with Dirichlet walls (ghost = -interior), assembled from the definition."""
    nz = zc.size
    dzf = np.diff(zf)
    M = np.eye(nz)
    for k in range(nz):
        # flux through the lower face
        if k > 0:
            w = 1 / (dzf[k] * (zc[k] - zc[k - 1]))
            M[k, k] += a * w
            M[k, k - 1] -= a * w
        else:
            M[k, k] += a * 2 / (dzf[0] * 2 * (zc[0] - zf[0]))       # (u_0 - (-u_0)) / dzw_0
        if k < nz - 1:
            w = 1 / (dzf[k] * (zc[k + 1] - zc[k]))
            M[k, k] += a * w
            M[k, k + 1] -= a * w
        else:
            M[k, k] += a * 2 / (dzf[-1] * 2 * (zf[-1] - zc[-1]))
    return M


@pytest.mark.parametrize("q", [1, 2, 7, 16])
@pytest.mark.parametrize("a", [0.0, 5e-5, 0.3])
def test_uniform_dirichlet_eigenfunctions(q, a):
    """sin(pi q (k+1/2)/nz), q = 1..nz, is an eigenvector: u = r / (1 + a 4 sin^2(pi q/(2nz))/dz^2)."""
    nx, ny, nz, lz = 4, 2, 16, 2.0
    zf = wl.z_faces(nz, lz)
    zc = wl.z_centres(zf)
    k = np.arange(nz)
    prof = np.sin(np.pi * q * (k + 0.5) / nz)
    r = prof[:, None, None] * (1 + np.arange(ny))[None, :, None] * (1 + np.arange(nx))[None, None, :]
    dz = lz / nz
    u = oracle.helmholtz_z_solve(zc, zf, a, r)
    expect = r / (1 + a * 4 * np.sin(np.pi * q / (2 * nz)) ** 2 / dz ** 2)
    assert np.abs(u - expect).max() <= 1e-13 * np.abs(expect).max()


@pytest.mark.parametrize("nz,beta,a", [(4, 0.0, 0.1), (8, 1.8, 5e-5), (8, 2.0, 1.0), (64, 1.8, 5e-5),
                                       (256, 1.8, 5e-5), (256, 1.8, 1e-2)])
def test_dense_lu_per_column(nz, beta, a):
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    rng = np.random.default_rng(nz)
    r = rng.standard_normal((nz, 3, 5))
    M = dense_helmholtz_matrix(zc, zf, a)
    ref = np.linalg.solve(M, r.reshape(nz, -1)).reshape(r.shape)
    got = oracle.helmholtz_z_solve(zc, zf, a, r)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    cols = oracle.helmholtz_z_solve_columns(zc, zf, a, r.reshape(nz, -1).T.copy())
    assert np.array_equal(cols.T.reshape(r.shape), got)
    lo, di, up = oracle.helmholtz_matrix(zc, zf, a)
    assert np.abs(np.diag(M) - di).max() <= 1e-13 * np.abs(di).max()
    assert np.abs(np.diag(M, -1) - lo[1:]).max() <= 1e-13 * np.abs(di).max()
    assert np.abs(np.diag(M, 1) - up[:-1]).max() <= 1e-13 * np.abs(di).max()


def test_maximum_principle_and_small_a_limit():
    w = wl.scaled(wl.CONFIGS["c1"], 8, 8, 128)
    zc, zf = wl.grid(w)
    r = wl.helmholtz_rhs(w)
    for a in (5e-5, 1e-2, 10.0):
        u = oracle.helmholtz_z_solve(zc, zf, a, r)
        assert np.abs(u).max() <= np.abs(r).max() * (1 + 1e-14)
    assert np.array_equal(oracle.helmholtz_z_solve(zc, zf, 0.0, r), r)
    u = oracle.helmholtz_z_solve(zc, zf, 1e-12, r)
    assert np.abs(u - r).max() <= 1e-5 * np.abs(r).max()


def test_uniform_matrix_reduces_to_textbook():
    """Uniform grid: (1/dz^2)(1,-2,1) inside, -3 on the Dirichlet wall rows."""
    nz, lz, a = 12, 2.0, 0.7
    zf = wl.z_faces(nz, lz)
    lo, di, up = oracle.helmholtz_matrix(wl.z_centres(zf), zf, a)
    h = a / (lz / nz) ** 2
    assert np.allclose(di[1:-1], 1 + 2 * h, rtol=1e-13)
    assert np.allclose([di[0], di[-1]], 1 + 3 * h, rtol=1e-13)
    assert np.allclose(lo[1:], -h, rtol=1e-13) and np.allclose(up[:-1], -h, rtol=1e-13)
    assert lo[0] == 0.0 and up[-1] == 0.0


# ------------------------------------------------------- Algorithm 1 / 2 / PCR (P7)

def _random_system(n, rng, dominance=1.05):
    lo, up = -rng.uniform(0.1, 1.0, n), -rng.uniform(0.1, 1.0, n)
    di = dominance * (np.abs(lo) + np.abs(up)) + rng.uniform(0, 0.1, n)
    lo[0] = 0.0
    up[-1] = 0.0
    d = rng.standard_normal(n)
    M = np.diag(di) + np.diag(lo[1:], -1) + np.diag(up[:-1], 1)
    return lo, di, up, d, np.linalg.solve(M, d)


@pytest.mark.parametrize("n,p", [(3, 1), (9, 3), (12, 4), (16, 2), (37, 5), (64, 8), (96, 32), (130, 7)])
@pytest.mark.parametrize("algorithm", [1, 2])
def test_chunked_algorithms_match_dense_lu(n, p, algorithm):
    """the parallel tridiagonal output equals the serial one to machine precision."""
    rng = np.random.default_rng(1000 * n + p)
    lo, di, up, d, ref = _random_system(n, rng)
    got = alg.solve_chunked(lo, di, up, d, p, algorithm)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(oracle.thomas(lo, di, up, d) - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("bounds", [[(0, 3), (3, 6)], [(0, 3), (3, 40), (40, 43), (43, 64)], [(0, 34), (34, 67), (67, 100)],
                                    [(0, 5), (5, 8), (8, 11), (11, 14), (14, 17), (17, 20), (20, 23), (23, 26)]])
@pytest.mark.parametrize("algorithm", [1, 2])
def test_uneven_slabs_match_dense_lu(bounds, algorithm):
    """The z-slabs of a distributed solve need not be equal: any contiguous
    partition with at least 3 rows per slab (reading R9) reproduces the serial solve, also on the
    Poisson systems of a low mode of a stretched grid (diagonal -(A+C) - sigma)."""
    n = bounds[-1][1]
    rng = np.random.default_rng(7 * n + len(bounds))
    lo, di, up, d, ref = _random_system(n, rng)
    got = alg.solve_chunked(lo, di, up, d, len(bounds), algorithm, bounds=bounds)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    zf = wl.z_faces(n, 2.0, 1.8)
    zc = wl.z_centres(zf)
    A, C = oracle.z_tables(zc, zf)[2:]
    sigma = 0.37
    lo2, up2, di2 = A.copy(), C.copy(), -(A + C) - sigma
    ref2 = oracle.thomas(lo2, di2, up2, d)
    got2 = alg.solve_chunked(lo2, di2, up2, d, len(bounds), algorithm, bounds=bounds)
    assert np.abs(got2 - ref2).max() <= 1e-10 * np.abs(ref2).max()


@pytest.mark.parametrize("algorithm", [1, 2])
def test_two_row_subdomains_are_not_supported(algorithm):
    """Reading R9: the algorithms as printed need m >= 3 rows per sub-domain."""
    rng = np.random.default_rng(0)
    lo, di, up, d, _ = _random_system(8, rng)
    with pytest.raises(AssertionError):
        alg.solve_chunked(lo, di, up, d, 4, algorithm)


@pytest.mark.parametrize("n", [1, 2, 5, 16, 33, 64])
def test_pcr_matches_dense_lu(n):
    rng = np.random.default_rng(n)
    lo, di, up, d, ref = _random_system(n, rng)
    assert np.abs(alg.pcr_solve(lo, di, up, d) - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("nz,p,a", [(64, 4, 5e-5), (256, 16, 5e-5), (256, 32, 2.5e-5), (96, 8, 1e-2)])
def test_algorithm2_on_the_helmholtz_matrix(nz, p, a):
    """The paper's use case: Alg. 2 tables depend on k only; the runtime
    touches d only; result equals the serial Thomas solve of O-H."""
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    lo, di, up = oracle.helmholtz_matrix(zc, zf, a)
    rng = np.random.default_rng(nz + p)
    d = rng.standard_normal(nz)
    ref = oracle.thomas(lo, di, up, d)
    got = alg.solve_chunked(lo, di, up, d, p, 2)
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max() * 10
