"""Poisson solve with other boundary conditions -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:88-90: the eigenfunction expansion uses "Fourier / cosine / sine" transforms and "allows
for multiple combinations of boundary conditions".  This module writes that out in REAL arithmetic,
straight from the definitions, independently of oracle.c (which handles the periodic / Neumann
case with complex DFTs) and of the CUDA path:

* along a horizontal direction with n cells the second-difference operator with periodic ('P'),
  zero-gradient ('N', ghost = interior) or zero-value ('D', ghost = -interior; the boundary is the
  cell FACE) ends has the real eigenvectors
      P:  1, cos(2 pi q i/n), sin(2 pi q i/n) (0 < q < n/2), (-1)^i      lam = -4 sin^2(pi q / n)
      N:  cos(pi q (i+1/2)/n), q = 0..n-1                                lam = -4 sin^2(pi q / (2n))
      D:  sin(pi (q+1) (i+1/2)/n), q = 0..n-1                            lam = -4 sin^2(pi (q+1) / (2n))
  (reading R17); they are orthogonal, so the transform is a matrix product and its
  inverse the transposed product divided by the squared norms;
* per pair of horizontal modes one tridiagonal system along z (Eq. 12) with the wall
  rows of the chosen condition: 'N' nothing, 'D' the extra diagonal term W = 2/(dzf dzw) of reading R7;
  solved by elimination in long double;
* if every direction has a constant eigenvector (no 'D' anywhere) that one mode is singular: it is
  solved by the closed form of oracle.c (two prefix sums) and the solution carries zero volume mean.
"""
from __future__ import annotations

import numpy as np

from . import cpu


def basis(n: int, bc: str):
    """(T, norm2, lam): rows of T are the eigenvectors, norm2 their squared 2-norms, lam the
    eigenvalues of the unit-spacing second difference."""
    i = np.arange(n, dtype=np.float64)
    if bc == "P":
        rows, lam = [np.ones(n)], [0.0]
        for q in range(1, (n + 1) // 2):
            rows += [np.cos(2 * np.pi * q * i / n), np.sin(2 * np.pi * q * i / n)]
            lam += [-4.0 * np.sin(np.pi * q / n) ** 2] * 2
        if n % 2 == 0:
            rows.append((-1.0) ** i)
            lam.append(-4.0)
    elif bc == "N":
        rows = [np.cos(np.pi * q * (i + 0.5) / n) for q in range(n)]
        lam = [-4.0 * np.sin(np.pi * q / (2 * n)) ** 2 for q in range(n)]
    elif bc == "D":
        rows = [np.sin(np.pi * (q + 1) * (i + 0.5) / n) for q in range(n)]
        lam = [-4.0 * np.sin(np.pi * (q + 1) / (2 * n)) ** 2 for q in range(n)]
    else:
        raise ValueError("bc must be 'P', 'N' or 'D'")
    T = np.array(rows)
    return T, np.einsum("qi,qi->q", T, T), np.array(lam)


def wall_terms(zc, zf, bcz: str):
    """(W0, W1): extra diagonal magnitude of the first / last z row; bcz = 'NN', 'DD', 'ND', 'DN'
    (bottom, top)."""
    zc, zf = np.asarray(zc, dtype=np.float64), np.asarray(zf, dtype=np.float64)
    dzf = np.diff(zf)
    w0 = 2.0 / (dzf[0] * (2.0 * (zc[0] - zf[0]))) if bcz[0] == "D" else 0.0
    w1 = 2.0 / (dzf[-1] * (2.0 * (zf[-1] - zc[-1]))) if bcz[1] == "D" else 0.0
    return w0, w1


def apply_operator(lx, ly, zc, zf, phi, bcx="P", bcy="P", bcz="NN"):
    """L_h phi with the chosen conditions, from the stencil and ghost values (long double sums)."""
    phi = np.asarray(phi, dtype=np.longdouble)
    nz, ny, nx = phi.shape
    dzf, dzc, A, C = cpu.z_tables(zc, zf)

    def second_difference(a, axis, bc):
        lo, hi = np.roll(a, 1, axis), np.roll(a, -1, axis)
        if bc != "P":
            first = [slice(None)] * 3
            last = [slice(None)] * 3
            first[axis], last[axis] = 0, -1
            sign = 1.0 if bc == "N" else -1.0
            lo[tuple(first)] = sign * a[tuple(first)]
            hi[tuple(last)] = sign * a[tuple(last)]
        return lo - 2 * a + hi

    out = second_difference(phi, 2, bcx) / np.longdouble(lx / nx) ** 2 + second_difference(phi, 1, bcy) / np.longdouble(ly / ny) ** 2
    Al, Cl = A.astype(np.longdouble)[:, None, None], C.astype(np.longdouble)[:, None, None]
    out[1:] += Al[1:] * (phi[:-1] - phi[1:])
    out[:-1] += Cl[:-1] * (phi[1:] - phi[:-1])
    w0, w1 = wall_terms(zc, zf, bcz)
    out[0] -= np.longdouble(w0) * phi[0]
    out[-1] -= np.longdouble(w1) * phi[-1]
    return out.astype(np.float64)


def poisson_solve(lx, ly, zc, zf, f, bcx="P", bcy="P", bcz="NN"):
    """f[nz][ny][nx] -> phi with L_h phi = f; zero volume mean where the problem is singular."""
    f = np.asarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    dzf, dzc, A, C = cpu.z_tables(zc, zf)
    Tx, n2x, lamx = basis(nx, bcx)
    Ty, n2y, lamy = basis(ny, bcy)
    lamx = lamx / (lx / nx) ** 2
    lamy = lamy / (ly / ny) ** 2
    # forward transforms: coefficient = <mode, f>
    c = np.einsum("pi,kji->kjp", Tx, f)
    c = np.einsum("qj,kjp->kqp", Ty, c)
    w0, w1 = wall_terms(zc, zf, bcz)
    sigma = -(lamy[:, None] + lamx[None, :]).astype(np.longdouble)       # [q][p] >= 0
    singular = (w0 == 0.0 and w1 == 0.0) and bool((sigma == 0).any())
    Al, Cl = A.astype(np.longdouble), C.astype(np.longdouble)
    d = c.astype(np.longdouble)
    # rows: -A x_{k-1} + (A + C + W + sigma) x_k - C x_{k+1} = -d_k; elimination for all modes at once
    W = np.zeros(nz, dtype=np.longdouble)
    W[0] += w0
    W[-1] += w1
    sg = np.where(sigma == 0, np.longdouble(1.0), sigma) if singular else sigma   # placeholder pivot for the singular mode
    cp = np.empty((nz, ny, nx), dtype=np.longdouble)
    dp = np.empty((nz, ny, nx), dtype=np.longdouble)
    for k in range(nz):
        diag = Al[k] + Cl[k] + W[k] + sg
        if k == 0:
            den = diag
            dp[0] = -d[0] / den
        else:
            den = diag - Al[k] * cp[k - 1]
            dp[k] = (-d[k] + Al[k] * dp[k - 1]) / den
        cp[k] = Cl[k] / den
    x = np.empty_like(dp)
    x[-1] = dp[-1]
    for k in range(nz - 2, -1, -1):
        x[k] = dp[k] + cp[k] * x[k + 1]
    x = x.astype(np.float64)
    if singular:
        q0, p0 = np.argwhere(np.asarray(sigma == 0))[0]
        x[:, q0, p0] = cpu.zero_mode_column(dzf, dzc, c[:, q0, p0])
    # inverse transforms
    x = np.einsum("qj,kqp->kjp", Ty / n2y[:, None], x)
    return np.einsum("pi,kjp->kji", Tx / n2x[:, None], x)
