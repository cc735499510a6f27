"""Step-by-step numpy transcriptions of the paper's tridiagonal algorithms -- TEST
INFRASTRUCTURE, NOT THE PRODUCT (see ``oracle/__init__.py``).

Pure-Python loops in the paper's order and notation, for small cases only:

* ``algorithm1_*``  Algorithm 1, PAPER.md:157-197 (cyclic-reduction step of the parallel
  tridiagonal algorithm, Laszlo et al.).
* ``algorithm2_*``  Algorithm 2, PAPER.md:205-248 (the paper's init / runtime split), with the
  line-numbering gaps of the extraction read as DESIGN.md reading R9.
* ``reduced_system`` / ``solve_chunked``  the boundary system of size 2p in the ordering
  (x_0^0, x_{m-1}^0, x_0^1, ...) of PAPER.md:128,153 (reading R10).
* ``pcr_solve``     textbook parallel cyclic reduction.
* ``pack_halfcomplex`` / ``unpack_halfcomplex``  Appendix A's n-reals-in / n-reals-out layout
  (the format equation itself is missing from the text, reading R8).

All of them are pinned in tests/test_oracle_helmholtz.py (and tests/test_oracle_dft.py for the
packed layout) against dense LU
(numpy.linalg.solve) -- the paper's own verification style.
"""
from __future__ import annotations

import numpy as np


# ------------------------------------------------------------------ Algorithm 1

def algorithm1_reduce(a, b, c, d):
    """Algorithm 1, Step 1 (lines 1-20) on ONE sub-domain of m >= 3 rows.

    Rows:  a_i x_{i-1} + b_i x_i + c_i x_{i+1} = d_i  (x_{-1}, x_m belong to the neighbours).
    Returns (a', c', d') with unit diagonal:  a'_i x_0 + x_i + c'_i x_{m-1} = d'_i  for
    1 <= i <= m-2, row 0 couples (x_{-1}, x_0, x_{m-1}), row m-1 couples (x_0, x_{m-1}, x_m).
    """
    a, b, c, d = (np.array(v, dtype=np.float64) for v in (a, b, c, d))
    m = d.size
    assert m >= 3, "Algorithm 1 needs m >= 3 rows per sub-domain (reading R9)"
    a[0], c[0], d[0] = a[0] / b[0], c[0] / b[0], d[0] / b[0]          # line 3
    a[1], c[1], d[1] = a[1] / b[1], c[1] / b[1], d[1] / b[1]          # line 4
    for i in range(2, m):                                              # lines 5-10
        r = 1.0 / (b[i] - a[i] * c[i - 1])
        d[i] = r * (d[i] - a[i] * d[i - 1])
        c[i] = r * c[i]
        a[i] = -r * a[i] * a[i - 1]
    for i in range(m - 3, 0, -1):                                      # lines 11-15
        d[i] = d[i] - c[i] * d[i + 1]
        a[i] = a[i] - c[i] * a[i + 1]
        c[i] = -c[i] * c[i + 1]
    r = 1.0 / (1.0 - a[1] * c[0])                                      # lines 16-19
    d[0] = r * (d[0] - c[0] * d[1])
    a[0] = r * a[0]
    c[0] = -r * c[0] * c[1]
    return a, c, d                                                     # line 20: b = 1


def algorithm1_reconstruct(a, c, d, x0, xm1):
    """Algorithm 1, Step 3 (lines 24-30)."""
    d = np.array(d, dtype=np.float64)
    m = d.size
    d[0] = x0
    d[m - 1] = xm1
    for i in range(1, m - 1):
        d[i] = d[i] - a[i] * x0 - c[i] * xm1
    return d


# ------------------------------------------------------------------ Algorithm 2

def algorithm2_init(A, B, C):
    """Algorithm 2, Step 1 (lines 1-17): coefficient tables (a, b, c) of one sub-domain."""
    A, B, C = (np.array(v, dtype=np.float64) for v in (A, B, C))
    m = B.size
    assert m >= 3, "Algorithm 2 needs m >= 3 rows per sub-domain (reading R9)"
    a, b, c = np.zeros(m), np.zeros(m), np.zeros(m)
    a[1] = A[1]                                                        # line 3
    b[1] = B[1]                                                        # line 4
    for i in range(2, m):                                              # lines 5-8
        b[i] = B[i] - A[i] * C[i - 1] / b[i - 1]
        a[i] = -A[i] * a[i - 1] / b[i - 1]
    c[m - 1] = C[m - 1]                                                # line 9
    c[m - 2] = C[m - 2]                                                # line 10
    for i in range(m - 3, 0, -1):                                      # lines 11-14
        a[i] = a[i] - C[i] * a[i + 1] / b[i + 1]
        c[i] = -C[i] * c[i + 1] / b[i + 1]
    a[0] = A[0]                                                        # line 15
    b[0] = B[0] - C[0] * a[1] / B[1]                                   # line 16
    c[0] = -C[0] * c[1] / B[1]                                         # line 17
    return a, b, c


def algorithm2_runtime(A, C, b, d):
    """Algorithm 2, Step 2 (lines 19-26): only d is modified."""
    d = np.array(d, dtype=np.float64)
    m = d.size
    for i in range(2, m):                                              # lines 21-23
        d[i] = d[i] - A[i] * d[i - 1] / b[i - 1]
    for i in range(m - 3, -1, -1):                                     # lines 24-26
        d[i] = d[i] - C[i] * d[i + 1] / b[i + 1]
    return d


def algorithm2_reconstruct(a, b, c, d, x0, xm1):
    """Algorithm 2, Step 4 (lines 30-36)."""
    d = np.array(d, dtype=np.float64)
    m = d.size
    d[0] = x0
    d[m - 1] = xm1
    for i in range(1, m - 1):
        d[i] = (d[i] - a[i] * x0 - c[i] * xm1) / b[i]
    return d


# --------------------------------------------------------- reduced system, driver

def _dense_tridiag_solve(lo, di, up, rhs):
    n = di.size
    M = np.zeros((n, n))
    for i in range(n):
        M[i, i] = di[i]
        if i > 0:
            M[i, i - 1] = lo[i]
        if i + 1 < n:
            M[i, i + 1] = up[i]
    return np.linalg.solve(M, rhs)


def reduced_system(rows):
    """Boundary system of size 2p (reading R10).

    rows: list over sub-domains s of ((a_0,b_0,c_0,d_0), (a_{m-1},b_{m-1},c_{m-1},d_{m-1})).
    Unknown order (x_0^0, x_{m-1}^0, x_0^1, x_{m-1}^1, ...).  Returns (lo, di, up, rhs).
    """
    p = len(rows)
    lo, di, up, rhs = (np.zeros(2 * p) for _ in range(4))
    for s, (r0, r1) in enumerate(rows):
        lo[2 * s], di[2 * s], up[2 * s], rhs[2 * s] = r0
        lo[2 * s + 1], di[2 * s + 1], up[2 * s + 1], rhs[2 * s + 1] = r1
    return lo, di, up, rhs


def _split(n, p):
    """p contiguous sub-domains covering 0..n-1, sizes differing by at most one."""
    base, extra = divmod(n, p)
    bounds, start = [], 0
    for s in range(p):
        size = base + (1 if s < extra else 0)
        bounds.append((start, start + size))
        start += size
    return bounds


def solve_chunked(lo, di, up, d, p, algorithm=2, bounds=None):
    """Solve lo_k x_{k-1} + di_k x_k + up_k x_{k+1} = d_k with p sub-domains, following
    PAPER.md:124-131 steps 4-6 with Algorithm 1 or Algorithm 2 inside each sub-domain.

    bounds: optional list of (start, end) row ranges of the sub-domains (the z-slabs owned by the
    ranks of a distributed solve), contiguous, each of at least 3 rows (reading
    R9); default: p sub-domains of sizes differing by at most one."""
    lo, di, up, d = (np.array(v, dtype=np.float64) for v in (lo, di, up, d))
    n = d.size
    lo[0] = 0.0
    up[n - 1] = 0.0
    chunks = _split(n, p) if bounds is None else [tuple(b) for b in bounds]
    assert chunks[0][0] == 0 and chunks[-1][1] == n and all(chunks[s][1] == chunks[s + 1][0] for s in range(len(chunks) - 1))
    red, state = [], []
    for (s0, s1) in chunks:
        if algorithm == 1:
            a, c, dd = algorithm1_reduce(lo[s0:s1], di[s0:s1], up[s0:s1], d[s0:s1])
            red.append(((a[0], 1.0, c[0], dd[0]), (a[-1], 1.0, c[-1], dd[-1])))
            state.append((a, None, c, dd))
        else:
            a, b, c = algorithm2_init(lo[s0:s1], di[s0:s1], up[s0:s1])
            dd = algorithm2_runtime(lo[s0:s1], up[s0:s1], b, d[s0:s1])
            red.append(((a[0], b[0], c[0], dd[0]), (a[-1], b[-1], c[-1], dd[-1])))
            state.append((a, b, c, dd))
    xb = _dense_tridiag_solve(*reduced_system(red))
    x = np.empty(n)
    for s, (s0, s1) in enumerate(chunks):
        a, b, c, dd = state[s]
        if algorithm == 1:
            x[s0:s1] = algorithm1_reconstruct(a, c, dd, xb[2 * s], xb[2 * s + 1])
        else:
            x[s0:s1] = algorithm2_reconstruct(a, b, c, dd, xb[2 * s], xb[2 * s + 1])
    return x


# ------------------------------------------------------------------ textbook PCR

def pcr_solve(lo, di, up, d):
    """Textbook parallel cyclic reduction: ceil(log2 n) levels; at distance h every row i
    eliminates x_{i-h} and x_{i+h} using rows i-h and i+h; finally x_i = d_i / b_i."""
    a, b, c, d = (np.array(v, dtype=np.float64) for v in (lo, di, up, d))
    n = d.size
    a[0] = 0.0
    c[n - 1] = 0.0
    h = 1
    while h < n:
        na, nb, nc, nd = a.copy(), b.copy(), c.copy(), d.copy()
        for i in range(n):
            k1 = a[i] / b[i - h] if i - h >= 0 else 0.0
            k2 = c[i] / b[i + h] if i + h < n else 0.0
            nb[i] = b[i] - (k1 * c[i - h] if i - h >= 0 else 0.0) - (k2 * a[i + h] if i + h < n else 0.0)
            nd[i] = d[i] - (k1 * d[i - h] if i - h >= 0 else 0.0) - (k2 * d[i + h] if i + h < n else 0.0)
            na[i] = -k1 * a[i - h] if i - h >= 0 else 0.0
            nc[i] = -k2 * c[i + h] if i + h < n else 0.0
        a, b, c, d = na, nb, nc, nd
        h *= 2
    return d / b


# ------------------------------------------------- Appendix A packed half-complex

def pack_halfcomplex(X):
    """X[0..n/2] complex (R2C output of n reals, n even) -> n reals
    [X_0^r, X_{n/2}^r, X_1^r, X_1^i, ..., X_{n/2-1}^r, X_{n/2-1}^i]   (reading R8)."""
    X = np.asarray(X, dtype=np.complex128)
    h = X.size - 1
    n = 2 * h
    out = np.empty(n)
    out[0] = X[0].real
    out[1] = X[h].real
    out[2::2] = X[1:h].real
    out[3::2] = X[1:h].imag
    return out


def unpack_halfcomplex(r):
    r = np.asarray(r, dtype=np.float64)
    n = r.size
    h = n // 2
    X = np.zeros(h + 1, dtype=np.complex128)
    X[0] = r[0]
    X[h] = r[1]
    X[1:h] = r[2::2] + 1j * r[3::2]
    return X
