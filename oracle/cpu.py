"""ctypes loader for ``oracle.c`` -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; every number is computed in ``oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so with gcc (-O2, OpenMP, strict IEEE)."""
    with _lock:
        if (not force and os.path.exists(_SO)
                and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
            return _SO
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fno-fast-math", "-ffp-contract=off",
               "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        return _SO


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.orc_num_threads.restype = ctypes.c_int
        _lib.orc_poisson_solve.restype = ctypes.c_int
        _lib.orc_helmholtz_z_solve.restype = ctypes.c_int
        _lib.orc_helmholtz_z_solve_columns.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def z_tables(zc, zf):
    zc, zf = _c(zc), _c(zf)
    nz = zc.size
    assert zf.size == nz + 1
    dzf, dzc = np.empty(nz), np.empty(max(nz - 1, 0))
    A, C = np.empty(nz), np.empty(nz)
    lib().orc_z_tables(ctypes.c_int(nz), _p(zc), _p(zf), _p(dzf),
                       _p(dzc) if nz > 1 else None, _p(A), _p(C))
    return dzf, dzc, A, C


def modified_wavenumbers(n: int, length: float) -> np.ndarray:
    lam = np.empty(n)
    lib().orc_lambda(ctypes.c_int(n), ctypes.c_double(length), _p(lam))
    return lam


def dft_naive(x: np.ndarray, sign: int = -1) -> np.ndarray:
    x = np.asarray(x, dtype=np.complex128)
    n = x.size
    re, im = _c(x.real), _c(x.imag)
    outr, outi = np.empty(n), np.empty(n)
    lib().orc_dft_naive(ctypes.c_int(n), ctypes.c_int(sign), _p(re), _p(im), _p(outr), _p(outi))
    return outr + 1j * outi


def fft_radix2(x: np.ndarray, sign: int = -1) -> np.ndarray:
    x = np.asarray(x, dtype=np.complex128)
    n = x.size
    assert n & (n - 1) == 0
    re, im = _c(x.real).copy(), _c(x.imag).copy()
    lib().orc_fft_radix2(ctypes.c_int(n), ctypes.c_int(sign), _p(re), _p(im))
    return re + 1j * im


def dft_xy(field: np.ndarray, sign: int = -1, variant: int = 1) -> np.ndarray:
    """2-D DFT (x then y) of every z-plane of a [nz][ny][nx] field; no scaling."""
    f = np.asarray(field)
    nz, ny, nx = f.shape
    re = _c(f.real).copy()
    im = _c(f.imag).copy() if np.iscomplexobj(f) else np.zeros_like(re)
    lib().orc_dft_xy(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz), ctypes.c_int(sign),
                     ctypes.c_int(variant), _p(re), _p(im))
    return re + 1j * im


def thomas(lo, di, up, d) -> np.ndarray:
    lo, di, up, d = _c(lo), _c(di), _c(up), _c(d)
    n = d.size
    x, work = np.empty(n), np.empty(2 * n)
    lib().orc_thomas(ctypes.c_int(n), _p(lo), _p(di), _p(up), _p(d), _p(x),
                     ctypes.c_size_t(1), _p(work))
    return x


def thomas_poisson(A, C, sigma: float, d) -> np.ndarray:
    A, C, d = _c(A), _c(C), _c(d)
    nz = d.size
    phi, work = np.empty(nz), np.empty(2 * nz)
    lib().orc_thomas_poisson(ctypes.c_int(nz), _p(A), _p(C), ctypes.c_double(sigma), _p(d),
                             _p(phi), ctypes.c_size_t(1), _p(work))
    return phi


def zero_mode_column(dzf, dzc, d) -> np.ndarray:
    dzf, dzc, d = _c(dzf), _c(dzc), _c(d)
    nz = d.size
    phi = np.empty(nz)
    lib().orc_zero_mode_column(ctypes.c_int(nz), _p(dzf), _p(dzc), _p(d), _p(phi),
                               ctypes.c_size_t(1))
    return phi


def apply_poisson_operator(lx: float, ly: float, zc, zf, phi: np.ndarray) -> np.ndarray:
    phi = _c(phi)
    nz, ny, nx = phi.shape
    zc, zf = _c(zc), _c(zf)
    out = np.empty_like(phi)
    lib().orc_apply_poisson_operator(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                     ctypes.c_double(lx), ctypes.c_double(ly),
                                     _p(zc), _p(zf), _p(phi), _p(out))
    return out


def helmholtz_matrix(zc, zf, a: float):
    zc, zf = _c(zc), _c(zf)
    nz = zc.size
    lo, di, up = np.empty(nz), np.empty(nz), np.empty(nz)
    lib().orc_helmholtz_matrix(ctypes.c_int(nz), _p(zc), _p(zf), ctypes.c_double(a),
                               _p(lo), _p(di), _p(up))
    return lo, di, up


def poisson_solve(lx: float, ly: float, zc, zf, f: np.ndarray, variant: int = 1) -> np.ndarray:
    """f[nz][ny][nx] -> phi, definition O-P.  variant 0: O(n^2) DFT; 1: radix-2 FFT."""
    f = _c(f)
    nz, ny, nx = f.shape
    zc, zf = _c(zc), _c(zf)
    assert zc.size == nz and zf.size == nz + 1
    phi = np.empty_like(f)
    rc = lib().orc_poisson_solve(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                 ctypes.c_double(lx), ctypes.c_double(ly), _p(zc), _p(zf),
                                 _p(f), _p(phi), ctypes.c_int(variant))
    if rc != 0:
        raise MemoryError("orc_poisson_solve: allocation failed")
    return phi


def helmholtz_z_solve(zc, zf, a: float, r: np.ndarray) -> np.ndarray:
    """r[nz][ny][nx] -> u, definition O-H."""
    r = _c(r)
    nz, ny, nx = r.shape
    zc, zf = _c(zc), _c(zf)
    u = np.empty_like(r)
    rc = lib().orc_helmholtz_z_solve(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                     _p(zc), _p(zf), ctypes.c_double(a), _p(r), _p(u))
    if rc != 0:
        raise MemoryError("orc_helmholtz_z_solve: allocation failed")
    return u


def helmholtz_w_matrix(zc, zf, a: float):
    """(lo, di, up) of I - a L_z^w for the face-centred wall-normal velocity (reading R16)."""
    zc, zf = _c(zc), _c(zf)
    nz = zc.size
    lo, di, up = np.empty(nz), np.empty(nz), np.empty(nz)
    lib().orc_helmholtz_w_matrix(ctypes.c_int(nz), _p(zc), _p(zf), ctypes.c_double(a), _p(lo), _p(di), _p(up))
    return lo, di, up


def helmholtz_w_solve(zc, zf, a: float, r: np.ndarray) -> np.ndarray:
    """r[nz][ny][nx] -> w on the z faces zf[1..nz] (w[nz-1] = the top wall face, unchanged)."""
    r = _c(r)
    nz, ny, nx = r.shape
    zc, zf = _c(zc), _c(zf)
    w = np.empty_like(r)
    rc = lib().orc_helmholtz_w_solve(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                     _p(zc), _p(zf), ctypes.c_double(a), _p(r), _p(w))
    if rc != 0:
        raise MemoryError("orc_helmholtz_w_solve: allocation failed")
    return w


def helmholtz_z_solve_columns(zc, zf, a: float, rcols: np.ndarray) -> np.ndarray:
    """rcols[ncols][nz] -> ucols; the same column solve on sampled columns only."""
    rcols = _c(rcols)
    ncols, nz = rcols.shape
    zc, zf = _c(zc), _c(zf)
    ucols = np.empty_like(rcols)
    rc = lib().orc_helmholtz_z_solve_columns(ctypes.c_int(nz), _p(zc), _p(zf), ctypes.c_double(a),
                                             ctypes.c_longlong(ncols), _p(rcols), _p(ucols))
    if rc != 0:
        raise MemoryError("orc_helmholtz_z_solve_columns: allocation failed")
    return ucols


def apply_helmholtz3d_operator(lx: float, ly: float, zc, zf, a: float, u: np.ndarray) -> np.ndarray:
    """u[nz][ny][nx] -> (I - a L_h) u, definition O-H3 (periodic x, y; Dirichlet walls in z)."""
    u = _c(u)
    nz, ny, nx = u.shape
    zc, zf = _c(zc), _c(zf)
    out = np.empty_like(u)
    lib().orc_apply_helmholtz3d_operator(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                         ctypes.c_double(lx), ctypes.c_double(ly), _p(zc), _p(zf),
                                         ctypes.c_double(a), _p(u), _p(out))
    return out


def helmholtz3d_solve(lx: float, ly: float, zc, zf, a: float, r: np.ndarray, variant: int = 1) -> np.ndarray:
    """r[nz][ny][nx] -> u with (I - a L_h) u = r (Eq. 8).  variant as poisson_solve."""
    r = _c(r)
    nz, ny, nx = r.shape
    zc, zf = _c(zc), _c(zf)
    u = np.empty_like(r)
    rc = lib().orc_helmholtz3d_solve(ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
                                     ctypes.c_double(lx), ctypes.c_double(ly), _p(zc), _p(zf),
                                     ctypes.c_double(a), _p(r), _p(u), ctypes.c_int(variant))
    if rc != 0:
        raise MemoryError("orc_helmholtz3d_solve: allocation failed")
    return u
