"""Oracle for the steps either side of the Poisson solve: the right-hand
side of Eq. (4), D u* / (gamma dt), and the correction of Eqs. (5)-(6), u -= gamma dt G Phi,
p += Phi, on the staggered (MAC) grid of PAPER.md:49.  TEST INFRASTRUCTURE ONLY.

Plain numpy, float64, written straight from the definitions (reading R15, the paper
gives no index convention): all arrays are [k][j][i];
  u[k][j][i]  x-velocity on the face between cells i and i+1 (periodic),
  v[k][j][i]  y-velocity on the face between cells j and j+1 (periodic),
  w[k][j][i]  z-velocity on the face zf[k+1] (top face of cell k); the bottom wall face zf[0]
              carries w = 0 and is not stored; w[nz-1] is the top wall face,
  p, Phi      cell centres.
  (D u)_ijk   = (u_i - u_{i-1})/dx + (v_j - v_{j-1})/dy + (w_k - w_{k-1})/dzf_k,  w_{-1} = 0
  (G Phi)^x_i = (Phi_{i+1} - Phi_i)/dx, (G Phi)^y_j likewise,
  (G Phi)^z_k = (Phi_{k+1} - Phi_k)/dzc_k for k <= nz-2 and 0 on the top wall face,
so that D G = L_h, the operator of the Poisson solve (definition O-P), exactly.
"""
from __future__ import annotations

import numpy as np


def divergence(lx: float, ly: float, zf, u: np.ndarray, v: np.ndarray, w: np.ndarray) -> np.ndarray:
    """(D u)[k][j][i] on cell centres."""
    nz, ny, nx = u.shape
    dx, dy = lx / nx, ly / ny
    dzf = np.diff(np.asarray(zf, dtype=np.float64))
    d = (u - np.roll(u, 1, axis=2)) / dx + (v - np.roll(v, 1, axis=1)) / dy
    wz = w.copy()
    wz[1:] -= w[:-1]                    # w_k - w_{k-1}; the bottom wall face is zero
    return d + wz / dzf[:, None, None]


def divergence_rhs(lx, ly, zf, u, v, w, inv_gdt: float) -> np.ndarray:
    """Right-hand side of Eq. (4): D u* / (gamma_k dt), inv_gdt = 1 / (gamma_k dt)."""
    return divergence(lx, ly, zf, u, v, w) * inv_gdt


def gradient(lx: float, ly: float, zc, phi: np.ndarray):
    """(G Phi) on the x-, y- and z-faces; zero on the top wall face."""
    nz, ny, nx = phi.shape
    dx, dy = lx / nx, ly / ny
    dzc = np.diff(np.asarray(zc, dtype=np.float64))
    gx = (np.roll(phi, -1, axis=2) - phi) / dx
    gy = (np.roll(phi, -1, axis=1) - phi) / dy
    gz = np.zeros_like(phi)
    gz[:-1] = (phi[1:] - phi[:-1]) / dzc[:, None, None]
    return gx, gy, gz


def project(lx, ly, zc, u, v, w, p, phi, gdt: float):
    """Eqs. (5)-(6): returns (u - gdt G Phi, v - ..., w - ..., p + Phi), gdt = gamma_k dt."""
    gx, gy, gz = gradient(lx, ly, zc, phi)
    return u - gdt * gx, v - gdt * gy, w - gdt * gz, p + phi


def helmholtz_z_rhs(zc, zf, a: float, ustar2: np.ndarray, uk: np.ndarray) -> np.ndarray:
    """Right-hand side of Eq. (11): u** - a L_z u^k with a = gamma_k nu dt / 2 and L_z
    the wall-normal operator of definition O-H (Dirichlet walls, reading R7):
    (L_z q)_k = A_k (q_{k-1} - q_k) + C_k (q_{k+1} - q_k) - W_k q_k."""
    zc, zf = np.asarray(zc, dtype=np.float64), np.asarray(zf, dtype=np.float64)
    dzf, dzc = np.diff(zf), np.diff(zc)
    nz = zc.size
    lz = np.zeros_like(uk)
    lz[1:] += (1.0 / (dzf[1:] * dzc))[:, None, None] * (uk[:-1] - uk[1:])
    lz[:-1] += (1.0 / (dzf[:-1] * dzc))[:, None, None] * (uk[1:] - uk[:-1])
    lz[0] -= 2.0 / (dzf[0] * (2.0 * (zc[0] - zf[0]))) * uk[0]
    lz[nz - 1] -= 2.0 / (dzf[nz - 1] * (2.0 * (zf[nz] - zc[nz - 1]))) * uk[nz - 1]
    return ustar2 - a * lz
