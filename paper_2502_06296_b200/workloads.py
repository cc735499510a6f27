"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module is the ONLY thing shared by the CUDA path's tests/bench and the CPU oracle's
tests: it builds grids and right-hand sides and holds none of the method's arithmetic (no
transforms, no tridiagonal coefficients, no solves).  The paper measures on its own DNS
fields (turbulent channel), which are not available; these inputs take
their structure -- channel-shaped box, tanh-stretched wall-normal grid, broadband or
few-mode right-hand sides -- and stand in for them.

Arrays are float64, C-order ``[k][j][i]`` (x fastest).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    lx: float
    ly: float
    lz: float
    beta: float          # tanh stretching factor, 0 = uniform
    poisson: bool
    n_helmholtz: int     # velocity components the Helmholtz solve is applied to
    dt_nu: float         # a = 0.5 * dt_nu  (gamma_k = 1)
    poisson_seed: int
    helmholtz_seeds: tuple
    rhs_kind: str        # "normal" | "modes"
    repeats: int         # solves with a fixed plan (configs 3 and 4)

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def a(self) -> float:
        return 0.5 * self.dt_nu


PI = math.pi

# BASELINE.json "configs", in order.
CONFIGS = {
    "c0": Workload("c0", 64, 64, 64, 2 * PI, 2 * PI, 2.0, 0.0, True, 0, 0.0, 0, (), "normal", 1),
    "c1": Workload("c1", 256, 256, 256, 4 * PI, 2 * PI, 2.0, 1.8, True, 1, 1e-4, 1, (2,), "normal", 1),
    "c2": Workload("c2", 512, 512, 512, 4 * PI, 2 * PI, 2.0, 1.8, True, 3, 1e-4, 3, (4, 5, 6), "modes", 1),
    "c3": Workload("c3", 2048, 1024, 512, 8 * PI, 3 * PI, 2.0, 2.0, True, 0, 0.0, 7, (), "normal", 20),
    "c4": Workload("c4", 1024, 1024, 1024, 4 * PI, 2 * PI, 2.0, 1.8, False, 3, 5e-5, 0, (8, 9, 10), "normal", 100),
}


def scaled(w: Workload, nx: int, ny: int, nz: int, name: str | None = None) -> Workload:
    """Same recipe on a smaller grid (CPU tests, ragged-tile parity cases)."""
    return dataclasses.replace(w, nx=nx, ny=ny, nz=nz, name=name or f"{w.name}_{nx}x{ny}x{nz}")


def z_faces(nz: int, lz: float = 2.0, beta: float = 0.0) -> np.ndarray:
    """Wall-normal cell faces zf[0..nz] on [0, lz].

    beta = 0: uniform ``lz*k/nz``.  beta > 0: BASELINE.json's
    ``z_k = 1 + tanh(beta*(2k/nz - 1))/tanh(beta)`` scaled by lz/2 (clustered at both walls).
    """
    k = np.arange(nz + 1, dtype=np.float64)
    if beta == 0.0:
        zf = lz * k / nz
    else:
        zf = 0.5 * lz * (1.0 + np.tanh(beta * (2.0 * k / nz - 1.0)) / math.tanh(beta))
    zf[0] = 0.0
    zf[-1] = lz
    return zf


def z_centres(zf: np.ndarray) -> np.ndarray:
    """Mid-point cell centres zc[k] = (zf[k] + zf[k+1]) / 2."""
    return 0.5 * (zf[:-1] + zf[1:])


def grid(w: Workload):
    zf = z_faces(w.nz, w.lz, w.beta)
    return z_centres(zf), zf


def remove_weighted_mean(f: np.ndarray, zf: np.ndarray) -> np.ndarray:
    """Make a Poisson right-hand side compatible: subtract its cell-volume (dzf-weighted) mean.

    The discrete Neumann problem is solvable iff sum_ijk dzf_k f_ijk = 0 (the left null vector
    of the wall-normal operator is dzf, not 1); on a uniform grid this is the arithmetic mean.
    """
    dzf = np.diff(zf)
    plane_means = f.mean(axis=(1, 2))
    mean = float(np.dot(dzf, plane_means) / dzf.sum())
    return f - mean


def _modes_field(w: Workload, seed: int, zc: np.ndarray) -> np.ndarray:
    """config 2: sum of 32 seeded Fourier-x,y times Chebyshev-z modes + N(0, 1e-3) noise."""
    rng = np.random.default_rng(seed)
    nm = 32
    p = rng.integers(0, max(w.nx // 8, 1), nm)
    r = rng.integers(0, max(w.ny // 8, 1), nm)
    q = rng.integers(0, 16, nm)
    amp = rng.standard_normal(nm)
    th = rng.uniform(0.0, 2 * PI, nm)
    vt = rng.uniform(0.0, 2 * PI, nm)
    x = (np.arange(w.nx) + 0.5) * (w.lx / w.nx)
    y = (np.arange(w.ny) + 0.5) * (w.ly / w.ny)
    zz = np.clip(zc * (2.0 / w.lz) - 1.0, -1.0, 1.0)
    f = 1e-3 * rng.standard_normal((w.nz, w.ny, w.nx))
    for m in range(nm):
        cx = np.cos(2 * PI * p[m] * x / w.lx + th[m])
        cy = np.cos(2 * PI * r[m] * y / w.ly + vt[m])
        tz = np.cos(q[m] * np.arccos(zz))
        f += amp[m] * tz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    return f


def field(w: Workload, seed: int, zc: np.ndarray | None = None) -> np.ndarray:
    """One seeded float64 field of the workload's kind (no mean removal)."""
    if w.rhs_kind == "modes":
        if zc is None:
            zc, _ = grid(w)
        return _modes_field(w, seed, zc)
    rng = np.random.default_rng(seed)
    return rng.standard_normal((w.nz, w.ny, w.nx))


def poisson_rhs(w: Workload) -> np.ndarray:
    zc, zf = grid(w)
    return remove_weighted_mean(field(w, w.poisson_seed, zc), zf)


def helmholtz_rhs(w: Workload, component: int = 0) -> np.ndarray:
    zc, _ = grid(w)
    return field(w, w.helmholtz_seeds[component], zc)


# ---- device-side generators for the two configurations too large to build on the host quickly

def device_field(w: Workload, seed: int, device="cuda"):
    """N(0,1) float64 field generated on the device by torch's seeded Philox generator.

    Used for c3 / c4 (about 1.07e9 points): both the CUDA path and -- on sampled columns or
    stencil points copied back to the host -- the oracle see the same values.
    """
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return torch.randn((w.nz, w.ny, w.nx), dtype=torch.float64, device=device, generator=g)


def device_remove_weighted_mean(f, zf: np.ndarray):
    import torch

    dzf = torch.as_tensor(np.diff(zf), dtype=torch.float64, device=f.device)
    plane_means = f.mean(dim=(1, 2))
    mean = torch.dot(dzf, plane_means) / dzf.sum()
    f -= mean
    return f
