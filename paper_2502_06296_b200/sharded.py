"""ONE problem spread over the GPUs of a node, one process per GPU.

* :class:`SlabPoisson` -- the paper's parallel tridiagonal solver with GPUs for its MPI tasks
  (PAPER.md:120-135): rank g owns the planes ``[kb[g], kb[g+1])``; x and y transforms are
  plane-local; ``poisson_solve_reduce`` leaves 2 nx ny boundary values per rank, ONE all-gather
  (NCCL over NVLink) moves them, ``poisson_solve_finish`` solves the size-2G reduced systems
  redundantly and reconstructs.  The reduced coefficients are computed by every rank at plan time
  (PAPER.md:199), so plan creation needs no collective.
* :class:`YSlabHelmholtz` -- wall-normal implicit diffusion: the columns are independent
  (Eq. 11), rank g owns the rows ``[j0, j1)`` of y and solves them with an ordinary
  plan of that ny; no collective at all.

Only marshalling lives here: every arithmetic step runs in libpz_b200.so.  The all-gather is the
caller's process group (``torch.distributed``: nccl on GPUs, gloo in the CPU plumbing tests).
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from . import ranks


class SlabPoisson:
    """Rank ``rank`` of ``world`` of one Poisson problem on the global grid (nx, ny, nz)."""

    def __init__(self, nx: int, ny: int, nz: int, lx: float, ly: float, zc, zf, rank: int, world: int,
                 kbounds: Optional[Sequence[int]] = None, device="cuda"):
        import torch

        from . import binding as pz

        self.pz, self.torch = pz, torch
        self.rank, self.world = rank, world
        self.kb = list(kbounds) if kbounds is not None else ranks.z_slab_bounds(nz, world)
        self.k0, self.k1 = self.kb[rank], self.kb[rank + 1]
        self.plan = pz.poisson_slab_plan_create(nx, ny, nz, lx, ly, zc, zf, world, rank, self.kb)
        self.stride = pz.poisson_slab_boundary_doubles(self.plan)
        self.bout = torch.zeros(self.stride, dtype=torch.float64, device=device)
        self.ball = torch.zeros(self.stride * world, dtype=torch.float64, device=device)

    @property
    def bytes_exchanged_per_solve(self) -> int:
        """Bytes this rank contributes to the all-gather of one solve."""
        return 8 * self.stride

    def solve(self, p_local, dist=None) -> None:
        """In place on this rank's planes ``p_local[k1 - k0][ny][nx]``: rhs in, phi out."""
        self.pz.poisson_solve_reduce(self.plan, p_local, self.bout)
        ranks.gather_boundaries(self.ball, self.bout, dist)
        self.pz.poisson_solve_finish(self.plan, p_local, self.ball)

    def destroy(self) -> None:
        self.pz.poisson_plan_destroy(self.plan)


class YSlabHelmholtz:
    """Rank ``rank`` of ``world`` of the wall-normal Helmholtz solve of fields on (nx, ny, nz):
    rows ``[j0, j1)`` of y, solved by an ordinary plan with ny = j1 - j0 (no collective)."""

    def __init__(self, nx: int, ny: int, nz: int, lx: float, ly: float, zc, zf, a: float, rank: int, world: int):
        from . import binding as pz

        self.pz = pz
        self.j0, self.j1 = ranks.y_slab_pow2(ny, rank, world)
        self.plan = pz.poisson_plan_create(nx, self.j1 - self.j0, nz, lx, ly * (self.j1 - self.j0) / ny, zc, zf)
        pz.helmholtz_z_setup(self.plan, a)

    def solve(self, fields_local) -> None:
        """In place on this rank's slabs ``u[nz][j1 - j0][nx]`` (contiguous)."""
        self.pz.helmholtz_z_solve_n(self.plan, list(fields_local))

    def destroy(self) -> None:
        self.pz.poisson_plan_destroy(self.plan)


def split_z(field: np.ndarray, kb: Sequence[int]):
    """Host helper for tests: the z-slabs of a global field, each contiguous."""
    return [np.ascontiguousarray(field[kb[g]:kb[g + 1]]) for g in range(len(kb) - 1)]
