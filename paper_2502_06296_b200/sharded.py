"""ONE problem spread over the GPUs of a node, one process per GPU.

* :class:`SlabPoisson` -- the paper's parallel tridiagonal solver with GPUs for its MPI tasks
  (PAPER.md:120-135): rank g owns the planes ``[kb[g], kb[g+1])``; x and y transforms are
  plane-local; ``poisson_solve_reduce`` leaves 2 nx ny boundary values per rank, ONE all-gather
  (NCCL over NVLink) moves them -- or the reduction kernel itself stores them into every rank's
  buffer over peer memory (``exchange="p2p"``) --, ``poisson_solve_finish`` solves the size-2G
  reduced systems redundantly and reconstructs.  The reduced coefficients are computed by every rank at plan time
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
    """Rank ``rank`` of ``world`` of one Poisson problem on the global grid (nx, ny, nz).

    exchange = "allgather": ``poisson_solve_reduce`` -> one ``all_gather_into_tensor`` (NCCL) ->
    ``poisson_solve_finish``.
    exchange = "p2p": the reduction kernel stores this rank's boundary block straight into every
    rank's gathered buffer over peer memory and raises a flag; the finish waits for the flags on the
    device (``poisson_solve_reduce_push`` / ``poisson_solve_finish_wait``): no collective, no host
    synchronisation.  With a process ``group`` the buffers live in
    ``torch.distributed._symmetric_memory`` (peer-mapped over NVLink; not run on hardware in this
    pool, which has single-GPU boxes); without one the ranks of a job live in ONE process and are
    wired together with :meth:`connect` (the emulation the GPU tests use).  Two buffer sets alternate
    between consecutive solves.
    """

    def __init__(self, nx: int, ny: int, nz: int, lx: float, ly: float, zc, zf, rank: int, world: int,
                 kbounds: Optional[Sequence[int]] = None, device="cuda", exchange: str = "allgather", group=None):
        import torch

        from . import binding as pz

        self.pz, self.torch = pz, torch
        self.rank, self.world = rank, world
        self.kb = list(kbounds) if kbounds is not None else ranks.z_slab_bounds(nz, world)
        self.k0, self.k1 = self.kb[rank], self.kb[rank + 1]
        self.plan = pz.poisson_slab_plan_create(nx, ny, nz, lx, ly, zc, zf, world, rank, self.kb)
        self.stride = pz.poisson_slab_boundary_doubles(self.plan)
        self.exchange = exchange
        self.epoch = 0
        self.peers = None
        if exchange == "allgather":
            self.bout = torch.zeros(self.stride, dtype=torch.float64, device=device)
            self.ball = torch.zeros(self.stride * world, dtype=torch.float64, device=device)
        elif exchange == "p2p":
            # one allocation per rank: [ball set 0 | ball set 1 | flags set 0 | flags set 1]
            self.nball = self.stride * world
            total = 2 * self.nball + 2 * world
            if group is not None:
                import torch.distributed._symmetric_memory as symm

                self.sym = symm.empty(total, dtype=torch.float64, device=device)
                self.sym.zero_()
                handle = symm.rendezvous(self.sym, group)
                base = [int(a) for a in handle.buffer_ptrs]
                handle.barrier()
            else:  # single process: the caller wires the ranks together with connect()
                self.sym = torch.zeros(total, dtype=torch.float64, device=device)
                base = None
            if base is not None:
                self._wire(base)
        else:
            raise ValueError("exchange must be 'allgather' or 'p2p'")

    def _wire(self, base):
        """base[r] = device address of rank r's allocation."""
        nb, w = self.nball, self.world
        self.peers = [([b + 8 * (s * nb) for b in base], [b + 8 * (2 * nb + s * w) for b in base]) for s in (0, 1)]
        self.ball_sets = [self.sym[s * nb:(s + 1) * nb] for s in (0, 1)]
        self.flag_sets = [self.sym[2 * nb + s * w:2 * nb + (s + 1) * w].view(self.torch.int64) for s in (0, 1)]

    @staticmethod
    def connect(jobs) -> None:
        """Wire the p2p ranks of ONE process to one another (emulation of a job on a single GPU)."""
        base = [int(j.sym.data_ptr()) for j in jobs]
        for j in jobs:
            j._wire(base)

    @property
    def bytes_exchanged_per_solve(self) -> int:
        """Bytes this rank contributes to the exchange of one solve (per destination rank)."""
        return 8 * self.stride

    def reduce(self, p_local) -> None:
        if self.exchange == "allgather":
            self.pz.poisson_solve_reduce(self.plan, p_local, self.bout)
        else:
            self.epoch += 1
            balls, flags = self.peers[self.epoch & 1]
            self.pz.poisson_solve_reduce_push(self.plan, p_local, balls, flags, self.epoch)

    def finish(self, p_local, dist=None) -> None:
        if self.exchange == "allgather":
            ranks.gather_boundaries(self.ball, self.bout, dist)
            self.pz.poisson_solve_finish(self.plan, p_local, self.ball)
        else:
            s = self.epoch & 1
            self.pz.poisson_solve_finish_wait(self.plan, p_local, self.ball_sets[s], self.flag_sets[s], self.epoch)

    def solve(self, p_local, dist=None) -> None:
        """In place on this rank's planes ``p_local[k1 - k0][ny][nx]``: rhs in, phi out."""
        self.reduce(p_local)
        self.finish(p_local, dist)

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
