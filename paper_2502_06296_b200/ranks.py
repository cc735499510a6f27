"""One process per GPU: how the hot path shards, and the rank plumbing bench.py and sharded.py use.



* Helmholtz: every (i, j) column is an independent tridiagonal system (Eq. 11),
  so a field splits into y-slabs ``[:, j0:j1, :]``, one per rank, each solved by an ordinary plan
  with ``ny = j1 - j0``; no collective.
* ONE Poisson problem: z-slabs ``[k0:k1, :, :]`` and the paper's parallel tridiagonal solver
  (PAPER.md:120-135): one all-gather of 2 nx ny boundary values per rank and solve
  (:func:`gather_boundaries`).
* Independent problems (replicas, ``bench.py --scaling weak``): every rank its own, no collective.

This module holds no arithmetic of the method and works with the ``gloo`` backend on CPU (tests)
and ``nccl`` on GPUs.
"""
from __future__ import annotations

import os
from typing import List, Tuple


def env_rank() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment (defaults: single process)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def y_slab(ny: int, rank: int, world: int, align: int = 1) -> Tuple[int, int]:
    """Rows [j0, j1) of the y direction owned by ``rank``: contiguous, in rank order, covering
    [0, ny) exactly, sizes differing by at most ``align``; every boundary is a multiple of ``align``."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world size")
    if ny % align:
        raise ValueError("ny must be a multiple of align")
    units = ny // align
    base, extra = divmod(units, world)
    j0 = rank * base + min(rank, extra)
    j1 = j0 + base + (1 if rank < extra else 0)
    return j0 * align, j1 * align


def y_slab_pow2(ny: int, rank: int, world: int) -> Tuple[int, int]:
    """y-slab of a Helmholtz field for a plan: the plan's transforms want ny' a multiple of 8, and
    equal slabs keep every rank's work the same; needs world | ny and ny / world >= 8."""
    if world < 1 or ny % world or (ny // world) % 8:
        raise ValueError(f"ny = {ny} does not split into {world} y-slabs of a multiple of 8 rows")
    return y_slab(ny, rank, world, align=ny // world)


def z_slab_bounds(nz: int, world: int) -> List[int]:
    """Plane bounds kb[0..world] of the z-slabs of one Poisson problem: contiguous, sizes differing
    by at most one, at least 3 planes each (Algorithms 1 and 2 need three rows per sub-domain,
    PAPER.md:284, reading R9)."""
    if world < 1 or nz < 3 * world:
        raise ValueError(f"nz = {nz} cannot be cut into {world} slabs of at least 3 planes")
    base, extra = divmod(nz, world)
    kb = [0]
    for g in range(world):
        kb.append(kb[-1] + base + (1 if g < extra else 0))
    return kb


def gather_boundaries(ball, bout, dist=None) -> None:
    """The ONE collective of a z-slab Poisson solve: every rank's boundary
    buffer ``bout`` (stride doubles) lands at ``ball[rank * stride : (rank + 1) * stride]`` on every
    rank.  Without a process group (single rank) it is a copy."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        ball[: bout.numel()].copy_(bout)
        return
    if ball.numel() != bout.numel() * dist.get_world_size():
        raise ValueError("gather_boundaries: ball must hold world_size buffers of bout's size")
    dist.all_gather_into_tensor(ball, bout)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the rank's own synthetic input in a weak-scaling run (rank 0 keeps the config's seed)."""
    return seed + 1000 * rank


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a per-rank device time (ms); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world: int, ms_max: float) -> float:
    """Whole-job throughput: units all ranks processed / slowest rank's time."""
    return units_per_rank * world / (ms_max * 1e-3)
