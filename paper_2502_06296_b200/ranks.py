"""One process per GPU: how the hot path shards, and the rank plumbing bench.py uses.

The path shards without any data-path collective:

* Helmholtz: every (i, j) column is an independent tridiagonal system (Eq. 11),
  so a field splits into y-slabs ``[:, j0:j1, :]``, one per rank, each solved by an ordinary plan
  with ``ny = j1 - j0``.
* Poisson on one GPU per problem: independent fields (time steps of independent simulations,
  ensemble members) are dealt round-robin to the ranks.

Only timing (max over ranks) and bookkeeping use ``torch.distributed``; this module holds no
arithmetic of the method and works with the ``gloo`` backend on CPU (tests) and ``nccl`` on GPUs.
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


def deal_fields(n_fields: int, rank: int, world: int) -> List[int]:
    """Indices of the independent fields solved by ``rank`` (round-robin)."""
    return list(range(rank, n_fields, world))


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
