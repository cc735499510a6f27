"""The N > 1 path on CPU: two gloo ranks shard a Helmholtz field into y-slabs (columns are
independent), each solves its slab with the ORACLE (this is a test of the
sharding and rank plumbing, not of the kernels), the slabs are gathered and must equal the
unsharded solve bit for bit; the timing reduction is a MAX over ranks."""
import os
import socket

import numpy as np
import pytest

from paper_2502_06296_b200 import ranks


def test_y_slab_partitions_cover_exactly():
    for ny in (8, 64, 96, 512):
        for world in (1, 2, 3, 8):
            for align in (1, 8):
                if ny % align:
                    continue
                edges = [ranks.y_slab(ny, r, world, align) for r in range(world)]
                assert edges[0][0] == 0 and edges[-1][1] == ny
                for (a0, a1), (b0, b1) in zip(edges, edges[1:]):
                    assert a1 == b0
                sizes = [b - a for a, b in edges]
                assert max(sizes) - min(sizes) <= align
                assert all(a % align == 0 for a, _ in edges)
    with pytest.raises(ValueError):
        ranks.y_slab(8, 2, 2)


def test_seeds_and_rates():
    assert ranks.rank_seed(5, 0) == 5 and ranks.rank_seed(5, 3) == 3005
    assert ranks.whole_job_rate(1e6, 4, 2.0) == pytest.approx(2e9)
    assert ranks.max_over_ranks(1.5) == 1.5


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist

    import oracle
    from paper_2502_06296_b200 import workloads as wl

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nx, ny, nz, a = 16, 24, 40, 3e-4
        zf = wl.z_faces(nz, 2.0, 1.8)
        zc = wl.z_centres(zf)
        r = np.random.default_rng(11).standard_normal((nz, ny, nx))   # same seed on every rank
        j0, j1 = ranks.y_slab(ny, rank, world, align=8)
        mine = oracle.helmholtz_z_solve(zc, zf, a, np.ascontiguousarray(r[:, j0:j1, :]))
        parts = [None] * world
        dist.all_gather_object(parts, (j0, j1, mine))
        full = np.empty_like(r)
        for b0, b1, part in parts:
            full[:, b0:b1, :] = part
        ms = ranks.max_over_ranks(10.0 + rank, dist)                 # slowest rank wins
        if rank == 0:
            ref = oracle.helmholtz_z_solve(zc, zf, a, r)
            np.save(os.path.join(out_dir, "ok.npy"), np.array([float(np.array_equal(full, ref)), ms]))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_helmholtz_by_y_slabs(tmp_path):
    import torch.multiprocessing as mp

    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    ok, ms = np.load(tmp_path / "ok.npy")
    assert ok == 1.0
    assert ms == 10.0 + world - 1


def test_z_slab_bounds_and_pow2_y_slabs():
    for nz, world in ((12, 4), (512, 8), (100, 3), (1594, 4), (30, 1)):
        kb = ranks.z_slab_bounds(nz, world)
        sizes = np.diff(kb)
        assert kb[0] == 0 and kb[-1] == nz and len(kb) == world + 1
        assert sizes.min() >= 3 and sizes.max() - sizes.min() <= 1
    with pytest.raises(ValueError):
        ranks.z_slab_bounds(8, 3)
    assert [ranks.y_slab_pow2(64, r, 4) for r in range(4)] == [(0, 16), (16, 32), (32, 48), (48, 64)]
    with pytest.raises(ValueError):
        ranks.y_slab_pow2(64, 0, 16)    # 4 rows per rank: below a plan's minimum
    with pytest.raises(ValueError):
        ranks.y_slab_pow2(64, 0, 3)


def _ptdma_worker(rank, world, port, out_dir):
    """The z-slab plumbing of sharded.SlabPoisson on CPU: every rank reduces ITS rows of a batch of
    tridiagonal systems with the oracle's Algorithm 1, the boundary rows go through
    ranks.gather_boundaries (the product's ONE collective), every rank solves the reduced systems
    of size 2 world redundantly and reconstructs its rows."""
    import torch
    import torch.distributed as dist

    from oracle import algorithms as alg

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nz, ncol = 23, 5
        rng = np.random.default_rng(3)                      # same systems on every rank
        lo, up = -rng.uniform(0.5, 1.5, (ncol, nz)), -rng.uniform(0.5, 1.5, (ncol, nz))
        di = np.abs(lo) + np.abs(up) + rng.uniform(0.01, 0.5, (ncol, nz))
        lo[:, 0] = 0.0
        up[:, -1] = 0.0
        d = rng.standard_normal((ncol, nz))
        kb = ranks.z_slab_bounds(nz, world)
        k0, k1 = kb[rank], kb[rank + 1]
        state, bout = [], torch.zeros(6 * ncol, dtype=torch.float64)
        for q in range(ncol):
            a, c, dd = alg.algorithm1_reduce(lo[q, k0:k1], di[q, k0:k1], up[q, k0:k1], d[q, k0:k1])
            state.append((a, c, dd))
            bout[6 * q:6 * q + 6] = torch.tensor([a[0], c[0], dd[0], a[-1], c[-1], dd[-1]])
        ball = torch.zeros(6 * ncol * world, dtype=torch.float64)
        ranks.gather_boundaries(ball, bout, dist)
        rows = ball.numpy().reshape(world, ncol, 6)
        mine = np.empty((ncol, k1 - k0))
        for q in range(ncol):
            red = [((rows[g, q, 0], 1.0, rows[g, q, 1], rows[g, q, 2]), (rows[g, q, 3], 1.0, rows[g, q, 4], rows[g, q, 5]))
                   for g in range(world)]
            xb = alg._dense_tridiag_solve(*alg.reduced_system(red))
            a, c, dd = state[q]
            mine[q] = alg.algorithm1_reconstruct(a, c, dd, xb[2 * rank], xb[2 * rank + 1])
        parts = [None] * world
        dist.all_gather_object(parts, (k0, k1, mine))
        if rank == 0:
            full = np.empty((ncol, nz))
            for b0, b1, part in parts:
                full[:, b0:b1] = part
            ref = np.stack([alg._dense_tridiag_solve(lo[q], di[q], up[q], d[q]) for q in range(ncol)])
            np.save(os.path.join(out_dir, "err.npy"), np.array([np.abs(full - ref).max() / np.abs(ref).max()]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_ranks_solve_z_slabs_through_gather_boundaries(tmp_path, world):
    import torch.multiprocessing as mp

    mp.spawn(_ptdma_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert np.load(tmp_path / "err.npy")[0] <= 1e-13
