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


def test_deal_fields_and_rates():
    assert ranks.deal_fields(3, 0, 2) == [0, 2] and ranks.deal_fields(3, 1, 2) == [1]
    assert sorted(sum((ranks.deal_fields(7, r, 4) for r in range(4)), [])) == list(range(7))
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
