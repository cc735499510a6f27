"""GPU parity of the sharded product paths, emulated on ONE GPU (the pool has single-GPU boxes): the
ranks of a job run one after the other in this process, each through its own plan and the C ABI,
and what NCCL's all-gather would do is a device copy in rank order.

* ONE Poisson problem cut into G z-slabs, the paper's parallel tridiagonal solver with GPUs for its
  MPI tasks: against the oracle (<= 1e-11) and against the single-plan
  CUDA solve (to rounding: "accurate up to machine precision"), for G in {2, 4, 8},
  uneven slabs and slabs of 3 planes (reading R9).
* Helmholtz fields cut into y-slabs (columns are independent): the gathered slabs
  equal the unsharded CUDA solve bit for bit and the oracle to <= 1e-11.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def env():
    import torch

    import oracle
    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import ranks, sharded
    from paper_2502_06296_b200 import workloads as wl

    assert torch.cuda.is_available()
    pz.lib()
    return torch, pz, wl, oracle, ranks, sharded


def rel_err(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def solve_by_slabs(torch, pz, sharded, w, zc, zf, f, kb):
    """Every rank's reduce, the all-gather as copies in rank order, every rank's finish."""
    G = len(kb) - 1
    jobs = [sharded.SlabPoisson(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, g, G, kb) for g in range(G)]
    parts = [torch.from_numpy(s).cuda() for s in sharded.split_z(f, kb)]
    stride = jobs[0].stride
    assert all(j.stride == stride for j in jobs)
    for j, p in zip(jobs, parts):
        pz.poisson_solve_reduce(j.plan, p, j.bout)
    ball = torch.cat([j.bout for j in jobs])
    for j, p in zip(jobs, parts):
        pz.poisson_solve_finish(j.plan, p, ball)
    torch.cuda.synchronize()
    out = np.concatenate([p.cpu().numpy() for p in parts], axis=0)
    for j in jobs:
        j.destroy()
    return out


SLAB_CASES = [
    # (base config, nx, ny, nz, plane bounds)
    ("c0", 16, 8, 12, [0, 6, 12]),
    ("c1", 32, 16, 48, [0, 24, 48]),
    ("c1", 32, 16, 12, [0, 3, 6, 9, 12]),                     # slabs of 3 planes, the minimum (R9)
    ("c1", 64, 32, 96, [0, 24, 48, 72, 96]),
    ("c3", 64, 32, 100, [0, 3, 40, 45, 100]),                 # uneven, beta = 2.0
    ("c3", 32, 64, 128, [0, 16, 32, 48, 64, 80, 96, 112, 128]),
    ("c1", 16, 16, 300, [0, 130, 133, 300]),                  # 130 and 167 rows: m = 8 per lane, ragged
    ("c2", 64, 64, 128, [0, 64, 128]),
    ("c3", 16, 32, 700, [0, 300, 700]),                       # m = 16 per lane, ragged
]


@pytest.mark.parametrize("base,nx,ny,nz,kb", SLAB_CASES)
def test_poisson_z_slabs_match_oracle_and_single_plan(env, base, nx, ny, nz, kb):
    torch, pz, wl, oracle, ranks, sharded = env
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    got = solve_by_slabs(torch, pz, sharded, w, zc, zf, f, kb)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    assert rel_err(got, ref) <= TOL
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    p = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    one = p.cpu().numpy()
    pz.poisson_plan_destroy(plan)
    assert rel_err(got, one) <= 1e-12
    # the solution carries zero volume mean whatever the cut
    dzf = np.diff(zf)
    assert abs(np.dot(dzf, got.mean(axis=(1, 2)))) / dzf.sum() <= 1e-13 * np.abs(got).max()


@pytest.mark.parametrize("world", [1, 2, 4, 8])
def test_poisson_z_slabs_at_512_columns_even_split(env, world):
    """c2's grid in x, y and the bounds bench.py's strong-scaling mode uses (ranks.z_slab_bounds)."""
    torch, pz, wl, oracle, ranks, sharded = env
    w = wl.scaled(wl.CONFIGS["c2"], 512, 512, 64)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    kb = ranks.z_slab_bounds(w.nz, world)
    got = solve_by_slabs(torch, pz, sharded, w, zc, zf, f, kb)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    assert rel_err(got, ref) <= TOL


@pytest.mark.parametrize("base,nx,ny,nz,kb", [("c1", 32, 16, 48, [0, 24, 48]), ("c3", 64, 32, 100, [0, 3, 40, 45, 100]),
                                            ("c3", 16, 32, 700, [0, 300, 700]), ("c2", 512, 512, 64, [0, 8, 16, 24, 32, 40, 48, 56, 64])])
def test_poisson_z_slabs_with_the_exchange_done_by_the_kernels(env, base, nx, ny, nz, kb):
    """exchange = "p2p": every rank's reduction kernel stores its boundary block into every rank's
    gathered buffer and raises a flag; the finish waits on the flags on the device.  The ranks of the
    job live in this process (their buffers are ordinary device memory of this GPU); all pushes are
    enqueued before any wait, as on a node.  Three solves in a row alternate the two buffer sets."""
    torch, pz, wl, oracle, ranks, sharded = env
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    G = len(kb) - 1
    jobs = [sharded.SlabPoisson(nx, ny, nz, w.lx, w.ly, zc, zf, g, G, kb, exchange="p2p") for g in range(G)]
    sharded.SlabPoisson.connect(jobs)
    for it in range(3):
        f = wl.remove_weighted_mean(np.random.default_rng(100 + it).standard_normal((nz, ny, nx)), zf)
        parts = [torch.from_numpy(s).cuda() for s in sharded.split_z(f, kb)]
        for j, p in zip(jobs, parts):
            j.reduce(p)
        for j, p in zip(jobs, parts):
            j.finish(p)
        torch.cuda.synchronize()
        got = np.concatenate([p.cpu().numpy() for p in parts], axis=0)
        assert rel_err(got, oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)) <= TOL
    for j in jobs:
        j.destroy()


def test_slab_driver_single_rank_and_error_paths(env):
    torch, pz, wl, oracle, ranks, sharded = env
    w = wl.scaled(wl.CONFIGS["c1"], 32, 16, 40)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    job = sharded.SlabPoisson(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, 0, 1)
    p = torch.from_numpy(f).cuda()
    job.solve(p)          # reduce, gather (a copy without a process group), finish
    torch.cuda.synchronize()
    assert rel_err(p.cpu().numpy(), oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)) <= TOL
    assert job.bytes_exchanged_per_solve >= 2 * w.nx * w.ny * 8
    with pytest.raises(RuntimeError):
        pz.poisson_solve(job.plan, p)               # a slab plan solves through reduce / finish
    with pytest.raises(RuntimeError):
        pz.helmholtz_z_setup(job.plan, 1e-4)        # columns are cut
    job.destroy()
    with pytest.raises(RuntimeError):
        pz.poisson_slab_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, 2, 0, [0, 2, 40])   # 2 planes
    with pytest.raises(RuntimeError):
        pz.poisson_slab_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, 2, 0, [0, 20, 39])  # not to nz
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    with pytest.raises((RuntimeError, ValueError)):
        pz.poisson_solve_reduce(plan, p, p)          # not a slab plan
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("nx,ny,nz,world", [(64, 64, 48, 2), (32, 128, 100, 4), (128, 64, 512, 8), (64, 256, 1100, 2)])
def test_helmholtz_y_slabs_equal_the_unsharded_solve_bitwise(env, nx, ny, nz, world):
    torch, pz, wl, oracle, ranks, sharded = env
    w = wl.scaled(wl.CONFIGS["c4"], nx, ny, nz)
    zc, zf = wl.grid(w)
    rs = [wl.helmholtz_rhs(w, c) for c in range(3)]
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    pz.helmholtz_z_setup(plan, w.a)
    whole = [torch.from_numpy(r).cuda() for r in rs]
    pz.helmholtz_z_solve_n(plan, whole)
    torch.cuda.synchronize()
    whole = [u.cpu().numpy() for u in whole]
    pz.poisson_plan_destroy(plan)
    gathered = [np.empty_like(r) for r in rs]
    for rank in range(world):
        job = sharded.YSlabHelmholtz(nx, ny, nz, w.lx, w.ly, zc, zf, w.a, rank, world)
        mine = [torch.from_numpy(np.ascontiguousarray(r[:, job.j0:job.j1, :])).cuda() for r in rs]
        job.solve(mine)
        torch.cuda.synchronize()
        for out, u in zip(gathered, mine):
            out[:, job.j0:job.j1, :] = u.cpu().numpy()
        job.destroy()
    for c in range(3):
        assert np.array_equal(gathered[c], whole[c])
    assert rel_err(gathered[0], oracle.helmholtz_z_solve(zc, zf, w.a, rs[0])) <= TOL
