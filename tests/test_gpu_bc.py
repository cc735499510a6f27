"""GPU parity of the Poisson solve with cosine / sine expansions in x, y and Dirichlet / mixed walls
in z (reading R17) against oracle/bc.py, element by element, 1e-11."""
import itertools

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def env():
    import torch

    from oracle import bc as obc
    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import workloads as wl

    assert torch.cuda.is_available()
    pz.lib()
    return torch, pz, wl, obc


def rel_err(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def solve(torch, pz, wl, obc, nx, ny, nz, beta, bcx, bcy, bcz, options=()):
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    lx, ly = 3.0, 2.0
    f = np.random.default_rng(nx + 3 * ny + 7 * nz).standard_normal((nz, ny, nx))
    if "D" not in bcx + bcy + bcz:
        f = wl.remove_weighted_mean(f, zf)
    plan = pz.poisson_plan_create(nx, ny, nz, lx, ly, zc, zf, pz.pz_bc(bcx, bcy, bcz))
    for k, v in options:
        pz.pz_set_option(plan, k, v)
    p = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    got = p.cpu().numpy()
    pz.poisson_plan_destroy(plan)
    return got, obc.poisson_solve(lx, ly, zc, zf, f, bcx, bcy, bcz), zf


@pytest.mark.parametrize("bcx,bcy,bcz", list(itertools.product("PND", "PND", ["NN", "DD", "ND", "DN"])))
def test_every_combination_on_a_small_stretched_grid(env, bcx, bcy, bcz):
    torch, pz, wl, obc = env
    got, ref, zf = solve(torch, pz, wl, obc, 24, 16, 20, 1.8, bcx, bcy, bcz)
    assert rel_err(got, ref) <= TOL
    if "D" not in bcx + bcy + bcz:
        dzf = np.diff(zf)
        assert abs(np.dot(dzf, got.mean(axis=(1, 2)))) <= 1e-13 * np.abs(got).max() * dzf.sum()


@pytest.mark.parametrize("nx,ny,nz,beta,bcx,bcy,bcz,options", [
    (64, 32, 48, 2.0, "N", "N", "NN", []),                      # cosines both ways, singular (0,0)
    (64, 64, 100, 1.8, "P", "N", "DD", []),                     # power-of-two x transform, cosine y
    (96, 40, 33, 1.8, "D", "P", "ND", []),                      # mixed radix, sine x, periodic y: all pairs converted
    (120, 56, 64, 2.0, "N", "D", "DN", [("zsolve_variant", 1)]),
    (32, 96, 300, 1.8, "P", "P", "DD", []),                     # only the walls differ: TMA pipeline, ragged
    (32, 32, 512, 1.8, "P", "P", "ND", []),
    (16, 16, 1100, 1.8, "N", "P", "DD", []),                    # beyond 1024 planes: thread-per-column sweep
    (256, 128, 40, 1.8, "D", "D", "NN", []),
])
def test_larger_shapes_and_kernel_variants(env, nx, ny, nz, beta, bcx, bcy, bcz, options):
    torch, pz, wl, obc = env
    got, ref, _ = solve(torch, pz, wl, obc, nx, ny, nz, beta, bcx, bcy, bcz, options)
    assert rel_err(got, ref) <= TOL


def test_calls_that_need_the_hot_path_conditions_refuse_other_plans(env):
    torch, pz, wl, obc = env
    zf = wl.z_faces(16, 2.0, 1.8)
    zc = wl.z_centres(zf)
    plan = pz.poisson_plan_create(16, 16, 16, 1.0, 1.0, zc, zf, pz.pz_bc("N", "P", "DD"))
    u = torch.zeros(16, 16, 16, dtype=torch.float64, device="cuda")
    pz.helmholtz3d_setup(plan, 1e-3)
    with pytest.raises(pz.PzError):
        pz.helmholtz3d_solve(plan, u)
    with pytest.raises(pz.PzError):
        pz.pz_divergence_rhs(plan, u, u, u, u.clone(), 1.0)
    pz.helmholtz_z_setup(plan, 1e-3)          # the wall-normal Helmholtz solve does not depend on bc
    pz.helmholtz_z_solve(plan, u)
    pz.poisson_plan_destroy(plan)
    with pytest.raises(pz.PzError):
        pz.poisson_plan_create(16, 16, 16, 1.0, 1.0, zc, zf, 3)     # bcx = 3 does not exist
    with pytest.raises(pz.PzError):
        pz.poisson_slab_plan_create(16, 16, 16, 1.0, 1.0, zc, zf, 2, 0, [0, 8, 16], pz.pz_bc("P", "P", "DD"))
