"""poisson_zsolve_noalloc (include/pz.h): step a3 with the library's static device workspace, for
callers that may not allocate.  Checked against the existing path -- pz_poisson_stage(PZ_STAGE_Z_SOLVE)
with zsolve_variant 0 (the same sweep with a cudaMalloc'ed workspace: equal bit for bit) and with the
plan's default variant (within the tolerance of the parity tests) -- on two calls in a row with
different inputs, a smaller problem after a larger one (the array keeps the previous call's
contents), a side stream, Dirichlet walls, and the size limit.

The file name sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def env():
    import torch

    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import workloads as wl

    assert torch.cuda.is_available()
    pz.lib()
    return torch, pz, wl


def rel_err(a, b):
    return float((a - b).abs().max() / b.abs().max())


def spectral_field(torch, plan_shape, seed, zf):
    """A field as the z stage sees it: any real array is a valid set of packed spectral coefficients;
    the (0,0) column gets zero weighted mean so that its singular system is solvable (reading R3)."""
    nz, ny, nx = plan_shape
    g = torch.Generator(device="cuda").manual_seed(seed)
    f = torch.randn(nz, ny, nx, dtype=torch.float64, device="cuda", generator=g)
    dzf = torch.from_numpy(np.diff(zf)).cuda()
    f[:, 0, 0] -= (dzf * f[:, 0, 0]).sum() / dzf.sum()
    return f


def existing_path(torch, pz, plan, f, variant=None):
    out = f.clone()
    if variant is not None:
        pz.pz_set_option(plan, "zsolve_variant", variant)
    pz.pz_poisson_stage(plan, out, pz.PZ_STAGE_Z_SOLVE)
    torch.cuda.synchronize()
    return out


@pytest.mark.parametrize("nx,ny,nz,beta,bc", [(64, 32, 48, 1.8, 0), (128, 64, 200, 2.0, 0), (32, 16, 1100, 1.8, 0), (48, 40, 33, 2.0, "DD")])
def test_two_calls_in_a_row_match_the_existing_path(env, nx, ny, nz, beta, bc):
    torch, pz, wl = env
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    code = pz.pz_bc("P", "P", bc) if bc else 0
    plan = pz.poisson_plan_create(nx, ny, nz, 4 * np.pi, 2 * np.pi, zc, zf, code)
    default_variant = pz.pz_get_option(plan, "zsolve_variant")
    inputs = [spectral_field(torch, (nz, ny, nx), seed, zf) for seed in (11, 12)]
    refs_default = [existing_path(torch, pz, plan, f) for f in inputs]
    refs_sweep = [existing_path(torch, pz, plan, f, 0) for f in inputs]
    pz.pz_set_option(plan, "zsolve_variant", default_variant)
    launches = pz.pz_launch_count()
    outs = []
    for f in inputs:                      # two calls in a row, nothing in between
        out = f.clone()
        pz.poisson_zsolve_noalloc(plan, out)
        outs.append(out)
    torch.cuda.synchronize()
    assert pz.pz_launch_count() == launches + 2
    for out, r0, rd in zip(outs, refs_sweep, refs_default):
        assert torch.equal(out, r0)       # the same kernel with another workspace
        assert rel_err(out, rd) <= TOL
    pz.poisson_plan_destroy(plan)


def test_smaller_problem_after_a_larger_one_and_a_side_stream(env):
    """The shared array keeps the larger call's contents; the smaller call must not see them."""
    torch, pz, wl = env
    big = (128, 128, 128)                 # exactly PZ_NOALLOC_MAX_POINTS
    small = (16, 16, 24)
    assert big[0] * big[1] * big[2] == pz.PZ_NOALLOC_MAX_POINTS
    res = {}
    side = torch.cuda.Stream()
    for shape, seed in ((big, 21), (small, 22), (big, 23)):
        nx, ny, nz = shape
        zf = wl.z_faces(nz, 2.0, 1.8)
        plan = pz.poisson_plan_create(nx, ny, nz, 2 * np.pi, 2 * np.pi, wl.z_centres(zf), zf)
        f = spectral_field(torch, (nz, ny, nx), seed, zf)
        ref = existing_path(torch, pz, plan, f)
        out = f.clone()
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            pz.poisson_zsolve_noalloc(plan, out, side)
        side.synchronize()
        res[seed] = rel_err(out, ref)
        pz.poisson_plan_destroy(plan)
    assert max(res.values()) <= TOL, res


def test_sizes_beyond_the_static_workspace_are_refused(env):
    torch, pz, wl = env
    nx, ny, nz = 256, 128, 128            # twice the limit
    zf = wl.z_faces(nz, 2.0, 1.8)
    plan = pz.poisson_plan_create(nx, ny, nz, 2 * np.pi, 2 * np.pi, wl.z_centres(zf), zf)
    f = torch.ones(nz, ny, nx, dtype=torch.float64, device="cuda")
    launches = pz.pz_launch_count()
    with pytest.raises(pz.PzError) as ei:
        pz.poisson_zsolve_noalloc(plan, f)
    assert ei.value.status == pz.PZ_EUNSUPPORTED
    assert "PZ_NOALLOC_MAX_POINTS" in str(ei.value)
    torch.cuda.synchronize()
    assert pz.pz_launch_count() == launches and bool((f == 1.0).all())   # nothing launched, field untouched
    pz.poisson_plan_destroy(plan)
