"""GPU parity of the mixed-radix (2, 3, 5, 7) transforms: the paper's in-house FFT is mixed-radix
 and all its grids have such lengths -- 7168 = 2^10 7, 3200 x 3456
(:278), 3456 x 3072 (:280).  Stage tests against numpy.fft (a library routine as an independent
check of lengths, radices and the packed layout), whole solves against the oracle's definition-level
variant (naive O(n^2) DFT, any length) element by element, bar 1e-11 as everywhere.
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
    from paper_2502_06296_b200 import workloads as wl

    assert torch.cuda.is_available()
    pz.lib()
    return torch, pz, wl, oracle


def rel_err(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


LENGTHS = [12, 24, 96, 120, 384, 896, 1536, 3072, 3200, 3456, 7168]


@pytest.mark.parametrize("nx,ny", [(n, 8) for n in LENGTHS] + [(8, n) for n in LENGTHS] +
                         [(12, 12), (20, 28), (96, 80), (120, 42), (14, 40), (8192, 8), (16, 8192), (360, 600)])
def test_mixed_radix_stages_against_numpy_fft(env, nx, ny):
    torch, pz, wl, oracle = env
    nz = 4
    w = wl.scaled(wl.CONFIGS["c0"], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = np.random.default_rng(nx * 7 + ny).standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    p = torch.from_numpy(f).cuda()
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_FWD)
    gx = p.cpu().numpy()
    X = np.fft.rfft(f, axis=2)
    sx = np.abs(X).max()
    assert np.abs(gx[:, :, 2::2] - X[:, :, 1:-1].real).max() <= 1e-12 * sx
    assert np.abs(gx[:, :, 3::2] - X[:, :, 1:-1].imag).max() <= 1e-12 * sx
    assert np.abs(gx[:, :, 0] - X[:, :, 0].real).max() <= 1e-12 * sx
    assert np.abs(gx[:, :, 1] - X[:, :, -1].real).max() <= 1e-12 * sx
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_FWD)
    g = p.cpu().numpy()
    F = np.fft.fft(X, axis=1)                       # [k][qy][qx], qx = 0..nx/2
    scale = np.abs(F).max()
    got = g[:, :, 2::2] + 1j * g[:, :, 3::2]        # complex pairs q = 1..nx/2-1: natural order in y
    assert np.abs(got - F[:, :, 1:-1]).max() <= 1e-12 * scale
    for col, q in ((0, 0), (1, nx // 2)):           # x-modes 0 and nx/2: packed order in y
        assert np.abs(g[:, 0, col] - F[:, 0, q].real).max() <= 1e-12 * scale
        assert np.abs(g[:, 1, col] - F[:, ny // 2, q].real).max() <= 1e-12 * scale
        assert np.abs(g[:, 2::2, col] - F[:, 1:ny // 2, q].real).max() <= 1e-12 * scale
        assert np.abs(g[:, 3::2, col] - F[:, 1:ny // 2, q].imag).max() <= 1e-12 * scale
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_INV)
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_INV)
    assert np.abs(p.cpu().numpy() - f).max() <= 1e-13 * np.abs(f).max()
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("base,nx,ny,nz", [("c1", 96, 80, 48), ("c3", 384, 120, 65), ("c0", 12, 12, 5), ("c1", 40, 56, 33),
                                           ("c3", 120, 64, 96), ("c1", 64, 42 * 2, 40), ("c2", 224, 96, 128)])
def test_mixed_radix_poisson_and_helmholtz3d_match_the_naive_dft_oracle(env, base, nx, ny, nz):
    torch, pz, wl, oracle = env
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    p = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    got = p.cpu().numpy()
    assert rel_err(got, oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 0)) <= TOL
    dzf = np.diff(zf)
    assert abs(np.dot(dzf, got.mean(axis=(1, 2)))) / dzf.sum() <= 1e-13 * np.abs(got).max()
    a = 3e-4
    pz.helmholtz3d_setup(plan, a)
    u = torch.from_numpy(f).cuda()
    pz.helmholtz3d_solve(plan, u)
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), oracle.helmholtz3d_solve(w.lx, w.ly, zc, zf, a, f, 0)) <= TOL
    # the wall-normal Helmholtz solve and the pressure-correction step do not care about the radices
    pz.helmholtz_z_setup(plan, a)
    r = torch.from_numpy(f).cuda()
    pz.helmholtz_z_solve(plan, r)
    torch.cuda.synchronize()
    assert rel_err(r.cpu().numpy(), oracle.helmholtz_z_solve(zc, zf, a, f)) <= TOL
    pz.poisson_plan_destroy(plan)


def test_mixed_radix_pressure_correction_is_divergence_free(env):
    torch, pz, wl, oracle = env
    from oracle import projection as proj

    w = wl.scaled(wl.CONFIGS["c1"], 96, 40, 33)
    zc, zf = wl.grid(w)
    rng = np.random.default_rng(5)
    u, v, ww = (rng.standard_normal((w.nz, w.ny, w.nx)) for _ in range(3))
    ww[-1] = 0.0
    pr = rng.standard_normal((w.nz, w.ny, w.nx))
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    du, dv, dw, dp = (torch.from_numpy(x).cuda() for x in (u, v, ww, pr))
    work = torch.empty_like(du)
    gdt = 2e-3
    pz.pz_pressure_correction(plan, du, dv, dw, dp, work, gdt)
    torch.cuda.synchronize()
    div0 = np.abs(proj.divergence(w.lx, w.ly, zf, u, v, ww)).max()
    div1 = np.abs(proj.divergence(w.lx, w.ly, zf, du.cpu().numpy(), dv.cpu().numpy(), dw.cpu().numpy())).max()
    assert div1 <= 1e-11 * div0
    pz.poisson_plan_destroy(plan)


def test_unsupported_lengths_are_refused(env):
    torch, pz, wl, oracle = env
    zf = wl.z_faces(8, 2.0, 0.0)
    zc = wl.z_centres(zf)
    for nx, ny in ((22, 8), (8, 26), (9, 8), (8, 9), (12, 10), (2 * 8192 + 2, 8)):   # prime 11 / 13, odd, nx ny % 16 != 0, too long
        with pytest.raises(RuntimeError):
            pz.poisson_plan_create(nx, ny, 8, 1.0, 1.0, zc, zf)
