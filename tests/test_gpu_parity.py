"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star): max|gpu - oracle| / max|oracle| <= 1e-11.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def torch():
    import torch as t

    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def pz():
    from paper_2502_06296_b200 import binding

    binding.lib()  # fails loudly if the extension is missing
    return binding


@pytest.fixture(scope="module")
def wl():
    from paper_2502_06296_b200 import workloads

    return workloads


@pytest.fixture(scope="module")
def oracle():
    import oracle as o

    return o


def rel_err(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def gpu_poisson(torch, pz, w, zc, zf, f, options=()):
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    for k, v in options:
        pz.pz_set_option(plan, k, v)
    p = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    out = p.cpu().numpy()
    pz.poisson_plan_destroy(plan)
    return out


# ------------------------------------------------------------------------ Poisson

POISSON_SHAPES = [
    # (base config, nx, ny, nz)   small enough for the oracle in seconds, several tiles + ragged tails
    ("c0", 64, 64, 64),       # BASELINE config 0 itself
    ("c0", 8, 8, 4),          # minimum sizes
    ("c0", 16, 8, 5),
    ("c3", 64, 32, 30),       # the 30 planes per GPU of the paper's weak-scaling grid
    ("c1", 32, 16, 32),
    ("c1", 32, 64, 48),       # stretched, nz not a multiple of 32
    ("c1", 128, 32, 100),
    ("c1", 64, 128, 129),     # one row past a sub-domain multiple
    ("c3", 256, 64, 96),      # beta = 2.0, long x
    ("c3", 32, 256, 33),
    ("c3", 160, 24, 57),      # thread-per-column range (nz <= 64), ragged last CTA
    ("c2", 64, 64, 128),      # few-mode right-hand side
    ("c1", 16, 16, 1024),     # one shared-memory stage (m = 32)
    ("c3", 32, 16, 700),      # ragged, m = 32
    ("c1", 16, 32, 300),      # ragged, m = 16
]


@pytest.mark.parametrize("base,nx,ny,nz", POISSON_SHAPES)
@pytest.mark.parametrize("variant", [0, 1, 2, 4])
def test_poisson_matches_oracle(torch, pz, wl, oracle, base, nx, ny, nz, variant):
    if variant == 4 and nz > 64:
        pytest.skip("variant 4 keeps the column on chip per thread: nz <= 64")
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 0 if nx * ny <= 64 * 64 else 1)
    got = gpu_poisson(torch, pz, w, zc, zf, f, [("zsolve_variant", variant)])
    assert rel_err(got, ref) <= TOL
    dzf = np.diff(zf)
    wm = np.einsum("k,kji->", dzf, got) / (dzf.sum() * nx * ny)
    assert abs(wm) <= 1e-13 * np.abs(got).max()


LONG_COLUMNS = [("c1", 16, 16, 1100), ("c3", 32, 16, 1594), ("c1", 16, 8, 2048), ("c1", 8, 8, 2500), ("c3", 64, 32, 900), ("c1", 32, 16, 513),
                ("c3", 16, 16, 1024), ("c1", 48, 32, 3000), ("c1", 16, 16, 4096), ("c1", 8, 8, 4500)]


@pytest.mark.parametrize("base,nx,ny,nz", LONG_COLUMNS)
# 3: the plan's own z cut through the pipeline (default above 1024 planes); 2: whole columns, one stage (default up to 1024);
# 0: thread-per-column sweep
@pytest.mark.parametrize("variant", [3, 2, 0])
def test_poisson_beyond_512_planes_matches_oracle(torch, pz, wl, oracle, base, nx, ny, nz, variant):
    """Columns longer than the pipeline's three-stage tile (the paper's wall-normal sizes are 900 and 1594)."""
    if (variant == 2) != (nz <= 1024) and variant != 0:
        pytest.skip("variant not defined for this nz")
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    assert pz.pz_get_option(plan, "zsolve_variant") == (2 if nz <= 1024 else 3)
    pz.pz_set_option(plan, "zsolve_variant", variant)
    p = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    got = p.cpu().numpy()
    pz.poisson_plan_destroy(plan)
    assert rel_err(got, ref) <= TOL
    dzf = np.diff(zf)
    assert abs(np.einsum("k,kji->", dzf, got)) / (dzf.sum() * nx * ny) <= 1e-13 * np.abs(got).max()


@pytest.mark.parametrize("slab", [1, 3, 1000])
def test_poisson_slab_size_does_not_change_the_result(torch, pz, wl, slab):
    w = wl.scaled(wl.CONFIGS["c1"], 64, 32, 40)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    a = gpu_poisson(torch, pz, w, zc, zf, f, [("slab_planes", slab)])
    b = gpu_poisson(torch, pz, w, zc, zf, f, [])
    assert np.array_equal(a, b)  # bitwise: no atomics, same arithmetic per point


def test_poisson_is_bitwise_deterministic_and_plan_is_reusable(torch, pz, wl):
    w = wl.scaled(wl.CONFIGS["c1"], 64, 64, 64)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    outs = []
    for _ in range(3):
        p = torch.from_numpy(f).cuda()
        pz.poisson_solve(plan, p)
        outs.append(p.cpu().numpy())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_poisson_on_a_side_stream_and_graph_capture(torch, pz, wl):
    w = wl.scaled(wl.CONFIGS["c1"], 32, 32, 64)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    p0 = torch.from_numpy(f).cuda()
    pz.poisson_solve(plan, p0)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    p1 = torch.from_numpy(f).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        pz.poisson_solve(plan, p1)
    s.synchronize()
    assert torch.equal(p0, p1)
    # CUDA graph: no allocation, no host sync inside the solve
    static = torch.from_numpy(f).cuda()
    g = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(g):
        pz.poisson_solve(plan, static)
    static.copy_(torch.from_numpy(f))
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(static, p0)


def test_poisson_stages_against_oracle_dft(torch, pz, wl, oracle):
    """Stage a1+a2 produce the 2-D DFT of every plane (in the packed spectral layout)."""
    from oracle import algorithms as alg

    w = wl.scaled(wl.CONFIGS["c1"], 32, 16, 6)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    p = torch.from_numpy(f).cuda()
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_FWD)
    gx = p.cpu().numpy()
    X = np.fft.rfft(f, axis=2)
    for k in range(w.nz):
        for j in range(w.ny):
            assert np.abs(alg.unpack_halfcomplex(gx[k, j])[1:-1] - X[k, j, 1:-1]).max() <= 1e-12 * np.abs(X).max()
            assert abs(gx[k, j, 0] - X[k, j, 0].real) <= 1e-12 * np.abs(X).max()
            assert abs(gx[k, j, 1] - X[k, j, -1].real) <= 1e-12 * np.abs(X).max()
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_FWD)
    gy = p.cpu().numpy()
    F = oracle.dft_xy(f, -1, 0)                      # full complex 2-D DFT, [k][qy][qx]
    scale = np.abs(F).max()
    nxh = w.nx // 2
    for q in range(1, nxh):                          # complex pairs: natural order in y
        got = gy[:, :, 2 * q] + 1j * gy[:, :, 2 * q + 1]
        assert np.abs(got - F[:, :, q]).max() <= 1e-12 * scale
    for col, q in ((0, 0), (1, nxh)):                # x-modes 0 and nx/2: packed order in y
        for k in range(w.nz):
            got = alg.unpack_halfcomplex(gy[k, :, col])
            assert np.abs(got - F[k, : w.ny // 2 + 1, q]).max() <= 1e-12 * scale
    # inverse stages undo the forward ones (up to the 1/(nx ny) applied in a5)
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_INV)
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_INV)
    back = p.cpu().numpy()
    assert np.abs(back - f).max() <= 1e-13 * np.abs(f).max()


@pytest.mark.parametrize("nx,ny", [(8, 8), (16, 8), (8, 32), (64, 16), (128, 64), (256, 128), (512, 256),
                                   (1024, 8), (8, 1024), (2048, 16), (16, 2048), (4096, 8), (8, 4096)])
def test_fft_roundtrip_and_spectrum_every_size(torch, pz, wl, nx, ny):
    """Every supported transform length: forward stages against numpy.fft (library routine as
    an independent check of the layout), then the inverse stages return the input."""
    nz = 4
    w = wl.scaled(wl.CONFIGS["c0"], nx, ny, nz)
    zc, zf = wl.grid(w)
    rng = np.random.default_rng(nx + ny)
    f = rng.standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    p = torch.from_numpy(f).cuda()
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_FWD)
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_FWD)
    g = p.cpu().numpy()
    F = np.fft.fft(np.fft.rfft(f, axis=2), axis=1)   # [k][qy][qx], qx = 0..nx/2
    scale = np.abs(F).max()
    for q in range(1, nx // 2):
        got = g[:, :, 2 * q] + 1j * g[:, :, 2 * q + 1]
        assert np.abs(got - F[:, :, q]).max() <= 1e-12 * scale, q
    assert np.abs(g[:, 0, 0] - F[:, 0, 0].real).max() <= 1e-12 * scale
    assert np.abs(g[:, 1, 1] - F[:, ny // 2, nx // 2].real).max() <= 1e-12 * scale
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_Y_INV)
    pz.pz_poisson_stage(plan, p, pz.PZ_STAGE_FFT_X_INV)
    assert np.abs(p.cpu().numpy() - f).max() <= 1e-13 * np.abs(f).max()


@pytest.mark.parametrize("nx,ny,nz,lag", [(256, 256, 5, 0), (512, 256, 4, 0), (256, 512, 40, 0), (256, 256, 40, 1),
                                          (256, 256, 40, 3), (1024, 256, 4, 0), (256, 1024, 4, 0), (2048, 256, 4, 0),
                                          (512, 512, 70, 0), (512, 512, 70, 2), (1024, 512, 9, 0), (2048, 1024, 5, 0)])
def test_fused_xy_transform_equals_the_separate_kernels(torch, pz, wl, nx, ny, nz, lag):
    """The fused x/y kernel (two-pass 32-point items fed by TMA, plane handed from phase one to
    phase two through L2, per-phase ticket counters) computes the same packed spectrum as the
    separate kernels (another factorisation of the same transforms: equal to rounding, and bitwise
    equal from one call to the next) and the same round trip."""
    w = wl.scaled(wl.CONFIGS["c0"], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = np.random.default_rng(nx + 3 * ny + nz).standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    pz.pz_set_option(plan, "xy_lag", lag)
    a = torch.from_numpy(f).cuda()
    b = torch.from_numpy(f).cuda()
    pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_X_FWD)
    pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_Y_FWD)
    first = None
    for _ in range(3):  # repeated: the counters are reset per call, the result does not depend on the item order
        b.copy_(torch.from_numpy(f))
        pz.pz_poisson_stage(plan, b, pz.PZ_STAGE_FFT_XY_FWD)
        assert float((a - b).abs().max()) <= 1e-13 * float(a.abs().max())
        if first is None:
            first = b.clone()
        assert torch.equal(first, b)
    # independent check of the fused spectrum against a library transform
    g = b.cpu().numpy()
    F = np.fft.fft(np.fft.rfft(f, axis=2), axis=1)   # [k][qy][qx], qx = 0..nx/2
    scale = np.abs(F).max()
    for q in (1, 2, nx // 4, nx // 2 - 1):
        got = g[:, :, 2 * q] + 1j * g[:, :, 2 * q + 1]
        assert np.abs(got - F[:, :, q]).max() <= 1e-12 * scale, q
    assert np.abs(g[:, 0, 0] - F[:, 0, 0].real).max() <= 1e-12 * scale
    assert np.abs(g[:, 1, 1] - F[:, ny // 2, nx // 2].real).max() <= 1e-12 * scale
    pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_Y_INV)
    pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_X_INV)
    pz.pz_poisson_stage(plan, b, pz.PZ_STAGE_FFT_XY_INV)
    assert float((a - b).abs().max()) <= 1e-13 * float(a.abs().max())
    assert np.abs(b.cpu().numpy() - f).max() <= 1e-13 * np.abs(f).max()
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("nx,ny,nz", [(8, 8, 4), (16, 32, 5), (64, 16, 6), (128, 512, 4), (32, 1024, 4), (8, 4096, 4)])
def test_pair0_conversion_inside_the_y_kernel_equals_the_separate_kernel(torch, pz, wl, nx, ny, nz):
    w = wl.scaled(wl.CONFIGS["c0"], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = np.random.default_rng(nx + ny).standard_normal((nz, ny, nx))
    outs = []
    for p0 in (0, 1):
        plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
        pz.pz_set_option(plan, "fft_y_p0", p0)
        a = torch.from_numpy(f).cuda()
        pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_X_FWD)
        pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_Y_FWD)
        spec = a.clone()
        pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_Y_INV)
        pz.pz_poisson_stage(plan, a, pz.PZ_STAGE_FFT_X_INV)
        outs.append((spec, a))
        pz.poisson_plan_destroy(plan)
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])


def test_poisson_fused_and_separate_transforms_agree_with_the_oracle(torch, pz, wl, oracle):
    w = wl.scaled(wl.CONFIGS["c3"], 512, 256, 48)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    fused = gpu_poisson(torch, pz, w, zc, zf, f, [("fft_fused", 1)])
    separate = gpu_poisson(torch, pz, w, zc, zf, f, [("fft_fused", 0)])
    assert rel_err(fused, ref) <= TOL and rel_err(separate, ref) <= TOL
    assert rel_err(fused, separate) <= 1e-12


# ---------------------------------------------------------------------- Helmholtz

HELM_CASES = [
    # (nx, ny, nz, beta, a, options)
    (8, 8, 4, 0.0, 0.1, []),
    (16, 8, 7, 1.8, 5e-5, []),
    (32, 16, 64, 1.8, 5e-5, []),
    (32, 16, 100, 1.8, 5e-5, []),
    (64, 8, 129, 2.0, 2.5e-5, []),
    (16, 16, 256, 1.8, 5e-5, []),
    (16, 16, 256, 1.8, 1e-2, [("helm_m", 4)]),
    (16, 16, 256, 1.8, 5e-5, [("helm_m", 16), ("helm_tx", 8)]),
    (8, 16, 512, 1.8, 5e-5, []),
    (8, 16, 512, 1.8, 5e-5, [("helm_tx", 32)]),
    (8, 8, 1024, 1.8, 2.5e-5, []),
    (8, 8, 1024, 1.8, 2.5e-5, [("helm_m", 16), ("helm_tx", 8)]),
    (8, 8, 1594, 1.8, 2.5e-5, []),       # the paper's nz
    (8, 8, 64, 0.0, 0.0, []),            # a = 0: identity
    (8, 8, 64, 1.8, 10.0, []),           # strongly implicit
    (256, 128, 300, 1.8, 5e-5, []),      # 2048 tiles of 16 columns: several per resident CTA; 2 TMA boxes
    (64, 32, 513, 1.8, 5e-5, []),        # column cut over the two CTAs of a cluster; padding rows in the second chunk
    (64, 32, 700, 2.0, 5e-5, []),
    (64, 32, 1024, 1.8, 2.5e-5, []),     # cut column, 32-column tiles, no padding
    (64, 32, 1024, 1.8, 2.5e-5, [("helm_zsplit", 1)]),   # whole columns per CTA
    (8, 8, 1024, 1.8, 10.0, []),         # strongly implicit across the cut
    (64, 32, 1024, 1.8, 2.5e-5, [("helm_zsplit", 4)]),                   # four chunks per column
    (64, 32, 512, 1.8, 10.0, [("helm_zsplit", 4)]),                      # strongly implicit across three cuts
    (64, 32, 512, 1.8, 5e-5, [("helm_zsplit", 4), ("helm_tx", 64)]),     # 64-column tiles
    (64, 32, 700, 2.0, 5e-5, [("helm_zsplit", 4)]),                      # padding rows in the last chunk
    (12, 12, 300, 1.8, 5e-5, [("helm_zsplit", 4)]),                      # 16-column tiles
    (64, 32, 1594, 1.8, 2.5e-5, [("helm_zsplit", 4)]),
    (12, 12, 600, 1.8, 5e-5, []),        # cut column, 16-column tiles (144 columns)
    (64, 32, 1594, 1.8, 2.5e-5, []),     # the paper's nz on the pipeline: 50 sub-domains per chunk
    (16, 8, 1920, 1.8, 2.5e-5, []),      # largest nz of the pipeline
    (16, 8, 2048, 1.8, 2.5e-5, []),      # beyond: four chunks per column
    (16, 8, 3000, 1.8, 2.5e-5, []),
    (16, 8, 3584, 1.8, 2.5e-5, []),      # largest nz of the pipeline
    (128, 64, 48, 1.8, 5e-5, []),
]


@pytest.mark.parametrize("nx,ny,nz,beta,a,options", HELM_CASES)
@pytest.mark.parametrize("variant", [0, 1])   # 0: register tile, direct loads; 1: persistent TMA pipeline
def test_helmholtz_matches_oracle(torch, pz, wl, oracle, nx, ny, nz, beta, a, options, variant):
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    rng = np.random.default_rng(nz * 7 + nx)
    r = rng.standard_normal((nz, ny, nx))
    ref = oracle.helmholtz_z_solve(zc, zf, a, r)
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    pz.pz_set_option(plan, "helm_variant", variant)
    for k, v in options:
        pz.pz_set_option(plan, k, v)
    pz.helmholtz_z_setup(plan, a)
    whole = ("helm_zsplit", 1) in options
    expect = variant if nz <= (1024 if whole else 3584) else 0
    if nz > 2048:
        expect = 1                                   # the register-tile kernel stops at 2048 planes
    assert pz.pz_get_option(plan, "helm_variant_actual") == expect
    u = torch.from_numpy(r).cuda()
    pz.helmholtz_z_solve(plan, u)
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), ref) <= TOL
    if a == 0.0:
        assert np.array_equal(u.cpu().numpy(), r)


@pytest.mark.parametrize("nx,ny,nz,beta,a", [(8, 8, 4, 0.0, 0.1), (32, 16, 100, 1.8, 5e-5), (16, 16, 256, 2.0, 1e-3),
                                             (64, 32, 512, 1.8, 5e-5), (64, 32, 700, 1.8, 5e-5), (16, 8, 1024, 1.8, 10.0),
                                             (16, 8, 1594, 1.8, 2.5e-5), (8, 8, 2048, 1.8, 2.5e-5), (8, 8, 3200, 1.8, 2.5e-5)])
def test_helmholtz_w_face_centred_matches_oracle(torch, pz, wl, oracle, nx, ny, nz, beta, a):
    """The wall-normal component on the z faces (reading R16) through every kernel variant the size
    selects, beside a cell-centred set-up with another coefficient on the same plan."""
    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    rng = np.random.default_rng(nz + 3 * nx)
    r = rng.standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    w = torch.from_numpy(r).cuda()
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz_w_solve(plan, w)
    assert ei.value.status == pz.PZ_ENOTSETUP
    pz.helmholtz_z_setup(plan, 3 * a)
    pz.helmholtz_w_setup(plan, a)
    u = torch.from_numpy(r).cuda()
    pz.helmholtz_w_solve(plan, w)
    pz.helmholtz_z_solve(plan, u)
    torch.cuda.synchronize()
    assert rel_err(w.cpu().numpy(), oracle.helmholtz_w_solve(zc, zf, a, r)) <= TOL
    assert rel_err(u.cpu().numpy(), oracle.helmholtz_z_solve(zc, zf, 3 * a, r)) <= TOL
    assert torch.equal(w[-1], torch.from_numpy(r[-1]).cuda())       # the top wall face keeps its value
    pz.helmholtz_w_setup(plan, 2 * a)                                 # re-set-up, cell-centred tables untouched
    w2, u2 = torch.from_numpy(r).cuda(), torch.from_numpy(r).cuda()
    pz.helmholtz_w_solve(plan, w2)
    pz.helmholtz_z_solve(plan, u2)
    torch.cuda.synchronize()
    assert rel_err(w2.cpu().numpy(), oracle.helmholtz_w_solve(zc, zf, 2 * a, r)) <= TOL
    assert torch.equal(u2, u)
    pz.poisson_plan_destroy(plan)


def test_helmholtz_beyond_3584_planes_is_refused(torch, pz, wl):
    zf = wl.z_faces(4000, 2.0, 1.8)
    plan = pz.poisson_plan_create(8, 8, 4000, 1.0, 1.0, wl.z_centres(zf), zf)
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz_z_setup(plan, 1e-4)
    assert ei.value.status == pz.PZ_EUNSUPPORTED
    pz.poisson_plan_destroy(plan)


def test_helmholtz_not_setup_and_resetup(torch, pz, wl, oracle):
    nx, ny, nz = 16, 16, 96
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    r = np.random.default_rng(1).standard_normal((nz, ny, nx))
    u = torch.from_numpy(r).cuda()
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz_z_solve(plan, u)
    assert ei.value.status == pz.PZ_ENOTSETUP
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz_z_setup(plan, -1.0)
    assert ei.value.status == pz.PZ_EINVAL
    # a changes every Runge-Kutta sub-step: re-setup between solves, no sync
    fields, refs = [], []
    for a in (8 / 15 * 5e-5, 2 / 15 * 5e-5, 1 / 3 * 5e-5, 1e-3):
        pz.helmholtz_z_setup(plan, a)
        v = torch.from_numpy(r).cuda()
        pz.helmholtz_z_solve(plan, v)
        fields.append(v)
        refs.append(oracle.helmholtz_z_solve(zc, zf, a, r))
    torch.cuda.synchronize()
    for v, ref in zip(fields, refs):
        assert rel_err(v.cpu().numpy(), ref) <= TOL
    # three components in one call
    pz.helmholtz_z_setup(plan, 5e-5)
    comps = [torch.from_numpy(r * (c + 1)).cuda() for c in range(3)]
    pz.helmholtz_z_solve_n(plan, comps)
    torch.cuda.synchronize()
    ref = oracle.helmholtz_z_solve(zc, zf, 5e-5, r)
    for c, v in enumerate(comps):
        assert rel_err(v.cpu().numpy(), ref * (c + 1)) <= TOL


def test_helmholtz_graph_capture_and_determinism(torch, pz, wl):
    """helmholtz_z_solve_n (TMA pipeline, cluster launch) inside a CUDA graph: no allocation, no
    host synchronisation; replays are bitwise equal to the eager solve."""
    nx, ny, nz = 64, 32, 512
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    pz.helmholtz_z_setup(plan, 5e-5)
    r = [np.random.default_rng(20 + c).standard_normal((nz, ny, nx)) for c in range(3)]
    eager = [torch.from_numpy(x).cuda() for x in r]
    pz.helmholtz_z_solve_n(plan, eager)
    torch.cuda.synchronize()
    static = [torch.from_numpy(x).cuda() for x in r]
    g = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(g):
        pz.helmholtz_z_solve_n(plan, static)
    for _ in range(2):
        for t, x in zip(static, r):
            t.copy_(torch.from_numpy(x))
        g.replay()
        torch.cuda.synchronize()
        for a, b in zip(static, eager):
            assert torch.equal(a, b)
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("nz,variant", [(512, 1), (96, 1), (1100, 0)])
def test_helmholtz_graph_replay_survives_later_setups(torch, pz, wl, oracle, nz, variant):
    """A captured helmholtz_z_solve keeps the coefficient tables of capture time: set-ups made after
    the capture (one per Runge-Kutta sub-step) go to other table sets, so a replay is
    still ordered correctly and solves with the captured coefficient, whatever was set up since; the
    step of Eq. (11) in one kernel likewise.  Eager solves use the newest set-up."""
    nx, ny = 32, 16
    zf = wl.z_faces(nz, 2.0, 1.8)
    zc = wl.z_centres(zf)
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    pz.pz_set_option(plan, "helm_variant", variant)
    a1, a2, a3 = 5e-5, 3e-4, 1e-3
    r = np.random.default_rng(77).standard_normal((nz, ny, nx))
    uk = np.random.default_rng(78).standard_normal((nz, ny, nx))
    ref1 = oracle.helmholtz_z_solve(zc, zf, a1, r)
    pz.helmholtz_z_setup(plan, a1)
    static, ukd, step = torch.from_numpy(r).cuda(), torch.from_numpy(uk).cuda(), torch.from_numpy(r).cuda()
    g = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(g):
        pz.helmholtz_z_solve(plan, static)
        pz.helmholtz_z_step(plan, step, ukd)
    g.replay()
    torch.cuda.synchronize()
    first, first_step = static.clone(), step.clone()
    assert rel_err(first.cpu().numpy(), ref1) <= TOL
    for a in (a2, a3, a2, a3, a1 * 7):          # more set-ups than there are spare table sets
        pz.helmholtz_z_setup(plan, a)
        static.copy_(torch.from_numpy(r))
        step.copy_(torch.from_numpy(r))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(static, first) and torch.equal(step, first_step)
    eager = torch.from_numpy(r).cuda()
    pz.helmholtz_z_solve(plan, eager)
    torch.cuda.synchronize()
    assert rel_err(eager.cpu().numpy(), oracle.helmholtz_z_solve(zc, zf, a1 * 7, r)) <= TOL
    pz.poisson_plan_destroy(plan)


def test_host_buffer_entry_points(torch, pz, wl, oracle):
    w = wl.scaled(wl.CONFIGS["c1"], 32, 32, 48)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    host = torch.from_numpy(f.copy()).pin_memory()
    pz.poisson_solve_host(plan, host)
    torch.cuda.synchronize()
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    assert rel_err(host.numpy(), ref) <= TOL
    r = wl.helmholtz_rhs(w)
    pz.helmholtz_z_setup(plan, w.a)
    hb = torch.from_numpy(r.copy()).pin_memory()
    pz.helmholtz_z_solve_host(plan, hb)
    torch.cuda.synchronize()
    assert rel_err(hb.numpy(), oracle.helmholtz_z_solve(zc, zf, w.a, r)) <= TOL


# ------------------------------------------- fully implicit (3-D) Helmholtz, Eq. (8)

H3_CASES = [
    # (base config, nx, ny, nz, a)
    ("c0", 8, 8, 4, 0.1),
    ("c0", 64, 64, 64, 5e-5),
    ("c1", 32, 64, 48, 5e-5),
    ("c1", 128, 32, 100, 1e-2),
    ("c1", 64, 128, 129, 5e-5),
    ("c3", 256, 64, 96, 2.5e-5),
    ("c3", 32, 256, 33, 1.0),
    ("c2", 64, 64, 512, 5e-5),
    ("c1", 16, 16, 1024, 2.5e-5),
]


@pytest.mark.parametrize("base,nx,ny,nz,a", [("c1", 16, 16, 1100, 2.5e-5), ("c3", 32, 16, 1594, 1e-3), ("c1", 16, 8, 40, 5e-5)])
def test_helmholtz3d_through_the_thread_per_column_sweep(torch, pz, wl, oracle, base, nx, ny, nz, a):
    """Above 1024 planes (and with zsolve_variant 0) the Eq. (8) systems take the sweep of pz_zsolve.cu."""
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    r = np.random.default_rng(nx + nz).standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    if nz <= 1024:
        pz.pz_set_option(plan, "zsolve_variant", 0)
    pz.helmholtz3d_setup(plan, a)
    u = torch.from_numpy(r).cuda()
    pz.helmholtz3d_solve(plan, u)
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), oracle.helmholtz3d_solve(w.lx, w.ly, zc, zf, a, r, 1)) <= TOL
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("base,nx,ny,nz,a", H3_CASES)
@pytest.mark.parametrize("variant", [1, 2])
def test_helmholtz3d_matches_oracle(torch, pz, wl, oracle, base, nx, ny, nz, a, variant):
    w = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w)
    r = np.random.default_rng(nx + 5 * ny + 11 * nz).standard_normal((nz, ny, nx))
    ref = oracle.helmholtz3d_solve(w.lx, w.ly, zc, zf, a, r, 0 if nx * ny <= 64 * 64 else 1)
    plan = pz.poisson_plan_create(nx, ny, nz, w.lx, w.ly, zc, zf)
    pz.pz_set_option(plan, "zsolve_variant", variant)
    u = torch.from_numpy(r).cuda()
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz3d_solve(plan, u)
    assert ei.value.status == pz.PZ_ENOTSETUP
    pz.helmholtz3d_setup(plan, a)
    pz.helmholtz3d_solve(plan, u)
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), ref) <= TOL
    # a second a on the same plan (a changes every Runge-Kutta sub-step), and a = 0 is the identity
    pz.helmholtz3d_setup(plan, 2 * a)
    v = torch.from_numpy(r).cuda()
    pz.helmholtz3d_solve(plan, v)
    assert rel_err(v.cpu().numpy(), oracle.helmholtz3d_solve(w.lx, w.ly, zc, zf, 2 * a, r, 1)) <= TOL
    pz.helmholtz3d_setup(plan, 0.0)
    v = torch.from_numpy(r).cuda()
    pz.helmholtz3d_solve(plan, v)
    assert rel_err(v.cpu().numpy(), r) <= 1e-13
    pz.poisson_plan_destroy(plan)


def test_helmholtz3d_config1_full_and_fused_transforms(torch, pz, wl, oracle):
    w = wl.CONFIGS["c1"]
    zc, zf = wl.grid(w)
    r = wl.helmholtz_rhs(w)
    ref = oracle.helmholtz3d_solve(w.lx, w.ly, zc, zf, w.a, r, 1)
    outs = []
    for fused in (0, 1):
        plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
        pz.pz_set_option(plan, "fft_fused", fused)
        pz.helmholtz3d_setup(plan, w.a)
        u = torch.from_numpy(r).cuda()
        pz.helmholtz3d_solve(plan, u)
        outs.append(u.cpu().numpy())
        pz.poisson_plan_destroy(plan)
    assert rel_err(outs[0], ref) <= TOL and rel_err(outs[1], ref) <= TOL
    assert rel_err(outs[0], outs[1]) <= 1e-12


# --------------------------------- the steps either side of the Poisson solve, Eqs. (4)-(6)

@pytest.mark.parametrize("base,nx,ny,nz", [("c0", 8, 8, 4), ("c1", 32, 16, 48), ("c3", 64, 32, 33), ("c1", 128, 64, 96)])
def test_divergence_rhs_and_projection_match_oracle(torch, pz, wl, oracle, base, nx, ny, nz):
    from oracle import projection as proj

    w_ = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w_)
    rng = np.random.default_rng(nx + 3 * nz)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    w[-1] = 0.0
    p, phi = rng.standard_normal((nz, ny, nx)), rng.standard_normal((nz, ny, nx))
    gdt = 2.5e-3
    plan = pz.poisson_plan_create(nx, ny, nz, w_.lx, w_.ly, zc, zf)
    du, dv, dw, dp, dphi = (torch.from_numpy(a).cuda() for a in (u, v, w, p, phi))
    rhs = torch.empty_like(du)
    pz.pz_divergence_rhs(plan, du, dv, dw, rhs, 1.0 / gdt)
    ref = proj.divergence_rhs(w_.lx, w_.ly, zf, u, v, w, 1.0 / gdt)
    scale = (np.abs(u).max() / (w_.lx / nx) + np.abs(v).max() / (w_.ly / ny) + np.abs(w).max() / np.diff(zf).min()) / gdt
    assert np.abs(rhs.cpu().numpy() - ref).max() <= 1e-14 * scale       # cancellation-aware bound
    pz.pz_project(plan, du, dv, dw, dp, dphi, gdt)
    ru, rv, rw, rp = proj.project(w_.lx, w_.ly, zc, u, v, w, p, phi, gdt)
    for got, want in ((du, ru), (dv, rv), (dw, rw), (dp, rp)):
        assert rel_err(got.cpu().numpy(), want) <= 1e-13
    assert torch.equal(dw[-1], torch.from_numpy(w[-1]).cuda())          # top wall face untouched
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("base,nx,ny,nz", [("c0", 64, 64, 64), ("c1", 64, 32, 96), ("c3", 128, 64, 129)])
def test_pressure_correction_step_is_divergence_free_and_matches_oracle(torch, pz, wl, oracle, base, nx, ny, nz):
    from oracle import projection as proj

    w_ = wl.scaled(wl.CONFIGS[base], nx, ny, nz)
    zc, zf = wl.grid(w_)
    rng = np.random.default_rng(7 * nx + nz)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    w[-1] = 0.0
    p = rng.standard_normal((nz, ny, nx))
    gdt = 1e-3
    plan = pz.poisson_plan_create(nx, ny, nz, w_.lx, w_.ly, zc, zf)
    du, dv, dw, dp = (torch.from_numpy(a).cuda() for a in (u, v, w, p))
    work = torch.empty_like(du)
    pz.pz_pressure_correction(plan, du, dv, dw, dp, work, gdt)
    torch.cuda.synchronize()
    gu, gv, gw, gp = (t.cpu().numpy() for t in (du, dv, dw, dp))
    div0 = np.abs(proj.divergence(w_.lx, w_.ly, zf, u, v, w)).max()
    assert np.abs(proj.divergence(w_.lx, w_.ly, zf, gu, gv, gw)).max() <= 1e-11 * div0
    # the oracle's own step
    phi = oracle.poisson_solve(w_.lx, w_.ly, zc, zf, proj.divergence_rhs(w_.lx, w_.ly, zf, u, v, w, 1.0 / gdt), 1)
    assert rel_err(work.cpu().numpy(), phi) <= TOL
    ru, rv, rw, rp = proj.project(w_.lx, w_.ly, zc, u, v, w, p, phi, gdt)
    for got, want in ((gu, ru), (gv, rv), (gw, rw), (gp, rp)):
        assert rel_err(got, want) <= TOL
    # the divergence formed inside the forward x transform (default) and as a separate pass: bitwise equal
    pz.pz_set_option(plan, "div_fused", 0)
    eu, ev, ew, ep = (torch.from_numpy(a).cuda() for a in (u, v, w, p))
    work2 = torch.empty_like(eu)
    pz.pz_pressure_correction(plan, eu, ev, ew, ep, work2, gdt)
    torch.cuda.synchronize()
    assert torch.equal(work, work2) and torch.equal(du, eu) and torch.equal(dw, ew) and torch.equal(dp, ep)
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("nx,ny,nz,beta,a", [(8, 8, 4, 0.0, 0.1), (32, 16, 100, 1.8, 5e-5), (64, 32, 512, 1.8, 5e-5),
                                            (16, 16, 1100, 2.0, 2.5e-5), (32, 16, 1024, 1.8, 2.5e-5), (16, 16, 700, 1.8, 2.5e-5)])
def test_helmholtz_z_rhs_and_step_match_oracle(torch, pz, wl, oracle, nx, ny, nz, beta, a):
    """Eq. (11) whole: r = u** - a L_z u^k (helmholtz_z_rhs), then the solve (helmholtz_z_step)."""
    from oracle import projection as proj

    zf = wl.z_faces(nz, 2.0, beta)
    zc = wl.z_centres(zf)
    rng = np.random.default_rng(nz + nx)
    u2, uk = rng.standard_normal((nz, ny, nx)), rng.standard_normal((nz, ny, nx))
    plan = pz.poisson_plan_create(nx, ny, nz, 1.0, 1.0, zc, zf)
    d2, dk = torch.from_numpy(u2).cuda(), torch.from_numpy(uk).cuda()
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz_z_rhs(plan, d2, dk)
    assert ei.value.status == pz.PZ_ENOTSETUP
    pz.helmholtz_z_setup(plan, a)
    pz.helmholtz_z_rhs(plan, d2, dk)
    ref_r = proj.helmholtz_z_rhs(zc, zf, a, u2, uk)
    bound = np.abs(u2).max() + 4 * a * np.abs(uk).max() / (np.diff(zf).min() * np.diff(zc).min())
    assert np.abs(d2.cpu().numpy() - ref_r).max() <= 1e-14 * bound     # cancellation-aware bound
    ref_u = oracle.helmholtz_z_solve(zc, zf, a, ref_r)
    for fused in (1, 2, 0):   # formed inside the solve kernel (u^k through shared memory where two tiles fit; 2: u^k from global memory) / separate pass
        pz.pz_set_option(plan, "step_fused", fused)
        e2 = torch.from_numpy(u2).cuda()
        pz.helmholtz_z_step(plan, e2, dk)
        torch.cuda.synchronize()
        assert rel_err(e2.cpu().numpy(), ref_u) <= TOL
    assert torch.equal(dk, torch.from_numpy(uk).cuda())                 # u^k is only read
    pz.poisson_plan_destroy(plan)


def test_error_paths_of_the_widened_entry_points(torch, pz, wl):
    zf = wl.z_faces(1100, 2.0, 1.8)
    plan = pz.poisson_plan_create(16, 16, 1100, 1.0, 1.0, wl.z_centres(zf), zf)
    assert pz.pz_get_option(plan, "zsolve_variant") == 3          # the plan's own z cut above nz = 1024
    with pytest.raises(pz.PzError) as ei:
        pz.helmholtz3d_setup(plan, -1e-3)
    assert ei.value.status == pz.PZ_EINVAL
    pz.helmholtz3d_setup(plan, 1e-3)
    u = torch.zeros(1100, 16, 16, dtype=torch.float64, device="cuda")
    pz.helmholtz3d_solve(plan, u)                                  # above 1024 planes: thread-per-column sweep
    with pytest.raises(pz.PzError) as ei:
        pz.pz_set_option(plan, "zsolve_variant", 2)
    assert ei.value.status == pz.PZ_EUNSUPPORTED
    h = torch.zeros(1100 * 256, dtype=torch.float64).pin_memory()
    with pytest.raises(pz.PzError) as ei:
        pz.pz_solve_host_batch(plan, None, [h])                    # Helmholtz field before helmholtz_z_setup
    assert ei.value.status == pz.PZ_ENOTSETUP
    pz.pz_solve_host_batch(plan, None, [])                         # nothing to do
    with pytest.raises(pz.PzError) as ei:
        pz.pz_set_option(plan, "no_such_option", 1)
    assert ei.value.status == pz.PZ_EUNSUPPORTED
    pz.poisson_plan_destroy(plan)


@pytest.mark.parametrize("nx,ny,nz", [(64, 32, 48), (24, 20, 33), (128, 64, 300)])
def test_host_batch_pipeline(torch, pz, wl, oracle, nx, ny, nz):
    """pz_solve_host_batch: Poisson + several Helmholtz fields on pinned host buffers, more fields
    than staging buffers, twice in a row on a side stream."""
    w = wl.scaled(wl.CONFIGS["c1"], nx, ny, nz)
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    rs = [np.random.default_rng(40 + c).standard_normal((w.nz, w.ny, w.nx)) for c in range(5)]
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    pz.helmholtz_z_setup(plan, w.a)
    ref_p = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    ref_u = [oracle.helmholtz_z_solve(zc, zf, w.a, r) for r in rs]
    s = torch.cuda.Stream()
    for _ in range(2):
        hp = torch.from_numpy(f.copy()).pin_memory()
        hu = [torch.from_numpy(r.copy()).pin_memory() for r in rs]
        with torch.cuda.stream(s):
            pz.pz_solve_host_batch(plan, hp, hu)
        s.synchronize()
        assert rel_err(hp.numpy(), ref_p) <= TOL
        for h, ref in zip(hu, ref_u):
            assert rel_err(h.numpy(), ref) <= TOL
    hu = [torch.from_numpy(rs[0].copy()).pin_memory()]
    pz.pz_solve_host_batch(plan, None, hu)               # Helmholtz only, default stream
    torch.cuda.synchronize()
    assert rel_err(hu[0].numpy(), ref_u[0]) <= TOL
    pz.poisson_plan_destroy(plan)


# ------------------------------------------------------- BASELINE configs 1 and 2 in full

def test_config1_poisson_and_helmholtz_full(torch, pz, wl, oracle):
    w = wl.CONFIGS["c1"]
    zc, zf = wl.grid(w)
    f = wl.poisson_rhs(w)
    ref = oracle.poisson_solve(w.lx, w.ly, zc, zf, f, 1)
    for variant in (0, 1, 2):
        got = gpu_poisson(torch, pz, w, zc, zf, f, [("zsolve_variant", variant)])
        assert rel_err(got, ref) <= TOL
    r = wl.helmholtz_rhs(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    pz.helmholtz_z_setup(plan, w.a)
    u = torch.from_numpy(r).cuda()
    pz.helmholtz_z_solve(plan, u)
    assert rel_err(u.cpu().numpy(), oracle.helmholtz_z_solve(zc, zf, w.a, r)) <= TOL
