"""The C-ABI library loads and exports every symbol include/pz.h declares; argument
validation works without a GPU; no compute is attempted here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "pz.h")).read()
    names = re.findall(r"PZ_API\s+[\w\s\*]+?\b(\w+)\s*\(", text)
    assert len(names) >= 12
    return names


@pytest.fixture(scope="module")
def built():
    from paper_2502_06296_b200 import build

    return build.build()


def test_library_exports_every_declared_symbol(built):
    lib = ctypes.CDLL(built)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/pz.h but not exported"


def test_binding_covers_every_declared_symbol(built):
    from paper_2502_06296_b200 import binding

    assert sorted(binding.SIGNATURES) == sorted(_declared_symbols())
    for name in _declared_symbols():
        assert callable(getattr(binding, name)), f"binding lacks {name}"
    assert binding.pz_version() >= 100
    assert binding.pz_launch_count() >= 0


def test_argument_validation_needs_no_gpu(built):
    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import workloads as wl

    zf = wl.z_faces(16)
    zc = wl.z_centres(zf)
    cases = [
        (dict(nx=22, ny=16, nz=16), pz.PZ_EUNSUPPORTED),   # nx / 2 = 11: a prime factor above 7
        (dict(nx=16, ny=26, nz=16), pz.PZ_EUNSUPPORTED),   # ny = 2 * 13
        (dict(nx=18, ny=12, nz=16), pz.PZ_EUNSUPPORTED),   # nx ny = 216 is not a multiple of 16 (column tiles)
        (dict(nx=15, ny=16, nz=16), pz.PZ_EUNSUPPORTED),   # odd
        (dict(nx=16, ny=4, nz=16), pz.PZ_EUNSUPPORTED),    # ny < 8
        (dict(nx=32768, ny=16, nz=16), pz.PZ_EUNSUPPORTED),
        (dict(nx=0, ny=16, nz=16), pz.PZ_EINVAL),
        (dict(nx=16, ny=16, nz=16, lx=-1.0), pz.PZ_EINVAL),
        (dict(nx=16, ny=16, nz=16, bc=7), pz.PZ_EUNSUPPORTED),
    ]
    for kw, status in cases:
        args = dict(nx=16, ny=16, nz=16, lx=1.0, ly=1.0, bc=0)
        args.update(kw)
        with pytest.raises(pz.PzError) as ei:
            pz.poisson_plan_create(args["nx"], args["ny"], args["nz"], args["lx"], args["ly"], zc, zf, args["bc"])
        assert ei.value.status == status, kw
        assert pz.pz_last_error() != ""
    # nz < 4
    zf3 = wl.z_faces(3)
    with pytest.raises(pz.PzError) as ei:
        pz.poisson_plan_create(16, 16, 3, 1.0, 1.0, wl.z_centres(zf3), zf3)
    assert ei.value.status == pz.PZ_EUNSUPPORTED
    # non-monotone faces / centre outside its cell
    bad = zf.copy()
    bad[5] = bad[4]
    with pytest.raises(pz.PzError) as ei:
        pz.poisson_plan_create(16, 16, 16, 1.0, 1.0, zc, bad)
    assert ei.value.status == pz.PZ_EINVAL
    badc = zc.copy()
    badc[3] = zf[5]
    with pytest.raises(pz.PzError) as ei:
        pz.poisson_plan_create(16, 16, 16, 1.0, 1.0, badc, zf)
    assert ei.value.status == pz.PZ_EINVAL


def test_no_cpu_fallback_without_a_device(built):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import workloads as wl

    zf = wl.z_faces(16)
    with pytest.raises(pz.PzError) as ei:
        pz.poisson_plan_create(16, 16, 16, 1.0, 1.0, wl.z_centres(zf), zf)
    assert ei.value.status == pz.PZ_ECUDA
    assert "no CPU fallback" in str(ei.value)


def test_product_never_imports_the_oracle():
    """The CUDA path and the oracle share no code: neither tree mentions the other."""
    pkg = os.path.join(ROOT, "paper_2502_06296_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text and "oracle.c" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libpz" not in text and "binding" not in text and "csrc" not in text.replace(
                "paper_2502_06296_b200/csrc/", ""), f
