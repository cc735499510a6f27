"""Thin ctypes binding of include/pz.h -- argument marshalling only.

Same names as the C ABI.  PyTorch is used for device memory and streams: a field is a
contiguous float64 CUDA tensor of shape (nz, ny, nx) (or any shape with nx*ny*nz elements),
passed by ``data_ptr()``; ``stream`` defaults to ``torch.cuda.current_stream()``.

There is no CPU fallback: if ``libpz_b200.so`` is missing, or no CUDA device is present, the
calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpz_b200.so")

PZ_OK, PZ_EINVAL, PZ_EUNSUPPORTED, PZ_ENOMEM, PZ_ECUDA, PZ_ENOTSETUP = range(6)
PZ_BC_PERIODIC_XY_NEUMANN_P_DIRICHLET_U = 0
PZ_STAGE_FFT_X_FWD, PZ_STAGE_FFT_Y_FWD, PZ_STAGE_Z_SOLVE, PZ_STAGE_FFT_Y_INV, PZ_STAGE_FFT_X_INV = range(5)
PZ_STAGE_FFT_XY_FWD, PZ_STAGE_FFT_XY_INV = 5, 6

# every symbol include/pz.h declares: (name, restype, argtypes)
_vp, _i, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
_dp = ctypes.POINTER(ctypes.c_double)
SIGNATURES = {
    "poisson_plan_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _d, _d, _dp, _dp, _i]),
    "poisson_solve": (_i, [_vp, _vp, _vp]),
    "poisson_slab_plan_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _d, _d, _dp, _dp, _i, _i, _i, ctypes.POINTER(_i)]),
    "poisson_slab_boundary_doubles": (ctypes.c_longlong, [_vp]),
    "poisson_solve_reduce": (_i, [_vp, _vp, _vp, _vp]),
    "poisson_solve_reduce_push": (_i, [_vp, _vp, ctypes.POINTER(_vp), ctypes.POINTER(_vp), ctypes.c_longlong, _vp]),
    "poisson_solve_finish_wait": (_i, [_vp, _vp, _vp, _vp, ctypes.c_longlong, _vp]),
    "poisson_solve_finish": (_i, [_vp, _vp, _vp, _vp]),
    "helmholtz_z_setup": (_i, [_vp, _d]),
    "helmholtz_w_setup": (_i, [_vp, _d]),
    "helmholtz_w_solve": (_i, [_vp, _vp, _vp]),
    "helmholtz_z_solve": (_i, [_vp, _vp, _vp]),
    "helmholtz_z_solve_n": (_i, [_vp, ctypes.POINTER(_vp), _i, _vp]),
    "poisson_solve_host": (_i, [_vp, _vp, _vp]),
    "helmholtz_z_solve_host": (_i, [_vp, _vp, _vp]),
    "helmholtz_z_rhs": (_i, [_vp, _vp, _vp, _vp]),
    "helmholtz_z_step": (_i, [_vp, _vp, _vp, _vp]),
    "helmholtz3d_setup": (_i, [_vp, ctypes.c_double]),
    "helmholtz3d_solve": (_i, [_vp, _vp, _vp]),
    "pz_divergence_rhs": (_i, [_vp, _vp, _vp, _vp, _vp, ctypes.c_double, _vp]),
    "pz_project": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_double, _vp]),
    "pz_pressure_correction": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_double, _vp]),
    "pz_solve_host_batch": (_i, [_vp, _vp, ctypes.POINTER(_vp), ctypes.c_int, _vp]),
    "poisson_zsolve_noalloc": (_i, [_vp, _vp, _vp]),
    "poisson_plan_destroy": (_i, [_vp]),
    "pz_last_error": (ctypes.c_char_p, []),
    "pz_poisson_stage": (_i, [_vp, _vp, _i, _vp]),
    "pz_set_option": (_i, [_vp, ctypes.c_char_p, _i]),
    "pz_get_option": (_i, [_vp, ctypes.c_char_p, ctypes.POINTER(_i)]),
    "pz_profile_enable": (_i, [_vp, _i]),
    "pz_profile_read": (_i, [_vp, _i, ctypes.POINTER(_d), ctypes.POINTER(ctypes.c_longlong)]),
    "pz_launch_count": (ctypes.c_longlong, []),
    "pz_version": (_i, []),
    "pz_fft_radices": (_i, [_i, _i, _i, ctypes.POINTER(ctypes.c_int), _i]),
}

_lib = None


def pz_bc(bcx: str = "P", bcy: str = "P", bcz: str = "NN") -> int:
    """PZ_BC(...) of include/pz.h from letters: x, y in 'P' (periodic), 'N' (zero gradient), 'D' (zero
    value at the end faces); z in 'NN', 'DD', 'ND', 'DN' (bottom, top)."""
    d = {"P": 0, "N": 1, "D": 2}
    z = {"NN": 0, "DD": 1, "ND": 2, "DN": 3}
    return d[bcx] + 4 * d[bcy] + 16 * z[bcz]


class PzError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"pz status {status}: {message}")
        self.status = status


def lib() -> ctypes.CDLL:
    """Load libpz_b200.so (built by ``python -m paper_2502_06296_b200.build``).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not found: build the CUDA extension with "
                "`python -m paper_2502_06296_b200.build` (there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(status: int):
    if status != PZ_OK:
        raise PzError(status, lib().pz_last_error().decode())


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _dev_ptr(t, n) -> int:
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("field must be a contiguous float64 CUDA tensor")
    if n is not None and t.numel() != n:
        raise ValueError(f"field has {t.numel()} elements, plan expects {n}")
    return t.data_ptr()


def _host_ptr(t, n: int) -> int:
    import torch

    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags["C_CONTIGUOUS"] or t.size != n:
            raise TypeError("host field must be a C-contiguous float64 array of nx*ny*nz elements")
        return t.ctypes.data
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("host field must be a contiguous float64 CPU tensor or numpy array")
    if t.numel() != n:
        raise ValueError(f"field has {t.numel()} elements, plan expects {n}")
    return t.data_ptr()


class Plan:
    """Owner of a ``pz_plan*``; destroyed with :func:`poisson_plan_destroy` or on garbage collection."""

    def __init__(self, handle: int, nx: int, ny: int, nz: int):
        self.handle, self.nx, self.ny, self.nz = handle, nx, ny, nz
        self.n = nx * ny * nz

    def __del__(self):
        try:
            poisson_plan_destroy(self)
        except Exception:
            pass


def poisson_plan_create(nx: int, ny: int, nz: int, lx: float, ly: float, zc, zf,
                        bc: int = PZ_BC_PERIODIC_XY_NEUMANN_P_DIRICHLET_U) -> Plan:
    zc = np.ascontiguousarray(zc, dtype=np.float64)
    zf = np.ascontiguousarray(zf, dtype=np.float64)
    if zc.size != nz or zf.size != nz + 1:
        raise ValueError("zc must have nz entries and zf nz+1")
    out = _vp()
    _check(lib().poisson_plan_create(ctypes.byref(out), nx, ny, nz, float(lx), float(ly),
                                     zc.ctypes.data_as(_dp), zf.ctypes.data_as(_dp), bc))
    return Plan(out.value, nx, ny, nz)


def poisson_slab_plan_create(nx: int, ny: int, nz: int, lx: float, ly: float, zc, zf, n_slabs: int, slab: int, kbounds,
                             bc: int = PZ_BC_PERIODIC_XY_NEUMANN_P_DIRICHLET_U) -> Plan:
    """Plan of rank `slab` of a Poisson problem cut into `n_slabs` z-slabs; the
    plan's field is the slab's planes [kbounds[slab], kbounds[slab+1]) of the global grid zc, zf."""
    zc = np.ascontiguousarray(zc, dtype=np.float64)
    zf = np.ascontiguousarray(zf, dtype=np.float64)
    kb = np.ascontiguousarray(kbounds, dtype=np.int32)
    if zc.size != nz or zf.size != nz + 1 or kb.size != n_slabs + 1:
        raise ValueError("zc must have nz entries, zf nz+1 and kbounds n_slabs+1")
    out = _vp()
    _check(lib().poisson_slab_plan_create(ctypes.byref(out), nx, ny, nz, float(lx), float(ly), zc.ctypes.data_as(_dp),
                                          zf.ctypes.data_as(_dp), bc, n_slabs, slab,
                                          kb.ctypes.data_as(ctypes.POINTER(_i))))
    return Plan(out.value, nx, ny, int(kb[slab + 1] - kb[slab]))


def poisson_slab_boundary_doubles(plan: Plan) -> int:
    return int(lib().poisson_slab_boundary_doubles(plan.handle))


def poisson_solve_reduce(plan: Plan, p, boundary_out, stream=None) -> None:
    _check(lib().poisson_solve_reduce(plan.handle, _dev_ptr(p, plan.n), _dev_ptr(boundary_out, poisson_slab_boundary_doubles(plan)),
                                      _stream_ptr(stream)))


def poisson_solve_reduce_push(plan: Plan, p, ball_ptrs, flag_ptrs, epoch: int, stream=None) -> None:
    """ball_ptrs / flag_ptrs: device addresses (ints) of every rank's gathered buffer / flag array."""
    n = len(ball_ptrs)
    a = (_vp * n)(*[int(x) for x in ball_ptrs])
    f = (_vp * n)(*[int(x) for x in flag_ptrs])
    _check(lib().poisson_solve_reduce_push(plan.handle, _dev_ptr(p, plan.n), a, f, int(epoch), _stream_ptr(stream)))


def poisson_solve_finish_wait(plan: Plan, p, boundary_all, flags, epoch: int, stream=None) -> None:
    _check(lib().poisson_solve_finish_wait(plan.handle, _dev_ptr(p, plan.n), _dev_ptr(boundary_all, None), int(flags.data_ptr()),
                                           int(epoch), _stream_ptr(stream)))


def poisson_solve_finish(plan: Plan, p, boundary_all, stream=None) -> None:
    _check(lib().poisson_solve_finish(plan.handle, _dev_ptr(p, plan.n), _dev_ptr(boundary_all, None), _stream_ptr(stream)))


def poisson_plan_destroy(plan: Plan) -> None:
    if plan is not None and plan.handle:
        h, plan.handle = plan.handle, 0
        _check(lib().poisson_plan_destroy(h))


def poisson_solve(plan: Plan, p, stream=None) -> None:
    _check(lib().poisson_solve(plan.handle, _dev_ptr(p, plan.n), _stream_ptr(stream)))


def helmholtz_z_setup(plan: Plan, a: float) -> None:
    _check(lib().helmholtz_z_setup(plan.handle, float(a)))


def helmholtz_z_solve(plan: Plan, u, stream=None) -> None:
    _check(lib().helmholtz_z_solve(plan.handle, _dev_ptr(u, plan.n), _stream_ptr(stream)))


def helmholtz_z_solve_n(plan: Plan, fields, stream=None) -> None:
    ptrs = (_vp * len(fields))(*[_dev_ptr(u, plan.n) for u in fields])
    _check(lib().helmholtz_z_solve_n(plan.handle, ptrs, len(fields), _stream_ptr(stream)))


def helmholtz_w_setup(plan: Plan, a: float) -> None:
    _check(lib().helmholtz_w_setup(plan.handle, float(a)))


def helmholtz_w_solve(plan: Plan, w, stream=None) -> None:
    _check(lib().helmholtz_w_solve(plan.handle, _dev_ptr(w, plan.n), _stream_ptr(stream)))


def poisson_solve_host(plan: Plan, p_host, stream=None) -> None:
    _check(lib().poisson_solve_host(plan.handle, _host_ptr(p_host, plan.n), _stream_ptr(stream)))


def helmholtz_z_rhs(plan: Plan, ustar2, uk, stream=None) -> None:
    _check(lib().helmholtz_z_rhs(plan.handle, _dev_ptr(ustar2, plan.n), _dev_ptr(uk, plan.n), _stream_ptr(stream)))


def helmholtz_z_step(plan: Plan, ustar2, uk, stream=None) -> None:
    _check(lib().helmholtz_z_step(plan.handle, _dev_ptr(ustar2, plan.n), _dev_ptr(uk, plan.n), _stream_ptr(stream)))


def helmholtz3d_setup(plan: Plan, a: float) -> None:
    _check(lib().helmholtz3d_setup(plan.handle, float(a)))


def helmholtz3d_solve(plan: Plan, u, stream=None) -> None:
    _check(lib().helmholtz3d_solve(plan.handle, _dev_ptr(u, plan.n), _stream_ptr(stream)))


def pz_divergence_rhs(plan: Plan, u, v, w, rhs, inv_gdt: float, stream=None) -> None:
    n = plan.n
    _check(lib().pz_divergence_rhs(plan.handle, _dev_ptr(u, n), _dev_ptr(v, n), _dev_ptr(w, n), _dev_ptr(rhs, n),
                                   float(inv_gdt), _stream_ptr(stream)))


def pz_project(plan: Plan, u, v, w, p, phi, gdt: float, stream=None) -> None:
    n = plan.n
    _check(lib().pz_project(plan.handle, _dev_ptr(u, n), _dev_ptr(v, n), _dev_ptr(w, n), _dev_ptr(p, n),
                            _dev_ptr(phi, n), float(gdt), _stream_ptr(stream)))


def pz_pressure_correction(plan: Plan, u, v, w, p, work, gdt: float, stream=None) -> None:
    n = plan.n
    _check(lib().pz_pressure_correction(plan.handle, _dev_ptr(u, n), _dev_ptr(v, n), _dev_ptr(w, n), _dev_ptr(p, n),
                                        _dev_ptr(work, n), float(gdt), _stream_ptr(stream)))


def pz_solve_host_batch(plan: Plan, p_host, u_hosts, stream=None) -> None:
    """p_host: pinned host tensor or None; u_hosts: sequence of pinned host tensors."""
    n = len(u_hosts)
    arr = (_vp * max(n, 1))(*[_host_ptr(u, plan.n) for u in u_hosts])
    _check(lib().pz_solve_host_batch(plan.handle, _host_ptr(p_host, plan.n) if p_host is not None else None,
                                     arr, n, _stream_ptr(stream)))


def helmholtz_z_solve_host(plan: Plan, u_host, stream=None) -> None:
    _check(lib().helmholtz_z_solve_host(plan.handle, _host_ptr(u_host, plan.n), _stream_ptr(stream)))


def pz_poisson_stage(plan: Plan, p, stage: int, stream=None) -> None:
    _check(lib().pz_poisson_stage(plan.handle, _dev_ptr(p, plan.n), int(stage), _stream_ptr(stream)))


PZ_NOALLOC_MAX_POINTS = 1 << 21


def poisson_zsolve_noalloc(plan: Plan, p, stream=None) -> None:
    """Step a3 on the spectral field p, in place, with the library's static workspace (no allocation)."""
    _check(lib().poisson_zsolve_noalloc(plan.handle, _dev_ptr(p, plan.n), _stream_ptr(stream)))


def pz_set_option(plan: Plan, key: str, value: int) -> None:
    _check(lib().pz_set_option(plan.handle, key.encode(), int(value)))


def pz_get_option(plan: Plan, key: str) -> int:
    v = _i()
    _check(lib().pz_get_option(plan.handle, key.encode(), ctypes.byref(v)))
    return v.value


KERNEL_CLASSES = ("fft_x_fwd", "fft_y_fwd", "pair0_fwd", "z_solve", "pair0_inv", "fft_y_inv", "fft_x_inv", "helmholtz",
                  "fft_xy_fwd", "fft_xy_inv", "div_rhs", "project", "helm_rhs")


def pz_profile_enable(plan: Plan, on: bool) -> None:
    _check(lib().pz_profile_enable(plan.handle, 1 if on else 0))


def pz_profile_read(plan: Plan, kernel_class: int):
    """-> (summed device milliseconds, launches) of one kernel class since pz_profile_enable(plan, True)."""
    ms, cnt = _d(), ctypes.c_longlong()
    _check(lib().pz_profile_read(plan.handle, int(kernel_class), ctypes.byref(ms), ctypes.byref(cnt)))
    return ms.value, cnt.value


def pz_launch_count() -> int:
    return int(lib().pz_launch_count())


def pz_version() -> int:
    return int(lib().pz_version())


def pz_fft_radices(n: int, min_points: int = 1, stride: int = 1):
    """Radices (first pass first) of the mixed-radix kernels for a complex length n; [] if unsupported."""
    buf = (ctypes.c_int * 20)()
    cnt = int(lib().pz_fft_radices(n, min_points, stride, buf, 20))
    return [int(buf[i]) for i in range(cnt)]


def pz_last_error() -> str:
    return lib().pz_last_error().decode()
