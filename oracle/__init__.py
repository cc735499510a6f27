"""CPU oracle for the Poisson / z-Helmholtz hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2502_06296_b200`` (the CUDA path) and must never import it.

``oracle.c``          the definition-level solves in plain C (double, OpenMP)
``cpu.py``            ctypes loader + numpy-facing wrappers (marshalling only)
``algorithms.py``     step-by-step numpy transcriptions of the paper's Algorithm 1
                      and Algorithm 2 and of the packed
                      half-complex layout of Appendix A
"""
from .cpu import (  # noqa: F401
    build,
    lib,
    num_threads,
    z_tables,
    modified_wavenumbers,
    dft_naive,
    fft_radix2,
    dft_xy,
    thomas,
    thomas_poisson,
    zero_mode_column,
    apply_poisson_operator,
    helmholtz_matrix,
    poisson_solve,
    helmholtz_z_solve,
    helmholtz_z_solve_columns,
    helmholtz_w_matrix,
    helmholtz_w_solve,
    apply_helmholtz3d_operator,
    helmholtz3d_solve,
)
