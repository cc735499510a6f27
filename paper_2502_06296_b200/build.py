"""Build libpz_b200.so (hand-written CUDA for sm_100a + the C ABI of include/pz.h) in-tree.

    python -m paper_2502_06296_b200.build [--force] [--verbose] [--probes]

nvcc cross-compiles without a GPU.  Objects go to csrc/build/, the library next to this file.
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libpz_b200.so")
SOURCES = ["pz_api.cu", "pz_fft_x.cu", "pz_fft_y.cu", "pz_fft_generic.cu", "pz_fft_xy_fwd.cu", "pz_fft_xy_inv.cu", "pz_zsolve.cu", "pz_zsolve_cr.cu", "pz_zsolve_tma.cu", "pz_zslab.cu", "pz_helmholtz.cu", "pz_helmholtz_tma.cu", "pz_projection.cu", "pz_tma.cu"]
HEADERS = ["pz_internal.h", "pz_fft.cuh", "pz_tma.cuh", "pz_zsolve_pair.cuh", "pz_fft_xy_impl.cuh", "pz_fft2.cuh", os.path.join("..", "..", "include", "pz.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--fmad=true"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def build(force: bool = False, verbose: bool = False, probes: bool = False) -> str:
    """probes: compile the timing-only diagnostics (-DPZ_PROBES; wrong results) in; forces a rebuild."""
    os.makedirs(OBJ, exist_ok=True)
    force = force or probes
    hdr = _newest_header()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr):
            cmd = [_nvcc(), *NVCC_FLAGS, *(["-DPZ_PROBES"] if probes else []), "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    if jobs:
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            for cmd, r in ex.map(run, jobs):
                if verbose or r.returncode != 0:
                    sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed for " + cmd[-3])
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if jobs or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        cmd = [_nvcc(), "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a",
               "-Xcompiler", "-fPIC"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, probes="--probes" in sys.argv))
