"""Build libxodiac.so in-tree with nvcc for sm_100a (B200).  `python -m paper_2512_06729_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
CHECKED = bool(os.environ.get("XOD_CHECK"))   # debugging build: bounds-checked table indices (csrc/xod_cta.cuh)
LIB = os.path.join(HERE, "libxodiac_check.so" if CHECKED else "libxodiac.so")
SOURCES = ["api.cu", "pack.cpp", "pack_fused.cpp", "pack_jac.cpp", "pack_lu.cpp", "pack_path.cpp"]
HEADERS = ["kernels.cuh", "fused.cuh", "jac_tiled.cuh", "newton.cuh", "photo.cuh", "transport.cuh", "pathway.cuh", "equil.cuh", "sched.cuh", "rates2.cuh", "xod_math.cuh", "xod_cta.cuh", "xod_internal.h", os.path.join("..", "..", "include", "xodiac.h")]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force=False, verbose=False):
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-I" + CSRC, "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    if CHECKED:
        cmd += ["-DXOD_CHECK"]
    cmd += [os.path.join(CSRC, f) for f in SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
