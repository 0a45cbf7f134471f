"""Build libdc.so (the CUDA path) in-tree with nvcc for sm_100a.  No JIT cache, no torch."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(_HERE, "csrc", "dc_kernels.cu")]
DEPS = SRC + [os.path.join(_HERE, "csrc", h) for h in ("dc_geom.cuh", "dc_narrow.cuh", "dc_newton.cuh", "dc_blank.cuh", "dc_paper.cuh", "dc_donor.cuh", "dc_far.cuh")] + [
              os.path.join(os.path.dirname(_HERE), "include", "dc.h")]
LIB = os.path.join(_HERE, "libdc.so")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--use_fast_math=false"]


def _nvcc() -> str:
    for p in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if p and os.path.exists(p):
            return p
    raise RuntimeError("nvcc not found: libdc.so cannot be built")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in DEPS)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    if verbose:
        flags += ["-Xptxas", "-v"]
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [_nvcc()] + flags + ["-o", tmp] + SRC
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build_lib(force=True, verbose="-v" in sys.argv))
