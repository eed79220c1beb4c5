"""Builds the CUDA shared library (C ABI of include/pt.h) in-tree for sm_100a with nvcc.

    python -m paper_1504_07433_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpt_b200.so")
SOURCES = [os.path.join(CSRC, "pt_kernels.cu")]
HEADERS = [os.path.join(CSRC, "pt_gimenez.cuh"), os.path.join(CSRC, "pt_epoch.cuh"), os.path.join(CSRC, "pt_direct.cuh"), os.path.join(CSRC, "pt_basis32.cuh"), os.path.join(CSRC, "pt_basis.cuh"), os.path.join(CSRC, "pt_orbit.cuh"), os.path.join(CSRC, "pt_math.cuh"), os.path.join(CSRC, "pt_flux.cuh"),
           os.path.join(HERE, "..", "include", "pt.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-DPT_BUILD_ARCH=100",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + SOURCES + ["-o", tmp]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
