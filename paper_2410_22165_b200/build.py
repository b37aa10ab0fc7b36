"""Build step: compile csrc/econojax.cu into libeconojax.so for sm_100a, in-tree.

nvcc cross-compiles without a GPU.  Flags: -fmad=false keeps every binary32 operation of
the state update a single correctly rounded operation (G31; the kernels also use the
__f*_rn intrinsics); -lineinfo maps the ncu source page to the code.
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "econojax.cu")
DEV = os.path.join(_HERE, "csrc", "ej_device.cuh")
HDR = os.path.join(os.path.dirname(_HERE), "include", "econojax.h")
LIB = os.path.join(_HERE, "libeconojax.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build_lib(force: bool = False, verbose: bool = False) -> str:
    csrc = os.path.dirname(SRC)
    newest = max([os.path.getmtime(HDR)] + [os.path.getmtime(os.path.join(csrc, f)) for f in os.listdir(csrc)])
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
