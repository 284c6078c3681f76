"""Builds paper_1412_1498_b200/libgf.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgf.so")
SOURCES = ["gf_kernels.cu", "gf_fftsd.cu", "gf_fft.cu", "gf_api.cu", "gf_peaks.cu", "gf_sun.cu", "gf_static.cu"]
HEADERS = ["gf_device.cuh", "gf_internal.h", os.path.join("..", "..", "include", "gf.h")]
# -split-compile 0: the back end compiles the kernels of a translation unit on all host cores (gf_kernels.cu: 4 min -> 1 min)
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
              "-split-compile", "0"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        import tempfile
        from concurrent.futures import ThreadPoolExecutor

        with tempfile.TemporaryDirectory() as tmp:
            def compile_one(src):  # one nvcc per translation unit, side by side
                obj = os.path.join(tmp, src + ".o")
                subprocess.check_call(["nvcc", *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c",
                                       os.path.join(CSRC, src), "-o", obj])
                return obj

            with ThreadPoolExecutor(len(SOURCES)) as pool:
                objs = list(pool.map(compile_one, SOURCES))
            subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs,
                                   "-lcufft"])
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
