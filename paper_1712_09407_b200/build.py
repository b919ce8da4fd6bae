"""Build step of the CUDA sector tracker: nvcc -> paper_1712_09407_b200/libtpcst.so (in-tree).

sm_100a only.  ``-fmad=false`` keeps one rounding per written fp32 operation (DESIGN.md section 3,
"Arithmetic"); div/sqrt stay IEEE (``-prec-div=true -prec-sqrt=true`` are nvcc's defaults).
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libtpcst.so")
SOURCES = ("api.cu", "kernels_ca.cu", "kernels_kalman.cu", "kernels_select.cu", "kernels_merge.cu",
           "static_select.cu", "selftest_l2.cu")
HEADERS = ("tpcst_internal.h", "kalman_math.cuh", os.path.join("..", "..", "include", "tpcst.h"))
NVCC_FLAGS = ("-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
              "-Xcompiler", "-fPIC", "-shared")


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA sector tracker cannot be built (there is no CPU fallback)")
    return exe


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if it is missing or older than its sources; return its path."""
    if force or stale():
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
