"""Build the CUDA path into paper_1305_4855_b200/libhough_b200.so (in-tree, sm_100a only).

nvcc cross-compiles without a GPU.  ``-fmad=false`` is belt and braces: the exact recipe
of the vote already uses __fmul_rn/__fadd_rn/__fsub_rn/__fdiv_rn, which are never
contracted; the flag keeps the compiler from fusing anything else in those kernels.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhough_b200.so")
SOURCES = ["hough_api.cu", "hough_sweep.cu", "hough_lists.cu", "hough_peaklists.cu", "hough_peaks.cu", "hough_vertex.cu",
           "hough_fit.cu", "hough_microbench.cu", "hough_noalloc.cu"]
HEADERS = [os.path.join(CSRC, "hough_internal.cuh"), os.path.join(CSRC, "hough_device.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "hough.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "-shared", "-cudart", "shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if missing or out of date; return the path of the shared library."""
    if not force and not _stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [NVCC, *FLAGS, *os.environ.get("HOUGH_NVCC_FLAGS", "").split(), "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
