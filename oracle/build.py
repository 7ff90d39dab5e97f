"""Build the CPU oracle (oracle/hough_oracle.c + oracle/hough_ext_oracle.c) into oracle/libhough_oracle.so.

TEST INFRASTRUCTURE ONLY (see the header of hough_oracle.c).  Flags matter for parity:
``-ffp-contract=off`` forbids GCC from fusing a*b+c into an FMA (it does so by default on
hosts with FMA units), ``-fno-fast-math`` keeps IEEE semantics, and no ``-march`` flag is
given so plain SSE2 scalar binary32 arithmetic is used (one rounding per operation, as
SURVEY.md section 8(c) A requires).
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hough_oracle.c")
SRC_EXT = os.path.join(HERE, "hough_ext_oracle.c")  # the rows SURVEY.md 8(f) marks "next"
LIB = os.path.join(HERE, "libhough_oracle.so")

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fno-unsafe-math-optimizations",
          "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile if the .so is missing or older than the source; return its path."""
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC_EXT)
            and os.path.getmtime(LIB) >= os.path.getmtime(__file__)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", *CFLAGS, "-o", tmp, SRC, SRC_EXT, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
