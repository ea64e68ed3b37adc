"""Build the CPU oracle (test infrastructure) into oracle/libozaki2_oracle.so.

    python oracle/build.py            # build if stale
    python oracle/build.py --force
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ozaki2_oracle.c")
LIB = os.path.join(HERE, "libozaki2_oracle.so")

# -frounding-math / no fast-math: the FP32 steps run under fesetround().
CFLAGS = ["-O2", "-std=gnu11", "-fopenmp", "-frounding-math", "-fno-fast-math", "-ffp-contract=off",
          "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", *CFLAGS, "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
