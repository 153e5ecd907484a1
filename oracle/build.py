"""Build the CPU oracle (test infrastructure, not the product): gcc -O2, no fast-math, OpenMP.

    python oracle/build.py        # writes oracle/libmp_oracle.so
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "mp_oracle.c")]
DEPS = SRC + [os.path.join(HERE, "mp_oracle.h"), os.path.join(HERE, "mp_oracle_body.inc")]
LIB = os.path.join(HERE, "libmp_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", *SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
