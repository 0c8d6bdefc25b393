"""Compile oracle/phx_oracle.c into oracle/libphx_oracle.so with gcc (TEST INFRASTRUCTURE).

Building the checker is not using it: __graft_entry__.build() calls this too.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "phx_oracle.c")
LIB = os.path.join(HERE, "libphx_oracle.so")

# -ffp-contract=off: no FMA contraction; every operation is one IEEE rounding.
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
          "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
