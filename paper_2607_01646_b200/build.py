"""Build libphx.so (the C-ABI library of include/phx.h) in-tree with nvcc for sm_100a.

    python -m paper_2607_01646_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.  The CUDA runtime
is linked statically, so the library LOADS on a machine without a GPU or driver (the CPU test
tier checks its exported symbols); every compute entry point needs a B200.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libphx.so")
SOURCES = [os.path.join(CSRC, f) for f in ("phx_api.cu", "phx_kernels.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "phx_kernels.cuh"),
                  os.path.join(os.path.dirname(HERE), "include", "phx.h")]

# No --use_fast_math, default -ftz=false -prec-div=true -prec-sqrt=true: the arithmetic contract
# of include/phx.h (every fp32 operation individually rounded) depends on it.
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-fvisibility=hidden,-Wall", "-shared", "-cudart", "static",
]


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def up_to_date() -> bool:
    return os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
