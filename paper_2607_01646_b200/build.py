"""Build libphx.so (the C-ABI library of include/phx.h) in-tree with nvcc for sm_100a.

    python -m paper_2607_01646_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.  The CUDA runtime
is linked statically, so the library LOADS on a machine without a GPU or driver (the CPU test
tier checks its exported symbols); every compute entry point needs a B200.

Also builds libphx_probe.so (csrc/probe/: the no-arithmetic HBM mix probe bench.py prints as roofline
context) — a BENCH-ONLY library of its own, so that libphx.so exports the product's calls only.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libphx.so")
SOURCES = [os.path.join(CSRC, f) for f in ("phx_api.cu", "phx_kernels.cu", "phx_no_alloc.cu")]
MAP = os.path.join(CSRC, "phx.map")
DEPS = SOURCES + [os.path.join(CSRC, "phx_kernels.cuh"), MAP,
                  os.path.join(os.path.dirname(HERE), "include", "phx.h")]
PROBE_LIB = os.path.join(HERE, "libphx_probe.so")
PROBE_SOURCES = [os.path.join(CSRC, "probe", "hbm_probe.cu")]
PROBE_DEPS = PROBE_SOURCES + [os.path.join(CSRC, "probe", "phx_probe.h")]

# No --use_fast_math, default -ftz=false -prec-div=true -prec-sqrt=true: the arithmetic contract
# of include/phx.h (every fp32 operation individually rounded) depends on it.  The HOST code derives the
# per-step scalars in binary64 and must round every operation too: -ffp-contract=off keeps gcc from fusing
# 1.0 - lr*wd into one fmsub on an FMA-capable host target (aarch64 Grace, -march with FMA), which would move
# `decay` by an ulp away from the oracle's.
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-fvisibility=hidden,-fvisibility-inlines-hidden,-Wall,-ffp-contract=off,-fno-fast-math",
    "-shared", "-cudart", "static",
]


# Tuning experiments only (profiles/ name the macro they set, e.g. PHX_NVCC_EXTRA=-DPHX_RESTORE_P2_CTAS=8): extra nvcc
# flags for the product library; unset in every build the tests, smoke() and bench.py's numbers come from.
def extra_flags():
    import shlex
    return shlex.split(os.environ.get("PHX_NVCC_EXTRA", ""))


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def _fresh(lib, deps) -> bool:
    return os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps)


def up_to_date() -> bool:
    return _fresh(LIB, DEPS) and _fresh(PROBE_LIB, PROBE_DEPS)


def _link(lib, sources, extra, verbose):
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [nvcc(), *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *sources]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or not _fresh(LIB, DEPS):
        # the version script exports phx_* only (no leaked template instantiations of the C++ runtime)
        _link(LIB, SOURCES, ["-Xlinker", f"--version-script={MAP}", *extra_flags()], verbose)
    if force or not _fresh(PROBE_LIB, PROBE_DEPS):
        _link(PROBE_LIB, PROBE_SOURCES, [], verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
