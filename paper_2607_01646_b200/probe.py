"""Binding of libphx_probe.so — a BENCH-ONLY diagnostic (csrc/probe/phx_probe.h), not the product.

`phx_hbm_probe_async` runs one no-arithmetic streaming pass with the fused step's access pattern; bench.py
prints the bandwidth it reaches for the step's own read:write mix next to the driver-measured copy peak.
"""
from __future__ import annotations

import ctypes as C
import os

from .binding import _ptr

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libphx_probe.so")
_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_01646_b200.build`")
        L = C.CDLL(LIB_PATH)
        L.phx_hbm_probe_async.restype = C.c_int
        L.phx_hbm_probe_async.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.phx_hbm_probe_persistent_async.restype = C.c_int
        L.phx_hbm_probe_persistent_async.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        _lib = L
    return _lib


def phx_hbm_probe_async(d_buf, plane_bytes: int, n_read: int, n_write: int, stream=None) -> int:
    """Returns the probe's status code (0 ok, -1 invalid argument, -2 alignment, -9 CUDA error)."""
    return lib().phx_hbm_probe_async(_ptr(d_buf), plane_bytes, n_read, n_write, _ptr(stream))


def phx_hbm_probe_persistent_async(d_buf, plane_bytes: int, n_read: int, n_write: int, grid: int, stream=None) -> int:
    """The same pass with `grid` persistent CTAs walking the groups with a grid stride."""
    return lib().phx_hbm_probe_persistent_async(_ptr(d_buf), plane_bytes, n_read, n_write, grid, _ptr(stream))
