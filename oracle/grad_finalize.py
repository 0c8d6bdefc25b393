"""grad_finalize.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle of the gradient producer's epilogue (second half: "single-pass
fusion of the sum-of-squares with the previous step's epilogue"; reading R34).

In the ZeRO-2 distributed optimizer the paper runs the optimizer's gradient shard is
the output of the reduce-scatter of the binary32 main gradients.  That producer is
the only place where the norm of step k+1's gradients can be had without a second pass over them
(the gradients of step k+1 do not exist while step k's kernel runs, and the clip coefficient must
be known before the first element of step k+1 moves).  What it computes, per shard:

    h   = g32 * scale          binary32 multiply, one rounding (scale: gradient averaging, 1.0 exact)
    g16 = RNE_bf16(h)          the optimizer's bf16 gradient bits (input of record of a1/a3)
    S   = sum widen(g16)^2     sum of squares of the ROUNDED values == phx_oracle_sumsq(g16)

so that handing S to the step (phx_set_clip_partials, count = 1) yields the same coefficient as the
optimizer's own a1 pass over g16.

Pins (tests/test_oracle_grad_finalize.py): torch's multiply + bf16 cast (a library routine),
math.fsum of the squares (the exactly rounded sum), exact-rational double rounding on crafted
inputs, enumerated ties, a hand-computable case, and the already pinned a1 (`oracle.sumsq`) on the
produced bits.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
from typing import Tuple

import numpy as np

from . import oracle as O

_ready = False


def _lib():
    global _ready
    L = O.lib()
    if not _ready:
        L.phx_oracle_grads_finalize.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.c_float,
                                                ctypes.POINTER(ctypes.c_uint16), ctypes.c_size_t]
        L.phx_oracle_grads_finalize.restype = ctypes.c_double
        _ready = True
    return L


def grads_finalize(g32: np.ndarray, scale: float = 1.0) -> Tuple[np.ndarray, float]:
    """(bf16 bits of RNE(g32 * scale), sum of squares of those rounded values) — reading R34."""
    g32 = np.ascontiguousarray(g32, dtype=np.float32)
    out = np.zeros(g32.shape[0], dtype=np.uint16)
    s = _lib().phx_oracle_grads_finalize(g32.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), float(np.float32(scale)),
                                         out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint16)), g32.shape[0])
    return out, float(s)
