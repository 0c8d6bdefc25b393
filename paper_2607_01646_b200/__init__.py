"""phx — B200-native fused AdamW + in-memory optimizer-state snapshot/restore.

The hot path of PHOENIX's zero-overhead in-memory checkpoint
(§V-B, 208-226 §VI-A, 248-254 §VI-E/F),
as a C-ABI library (`include/phx.h`) plus this thin ctypes binding.

Importing the package has no side effects; `binding` loads `libphx.so` on
first use and raises if it is missing (there is no CPU fallback).
"""

__all__ = ["binding", "workloads", "build"]
