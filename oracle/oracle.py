"""oracle.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

The CPU oracle of the phx hot path: shard definition (a0), AdamW step (a3, via
phx_oracle.c), optional clip (a1), snapshot into ping-pong replica slots
(a4/a5) and restore (a6) as ordinary byte copies.  One element at a time, one
step at a time, in the order of SURVEY.md §8(a); every function cites the
passage or the DESIGN.md reading (R#) it follows.

The GPU path reaches exactly the plain result (it is a fusion and an overlap,
not an approximation), so this is the plain definition written out.

Parity status: every function here is pinned by tests/test_oracle_pins.py and
tests/test_oracle_shard.py (closed forms, exact rationals, torch.optim.AdamW,
float64 shadow, brute-force partition, round-trip invariants).  Nothing is
"parity unpinned".
"""
from __future__ import annotations

import ctypes
import struct
from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import build_oracle

# ----------------------------------------------------------------------------
# C arithmetic core (phx_oracle.c)
# ----------------------------------------------------------------------------

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build_oracle.build())
        f32p = ctypes.POINTER(ctypes.c_float)
        u16p = ctypes.POINTER(ctypes.c_uint16)
        L.phx_oracle_rne_bf16.argtypes = [ctypes.c_float]
        L.phx_oracle_rne_bf16.restype = ctypes.c_uint16
        L.phx_oracle_scalars.argtypes = [ctypes.c_float] * 5 + [ctypes.c_uint64, f32p]
        L.phx_oracle_scalars.restype = None
        L.phx_oracle_adamw_step.argtypes = [f32p, f32p, f32p, u16p, u16p, ctypes.c_size_t] + \
            [ctypes.c_float] * 5 + [ctypes.c_uint64, ctypes.c_float, ctypes.c_int]
        L.phx_oracle_adamw_step.restype = None
        L.phx_oracle_sumsq.argtypes = [u16p, ctypes.c_size_t]
        L.phx_oracle_sumsq.restype = ctypes.c_double
        L.phx_oracle_clip_coef.argtypes = [ctypes.c_double, ctypes.c_float]
        L.phx_oracle_clip_coef.restype = ctypes.c_float
        L.phx_oracle_regen_bf16.argtypes = [f32p, u16p, ctypes.c_size_t]
        L.phx_oracle_regen_bf16.restype = None
        u8p = ctypes.POINTER(ctypes.c_uint8)
        L.phx_oracle_adamw_step_ex.argtypes = [f32p, f32p, f32p, u16p, f32p, u16p, u8p, ctypes.c_size_t] + \
            [ctypes.c_float] * 5 + [ctypes.c_uint64, ctypes.c_float, ctypes.c_int]
        L.phx_oracle_adamw_step_ex.restype = None
        L.phx_oracle_sumsq_f32.argtypes = [f32p, ctypes.c_size_t]
        L.phx_oracle_sumsq_f32.restype = ctypes.c_double
        _lib = L
    return _lib


def _f32p(a: np.ndarray):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _u16p(a: np.ndarray):
    assert a.dtype == np.uint16 and a.flags.c_contiguous
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint16))


def scalars(lr, beta1, beta2, eps, wd, step) -> np.ndarray:
    """{decay, omb1, omb2, ss, sbc2} as fp32 (reading R6)."""
    out = np.zeros(5, dtype=np.float32)
    lib().phx_oracle_scalars(lr, beta1, beta2, eps, wd, int(step), _f32p(out))
    return out


def adamw_step(p, m, v, g_bits, p16, lr, beta1, beta2, eps, wd, step, coef=1.0, nthreads=1):
    """In-place canonical AdamW step (a3, reading R1) over numpy arrays."""
    n = p.shape[0]
    assert m.shape[0] == n and v.shape[0] == n and g_bits.shape[0] == n and p16.shape[0] == n
    lib().phx_oracle_adamw_step(_f32p(p), _f32p(m), _f32p(v), _u16p(g_bits), _u16p(p16), n,
                                lr, beta1, beta2, eps, wd, int(step), coef, int(nthreads))


def adamw_step_ex(p, m, v, g, p16, no_decay, lr, beta1, beta2, eps, wd, step, coef=1.0, nthreads=1):
    """In-place step of the general routine: `g` is uint16 bf16 bits or
    float32 gradients, `p16` may be None (no bf16 copy), `no_decay` may be None
    or a uint8 mask, one byte per element (reading R5b)."""
    n = p.shape[0]
    assert m.shape[0] == n and v.shape[0] == n and g.shape[0] == n
    null16 = ctypes.POINTER(ctypes.c_uint16)()
    null32 = ctypes.POINTER(ctypes.c_float)()
    g16, g32 = (_u16p(g), null32) if g.dtype == np.uint16 else (null16, _f32p(g))
    nd = ctypes.POINTER(ctypes.c_uint8)()
    if no_decay is not None:
        assert no_decay.dtype == np.uint8 and no_decay.shape[0] == n and no_decay.flags.c_contiguous
        nd = no_decay.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))
    lib().phx_oracle_adamw_step_ex(_f32p(p), _f32p(m), _f32p(v), g16, g32,
                                   null16 if p16 is None else _u16p(p16), nd, n,
                                   lr, beta1, beta2, eps, wd, int(step), coef, int(nthreads))


def sumsq(g: np.ndarray) -> float:
    """Sum of squares of the gradients (bf16 bits or float32), a1 / reading R7."""
    if g.dtype == np.float32:
        return float(lib().phx_oracle_sumsq_f32(_f32p(g), g.shape[0]))
    return float(lib().phx_oracle_sumsq(_u16p(g), g.shape[0]))


def clip_coef(sumsq_value: float, max_norm: float) -> np.float32:
    """fp32(min(1, max_norm/(sqrt(S)+1e-6))) (a1, reading R7)."""
    return np.float32(lib().phx_oracle_clip_coef(float(sumsq_value), float(max_norm)))


def rne_bf16(x: np.ndarray) -> np.ndarray:
    """bf16 bits of fp32 values, round-to-nearest-even (reading R1, last line)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.zeros(x.shape[0], dtype=np.uint16)
    lib().phx_oracle_regen_bf16(_f32p(x), _u16p(out), x.shape[0])
    return out


# ----------------------------------------------------------------------------
# a0: shard definition (readings R15, R14; "sharded model and optimizer states",
# PAPER.md:27; ZeRO-2)
# ----------------------------------------------------------------------------

TENSOR_NO_DECAY = 1  # phx_tensor_desc_t.flags bit: the tensor takes weight decay 0 (reading R5b)
PAD_UNIT = 64  # elements: every rank's range is a multiple of 64 (256 B of fp32, 128 B of bf16)
HEADER_BYTES = 256
MAGIC = b"PHXSNAP1"
VERSION = 1
FNV_OFFSET = 0xCBF29CE484222325
FNV_PRIME = 0x100000001B3
M64 = (1 << 64) - 1


def fnv1a64(data: bytes) -> int:
    h = FNV_OFFSET
    for b in data:
        h ^= b
        h = (h * FNV_PRIME) & M64
    return h


def define_shard(layout: Sequence[Tuple[int, int]], dp_size: int, dp_rank: int,
                 tp=(1, 0), pp=(1, 0), flags: Optional[Sequence[int]] = None):
    """Flatten the rank's tensor list in list order, pad the total up to a multiple of
    PAD_UNIT*dp_size, cut equal contiguous ranges; rank r owns [r*L, (r+1)*L).

    Returns dict(n, n_padded, total_numel, shard_begin, segments, layout_hash), with
    segments = [(tensor_id, off_in_tensor, off_in_shard, length)].
    """
    assert dp_size >= 1 and 0 <= dp_rank < dp_size
    total = sum(int(numel) for numel, _ in layout)
    unit = PAD_UNIT * dp_size
    L = ((total + unit - 1) // unit) * PAD_UNIT
    begin = dp_rank * L
    end = begin + L
    n = min(max(total - begin, 0), L)
    segments = []
    t0 = 0
    for numel, tid in layout:
        t1 = t0 + int(numel)
        lo, hi = max(t0, begin), min(t1, end)
        if hi > lo:
            segments.append((int(tid), lo - t0, lo - begin, hi - lo))
        t0 = t1
    fl = list(flags) if flags is not None else [0] * len(layout)
    blob = b"".join(struct.pack("<QII", int(numel), int(tid), int(f))
                    for (numel, tid), f in zip(layout, fl))
    blob += struct.pack("<5I", dp_size, tp[0], tp[1], pp[0], pp[1])
    return dict(n=n, n_padded=L, total_numel=total, shard_begin=begin,
                segments=segments, layout_hash=fnv1a64(blob))


# ----------------------------------------------------------------------------
# D5: metadata envelope ("step index, parallelism configuration,
# RNG states"; reading R10) — 256-byte little-endian header
# ----------------------------------------------------------------------------

_HDR_FMT = "<8sIIQQQQQQQ6IQII128s"  # 240 bytes, then header_hash (Q) and seq_end (Q)
assert struct.calcsize(_HDR_FMT) == 240


def pack_header(*, step, n, n_padded, total_numel, shard_begin, layout_hash, dp, tp, pp,
                chunk_bytes, user=b"", committed=True, payload=0) -> bytes:
    """`payload` (the u32 after user_len): 0 = optimizer-only payload (the H2H payload);
    1 | elem_bytes << 8 = full rank state, the model-parameter buffer follows p ‖ m ‖ v
    (the D2H payload, reading R31 — see oracle/rank_state.py)."""
    assert len(user) <= 128
    body = struct.pack(_HDR_FMT, MAGIC, VERSION, HEADER_BYTES, step, step, n, n_padded,
                       total_numel, shard_begin, layout_hash, dp[0], dp[1], tp[0], tp[1],
                       pp[0], pp[1], chunk_bytes, len(user), payload, user.ljust(128, b"\0"))
    return body + struct.pack("<QQ", fnv1a64(body), step if committed else 0)


def parse_header(raw: bytes) -> Optional[dict]:
    """None unless magic/version/size are right, the header hash matches and
    seq_begin == seq_end (commit rule, reading R12 / SURVEY 8c-3)."""
    if len(raw) < HEADER_BYTES:
        return None
    f = struct.unpack(_HDR_FMT, raw[:240])
    hh, seq_end = struct.unpack("<QQ", raw[240:256])
    if f[0] != MAGIC or f[1] != VERSION or f[2] != HEADER_BYTES:
        return None
    if hh != fnv1a64(raw[:240]) or f[3] != seq_end:
        return None
    return dict(seq=f[3], step=f[4], n=f[5], n_padded=f[6], total_numel=f[7], shard_begin=f[8],
                layout_hash=f[9], dp=(f[10], f[11]), tp=(f[12], f[13]), pp=(f[14], f[15]),
                chunk_bytes=f[16], user=f[19][:f[17]], payload=f[18])


# ----------------------------------------------------------------------------
# The oracle shard: state + two replica slots
# ----------------------------------------------------------------------------


class OracleError(Exception):
    pass


class OracleShard:
    """Oracle state: p, m, v (fp32[n_padded]), p16 (bf16 bits), last_step, and two
    replica slots each `header ‖ p ‖ m ‖ v` (ping-pong)."""

    def __init__(self, layout, dp_size, dp_rank, tp=(1, 0), pp=(1, 0),
                 chunk_bytes=64 << 20, max_grad_norm=0.0, user=b"", flags=None, precision="bf16"):
        assert precision in ("bf16", "fp32")
        self.layout = [(int(a), int(b)) for a, b in layout]
        self.dp, self.tp, self.pp = (dp_size, dp_rank), tuple(tp), tuple(pp)
        self.precision = precision  # "fp32": binary32 gradients, no bf16 copy
        d = define_shard(self.layout, dp_size, dp_rank, tp, pp, flags)
        self.n, self.n_padded = d["n"], d["n_padded"]
        self.total_numel, self.shard_begin = d["total_numel"], d["shard_begin"]
        self.segments, self.layout_hash = d["segments"], d["layout_hash"]
        self.chunk_bytes = int(chunk_bytes)
        self.max_grad_norm = float(max_grad_norm)
        self.user = bytes(user)
        N = self.n_padded
        self.p = np.zeros(N, np.float32)
        self.m = np.zeros(N, np.float32)
        self.v = np.zeros(N, np.float32)
        self.p16 = np.zeros(N, np.uint16)
        self.last_step = 0
        self.snapshot_bytes = HEADER_BYTES + 12 * N
        self.replica = [np.zeros(self.snapshot_bytes, np.uint8) for _ in range(2)]
        self.last_coef = np.float32(1.0)
        # decay groups (reading R5b): one byte per element, 1 where the owning tensor is flagged no-decay
        self.no_decay = None
        if flags is not None and any(int(f) & TENSOR_NO_DECAY for f in flags):
            by_id = {tid: int(f) for (_, tid), f in zip(self.layout, flags)}
            self.no_decay = np.zeros(N, np.uint8)
            for tid, _, off, ln in self.segments:
                if by_id[tid] & TENSOR_NO_DECAY:
                    self.no_decay[off:off + ln] = 1

    # -- state ---------------------------------------------------------------
    def set_state(self, p, m=None, v=None, step=0):
        """Declare p, m, v as 'state after `step`' (init: step 0, m=v=0)."""
        self.p[:] = p
        self.m[:] = 0 if m is None else m
        self.v[:] = 0 if v is None else v
        self.p16[:] = rne_bf16(self.p) if self.precision == "bf16" else 0
        self.last_step = int(step)

    # -- a1 + a3 ---------------------------------------------------------------
    def step(self, g_bits: np.ndarray, lr, beta1, beta2, eps, wd, step, nthreads=1, coef=None):
        """One optimizer step; `step` is 1-based and must be last_step+1 (I4 step
        atomicity; reading R3).  `coef`: a clip coefficient decided outside
        the shard (the DP-global norm of oracle/global_clip.py); None = the
        shard-local rule of reading R7."""
        if int(step) != self.last_step + 1:
            raise OracleError("step order")
        g_bits = np.ascontiguousarray(g_bits, dtype=np.uint16 if self.precision == "bf16" else np.float32)
        if coef is not None:
            coef = np.float32(coef)
        elif self.max_grad_norm > 0.0:
            coef = clip_coef(sumsq(g_bits), self.max_grad_norm)
        else:
            coef = np.float32(1.0)
        self.last_coef = coef
        if self.precision == "bf16" and self.no_decay is None:
            adamw_step(self.p, self.m, self.v, g_bits, self.p16, lr, beta1, beta2, eps, wd,
                       step, float(coef), nthreads)
        else:  # fp32 gradients / no bf16 copy / decay groups
            adamw_step_ex(self.p, self.m, self.v, g_bits, self.p16 if self.precision == "bf16" else None,
                          self.no_decay, lr, beta1, beta2, eps, wd, step, float(coef), nthreads)
        self.last_step = int(step)

    # -- a4/a5: snapshot = byte copy of (header, p, m, v) after the step --------
    def _header(self, committed=True) -> bytes:
        return pack_header(step=self.last_step, n=self.n, n_padded=self.n_padded,
                           total_numel=self.total_numel, shard_begin=self.shard_begin,
                           layout_hash=self.layout_hash, dp=self.dp, tp=self.tp, pp=self.pp,
                           chunk_bytes=self.chunk_bytes, user=self.user, committed=committed)

    def packed_snapshot(self) -> np.ndarray:
        """The packed contiguous buffer: header ‖ p ‖ m ‖ v."""
        buf = np.empty(self.snapshot_bytes, np.uint8)
        buf[:HEADER_BYTES] = np.frombuffer(self._header(True), np.uint8)
        N4 = 4 * self.n_padded
        buf[HEADER_BYTES:HEADER_BYTES + N4] = self.p.view(np.uint8)
        buf[HEADER_BYTES + N4:HEADER_BYTES + 2 * N4] = self.m.view(np.uint8)
        buf[HEADER_BYTES + 2 * N4:] = self.v.view(np.uint8)
        return buf

    def snapshot(self, abort_after_chunks: Optional[int] = None) -> int:
        """Copy the packed snapshot into host slot (step mod 2) (ping-pong).
        The slot's header is invalidated first, the payload follows in chunk_bytes
        pieces, the valid header lands last (commit).  abort_after_chunks=j stops after
        j payload chunks and never commits: the slot stays torn."""
        slot = self.last_step % 2
        dst = self.replica[slot]
        src = self.packed_snapshot()
        dst[:HEADER_BYTES] = 0
        payload = self.snapshot_bytes - HEADER_BYTES
        nchunks = (payload + self.chunk_bytes - 1) // self.chunk_bytes
        for j in range(nchunks):
            if abort_after_chunks is not None and j >= abort_after_chunks:
                return slot
            lo = HEADER_BYTES + j * self.chunk_bytes
            hi = min(lo + self.chunk_bytes, self.snapshot_bytes)
            dst[lo:hi] = src[lo:hi]
        if abort_after_chunks is not None:
            return slot
        dst[:HEADER_BYTES] = src[:HEADER_BYTES]
        return slot

    # -- a6: restore -----------------------------------------------------------
    def newest_committed(self) -> Optional[Tuple[int, dict]]:
        best = None
        for s in range(2):
            h = parse_header(self.replica[s][:HEADER_BYTES].tobytes())
            if h is None:
                continue
            if best is None or h["step"] > best[1]["step"]:
                best = (s, h)
        return best

    def restore(self) -> int:
        """Choose the valid slot with the largest step, check logical identity
        (PAPER.md:250), copy p, m, v back, regenerate p16 = RNE(p), last_step = header.step."""
        best = self.newest_committed()
        if best is None:
            raise OracleError("no committed snapshot")
        s, h = best
        if (h["layout_hash"] != self.layout_hash or h["dp"] != self.dp or h["tp"] != self.tp
                or h["pp"] != self.pp or h["n_padded"] != self.n_padded or h["n"] != self.n):
            raise OracleError("layout mismatch")
        N4 = 4 * self.n_padded
        raw = self.replica[s]
        self.p[:] = raw[HEADER_BYTES:HEADER_BYTES + N4].view(np.float32)
        self.m[:] = raw[HEADER_BYTES + N4:HEADER_BYTES + 2 * N4].view(np.float32)
        self.v[:] = raw[HEADER_BYTES + 2 * N4:].view(np.float32)
        self.p16[:] = rne_bf16(self.p) if self.precision == "bf16" else 0
        self.last_step = h["step"]
        self.restored_user = h["user"]
        return self.last_step

    # -- a6 in two phases (reading R37) ---------------------------------
    # "Execution resumes from the last completed step": the recomputed iteration's
    # forward/backward reads only the model parameters; the moments are first read by its optimizer
    # step.  Phase 1 brings back p and regenerates p16 ("parameters ready"); phase 2 brings back m, v.
    # The state after both phases is the state after restore(); step() refuses to run in between.
    def restore_params_first(self) -> int:
        best = self.newest_committed()
        if best is None:
            raise OracleError("no committed snapshot")
        s, h = best
        if (h["layout_hash"] != self.layout_hash or h["dp"] != self.dp or h["tp"] != self.tp
                or h["pp"] != self.pp or h["n_padded"] != self.n_padded or h["n"] != self.n):
            raise OracleError("layout mismatch")
        N4 = 4 * self.n_padded
        self.p[:] = self.replica[s][HEADER_BYTES:HEADER_BYTES + N4].view(np.float32)
        self.p16[:] = rne_bf16(self.p) if self.precision == "bf16" else 0
        self._restoring = (s, h)
        self.last_step = -1          # no optimizer step may run until restore_finish()
        return h["step"]

    def restore_finish(self) -> int:
        s, h = self._restoring
        N4 = 4 * self.n_padded
        raw = self.replica[s]
        self.m[:] = raw[HEADER_BYTES + N4:HEADER_BYTES + 2 * N4].view(np.float32)
        self.v[:] = raw[HEADER_BYTES + 2 * N4:].view(np.float32)
        self.last_step = h["step"]
        self.restored_user = h["user"]
        self._restoring = None
        return self.last_step

    def drop_live(self):
        """'Drop the live shard' (BASELINE.json:configs[3], reading R16)."""
        self.p[:] = 0
        self.m[:] = 0
        self.v[:] = 0
        self.p16[:] = 0
