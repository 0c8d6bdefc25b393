"""rank_state.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

CPU oracle of SURVEY.md §8(f4): the FULL RANK STATE local snapshot — "the optimizer-state shard,
the local model-parameter shard, and a metadata envelope (step index, parallelism configuration,
RNG states) ... packed into a contiguous buffer and copied asynchronously to pinned host memory
... Retaining the complete rank state on the host enables fast local recovery (e.g., after a
transient GPU error) without any network transfer" (§V-B a) — and the in-place
recovery it enables (PAPER.md:160 transient failures, 230 "local reset by clearing the node's
state and reinitializing it").  The payload is asymmetric: the ring peer still
receives the optimizer-only snapshot of oracle/ring.py.  Plain byte copies between numpy buffers;
it shares no code with paper_2607_01646_b200/.

Readings (R31-R33):
  R31  "local model-parameter shard" = the model-parameter buffer W the rank holds for its TP/PP
       partition (R29: the flat padded space of a0 in the model dtype, dp_size * n_padded elements,
       bf16 — or float32 in the all-FP32 precision).  The full rank state is
           header(256 B, payload = 1 | elem_bytes << 8) ‖ p ‖ m ‖ v ‖ W
       i.e. the optimizer-only snapshot with W appended, so the optimizer part sits at the same
       offsets in both payloads.  W in the snapshot of step k is W after the all-gather of step k.
  R32  transfer order of the local flush: header invalidated, W in chunk_bytes pieces, then
       p ‖ m ‖ v in chunk_bytes pieces, valid header last.  (W first: W is the part other ranks
       overwrite at the next publication, so its window of exposure is the shortest possible.)
  R33  in-place recovery: the rank's p, m, v, W are rebuilt from its OWN host slot — the valid,
       identity-matching slot with the largest step — and nothing is read from any other rank;
       last_step = header.step; the rank's own range of W equals RNE_bf16(p) (or p) again.

Pins (tests/test_oracle_rank_state.py): W against the rank-order all-gather of torch's bf16 cast;
the optimizer part byte-identical to the optimizer-only snapshot and the header differing from it
in the payload word and the hash only; restore == state bit for bit with every other rank's
memory poisoned; torn flush (in W or in p ‖ m ‖ v) never chosen; resume == uninterrupted.
"""
from __future__ import annotations

from typing import Optional

import numpy as np

from . import oracle as O

PAYLOAD_OPTIMIZER = 0
PAYLOAD_FULL = 1


def payload_word(elem_bytes: int) -> int:
    """R31: the envelope's payload word for a full rank state."""
    assert elem_bytes in (2, 4)
    return PAYLOAD_FULL | (elem_bytes << 8)


class FullRankState:
    """One rank: its OracleShard (p, m, v, own model-param copy) + its model-parameter buffer W
    + two local host slots holding the full rank state (ping-pong)."""

    def __init__(self, shard: O.OracleShard):
        self.o = shard
        self.D = shard.dp[0]
        self.r = shard.dp[1]
        self.elem_bytes = 4 if shard.precision == "fp32" else 2
        self.wdtype = np.float32 if shard.precision == "fp32" else np.uint16
        N = shard.n_padded
        self.W = np.zeros(self.D * N, self.wdtype)
        self.w_bytes = self.D * N * self.elem_bytes
        self.snapshot_bytes = O.HEADER_BYTES + 12 * N + self.w_bytes
        self.slots = [np.zeros(self.snapshot_bytes, np.uint8) for _ in range(2)]

    # -- the rank's own range of W is its model-param copy (R29) -----------------------------------
    def own_range(self) -> np.ndarray:
        N = self.o.n_padded
        return self.W[self.r * N:(self.r + 1) * N]

    def write_own_range(self):
        self.own_range()[:] = self.o.p if self.o.precision == "fp32" else self.o.p16

    # -- R31: the packed full rank state ----------------------------------------------------------
    def _header(self, committed=True) -> bytes:
        o = self.o
        return O.pack_header(step=o.last_step, n=o.n, n_padded=o.n_padded, total_numel=o.total_numel,
                             shard_begin=o.shard_begin, layout_hash=o.layout_hash, dp=o.dp, tp=o.tp, pp=o.pp,
                             chunk_bytes=o.chunk_bytes, user=o.user, committed=committed,
                             payload=payload_word(self.elem_bytes))

    def packed(self) -> np.ndarray:
        o = self.o
        N4 = 4 * o.n_padded
        buf = np.empty(self.snapshot_bytes, np.uint8)
        H = O.HEADER_BYTES
        buf[:H] = np.frombuffer(self._header(True), np.uint8)
        buf[H:H + N4] = o.p.view(np.uint8)
        buf[H + N4:H + 2 * N4] = o.m.view(np.uint8)
        buf[H + 2 * N4:H + 3 * N4] = o.v.view(np.uint8)
        buf[H + 3 * N4:] = self.W.view(np.uint8)
        return buf

    # -- R32: the local flush ---------------------------------------------------------------------
    def snapshot(self, abort_after_chunks: Optional[int] = None) -> int:
        """Copy the full rank state into local slot (step mod 2).  abort_after_chunks = j stops after j
        chunks in TRANSFER order (W chunks first, then p ‖ m ‖ v chunks) and never commits."""
        o = self.o
        slot = o.last_step % 2
        dst, src = self.slots[slot], self.packed()
        H, cb = O.HEADER_BYTES, o.chunk_bytes
        dst[:H] = 0
        w0 = H + 12 * o.n_padded
        regions = [(w0, self.snapshot_bytes), (H, w0)]          # W, then the optimizer part
        done = 0
        for lo_r, hi_r in regions:
            for lo in range(lo_r, hi_r, cb):
                if abort_after_chunks is not None and done >= abort_after_chunks:
                    return slot
                hi = min(lo + cb, hi_r)
                dst[lo:hi] = src[lo:hi]
                done += 1
        if abort_after_chunks is not None:
            return slot
        dst[:H] = src[:H]
        return slot

    # -- R33: in-place recovery -------------------------------------------------------------------
    def newest_committed(self):
        best = None
        o = self.o
        for s in range(2):
            h = O.parse_header(self.slots[s][:O.HEADER_BYTES].tobytes())
            if h is None or h["payload"] != payload_word(self.elem_bytes):
                continue
            if (h["layout_hash"] != o.layout_hash or h["dp"] != o.dp or h["tp"] != o.tp or h["pp"] != o.pp
                    or h["n"] != o.n or h["n_padded"] != o.n_padded):
                continue
            if best is None or h["step"] > best[1]["step"]:
                best = (s, h)
        return best

    def drop_live(self):
        """Transient GPU fault followed by a local reset: everything device-resident is gone."""
        self.o.drop_live()
        self.W[:] = 0

    def restore_in_place(self) -> int:
        best = self.newest_committed()
        if best is None:
            raise O.OracleError("no committed full rank state in the local slots")
        s, h = best
        o = self.o
        raw = self.slots[s]
        H, N4 = O.HEADER_BYTES, 4 * o.n_padded
        o.p[:] = raw[H:H + N4].view(np.float32)
        o.m[:] = raw[H + N4:H + 2 * N4].view(np.float32)
        o.v[:] = raw[H + 2 * N4:H + 3 * N4].view(np.float32)
        self.W[:] = raw[H + 3 * N4:].view(self.wdtype)
        o.p16[:] = O.rne_bf16(o.p) if o.precision == "bf16" else 0
        o.last_step = h["step"]
        o.restored_user = h["user"]
        return o.last_step

    # -- R33 in two phases (reading R37): the parameters first, the optimizer state second.  For a full
    # rank state "the parameters" are W itself — the forward/backward of the recomputed iteration reads W and nothing
    # else; the rank's own range of W (its model-param copy, R29) is part of the snapshot's W — so phase 1 is W
    # ALONE and the fp32 master p comes back in phase 2 with the moments.
    def restore_in_place_params_first(self) -> int:
        best = self.newest_committed()
        if best is None:
            raise O.OracleError("no committed full rank state in the local slots")
        s, h = best
        o = self.o
        raw = self.slots[s]
        H, N4 = O.HEADER_BYTES, 4 * o.n_padded
        self.W[:] = raw[H + 3 * N4:].view(self.wdtype)
        if o.precision == "bf16":
            o.p16[:] = self.own_range()            # the model-param copy IS the rank's range of W
        self._restoring = (s, h)
        o.last_step = -1
        return h["step"]

    def restore_in_place_finish(self) -> int:
        s, h = self._restoring
        o = self.o
        raw = self.slots[s]
        H, N4 = O.HEADER_BYTES, 4 * o.n_padded
        o.p[:] = raw[H:H + N4].view(np.float32)
        o.m[:] = raw[H + N4:H + 2 * N4].view(np.float32)
        o.v[:] = raw[H + 2 * N4:H + 3 * N4].view(np.float32)
        o.last_step = h["step"]
        o.restored_user = h["user"]
        self._restoring = None
        return o.last_step
