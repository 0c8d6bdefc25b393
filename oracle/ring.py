"""ring.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

CPU oracle of SURVEY.md §8(f1): peer replication of the optimizer-state shard around the
data-parallel ring (§V-B b "Host-to-host"), the peer-side ping-pong
"receiving / committed" buffers (Fig. 5, 224), k-peer replication
 and recovery of a lost shard from a surviving replica holder
(PAPER.md:171 stage 3, 248-250).  Plain byte copies between numpy buffers, one rank at a
time; it shares no code with paper_2607_01646_b200/.

Readings (R25-R28):
  R25  ring peer j of rank r (j = 1..k) is (r + j) mod D — "the rank sharing the same
       tensor-parallel and pipeline-parallel positions but with a different data-parallel
       index", "in a ring topology"; k distinct peers need k <= D - 1.
  R26  the H2H payload is the packed optimizer snapshot: envelope ‖ p ‖ m ‖ v, no model
       parameters — byte-identical to the local snapshot slot.
  R27  the buffer a rank holds for predecessor (r - j) mod D has two slots; the snapshot of
       step s lands in slot s mod 2 with the same protocol as the local pair: header
       invalidated, payload in chunks, valid header last ("follows the same alternation
       logic").
  R28  a shard is lost only if its owner and all k holders fail within the same step
       (PAPER.md:175); recovery takes the valid slot with the largest step among the
       surviving holders (and the owner's own local replica if the owner survived).

Pins (tests/test_oracle_ring.py): brute force over every failure subset for small D, k
against R28 and against the paper's Eq. (1) P_loss <= D p^(k+1) evaluated in
exact rationals, and the paper's printed value 1.28e-10 for D = 128, k = 1, p = 1e-6
(PAPER.md:181); byte identity of received slots with the owner's local slots; the torn-slot
and resume invariants of the single-rank oracle carried over to the ring.
"""
from __future__ import annotations

from typing import Dict, Iterable, List, Optional, Sequence, Tuple

import numpy as np

from . import oracle as O


def ring_peer(dp_size: int, dp_rank: int, j: int) -> int:
    """R25: the j-th ring successor of rank r (j >= 1); j = -1, -2.. gives predecessors."""
    assert dp_size >= 1 and 0 <= dp_rank < dp_size and j != 0 and abs(j) <= dp_size - 1
    return (dp_rank + j) % dp_size


def holders(dp_size: int, dp_rank: int, k: int) -> List[int]:
    """Ranks that hold a replica of rank r's shard (k distinct ring successors)."""
    assert 0 <= k <= dp_size - 1
    return [ring_peer(dp_size, dp_rank, j) for j in range(1, k + 1)]


def recoverable(dp_size: int, k: int, failed: Iterable[int]) -> bool:
    """R28 as a predicate on a set of ranks that failed within one step."""
    f = set(failed)
    return all(any(h not in f for h in holders(dp_size, r, k)) for r in f)


# ---- topology-aware placement (reading R38) ------------------------------------------------------
# "PHOENIX can leverage cluster topology information to place the k replicas on nodes under k distinct
# switches or racks, ensuring that a single infrastructure event affects at most one copy of any given
# shard".  A shard has k + 1 copies (the owner's and the k replicas), so all k + 1 must sit
# in pairwise distinct failure domains.  The paper does not say WHICH ranks are taken; R38: walk the DP
# ring from the owner (r+1, r+2, ...) and take a rank iff its domain differs from the owner's and from the
# domain of every rank already taken — the nearest admissible ranks in ring order.


def holders_topology_aware(domains: Sequence[int], dp_rank: int, k: int) -> List[int]:
    D = len(domains)
    assert 0 <= dp_rank < D and 0 <= k <= D - 1
    used = {domains[dp_rank]}
    out: List[int] = []
    for j in range(1, D):
        if len(out) == k:
            break
        q = (dp_rank + j) % D
        if domains[q] not in used:
            used.add(domains[q])
            out.append(q)
    if len(out) < k:
        raise O.OracleError("fewer than k + 1 distinct failure domains")
    return out


def placement(dp_size: int, k: int, domains: Optional[Sequence[int]] = None) -> List[List[int]]:
    """place[r] = the ranks that hold rank r's replicas: the plain ring (R25) or, with failure domains, R38."""
    if domains is None:
        return [holders(dp_size, r, k) for r in range(dp_size)]
    assert len(domains) == dp_size
    return [holders_topology_aware(domains, r, k) for r in range(dp_size)]


def recoverable_with(place: Sequence[Sequence[int]], failed: Iterable[int]) -> bool:
    """R28 for an arbitrary placement."""
    f = set(failed)
    return all(any(h not in f for h in place[r]) for r in f)


def max_copies_in_one_domain(domains: Sequence[int], place: Sequence[Sequence[int]]) -> int:
    """The largest number of copies (owner's + replicas) of any one shard that share a failure domain."""
    worst = 0
    for r, hs in enumerate(place):
        doms = [domains[r]] + [domains[h] for h in hs]
        worst = max(worst, max(doms.count(d) for d in set(doms)))
    return worst


class OracleRing:
    """D OracleShards of one DP group (same layout, tp/pp coordinates; dp_rank = 0..D-1) plus, on every
    rank, the received buffers it holds for the ranks whose replicas are placed on it: the k ring
    predecessors (plain ring), or whoever the topology-aware placement R38 sends there (`domains`)."""

    def __init__(self, layout, dp_size: int, k: int, *, tp=(1, 0), pp=(1, 0), chunk_bytes=64 << 20,
                 flags=None, precision="bf16", max_grad_norm=0.0, domains: Optional[Sequence[int]] = None):
        assert 1 <= k <= dp_size - 1
        self.D, self.k = dp_size, k
        self.domains = None if domains is None else list(domains)
        self.place = placement(dp_size, k, self.domains)
        self.shards = [O.OracleShard(layout, dp_size, r, tp, pp, chunk_bytes=chunk_bytes, flags=flags,
                                     precision=precision, max_grad_norm=max_grad_norm) for r in range(dp_size)]
        nbytes = self.shards[0].snapshot_bytes
        # recv[(h, r)][slot]: what rank h holds for owner r
        self.recv: Dict[Tuple[int, int], List[np.ndarray]] = {
            (h, r): [np.zeros(nbytes, np.uint8) for _ in range(2)] for r in range(dp_size) for h in self.place[r]}
        self.alive = [True] * dp_size

    @property
    def received(self) -> List[List[List[np.ndarray]]]:
        """Plain ring only: received[h][j-1][slot] = what rank h holds for its j-th predecessor (h - j) mod D."""
        assert self.domains is None
        return [[self.recv[(h, ring_peer(self.D, h, -j))] for j in range(1, self.k + 1)] for h in range(self.D)]

    # -- H2H phase: owner r -> its k holders (R26, R27) ---------------------------------------
    def replicate(self, r: int, abort_after_chunks: Optional[Dict[int, int]] = None):
        """Send rank r's packed snapshot of its last step to every holder.  abort_after_chunks[j]
        = c tears the transfer to holder number j (1-based) after c payload chunks (never commits)."""
        o = self.shards[r]
        src = o.packed_snapshot()
        slot = o.last_step % 2
        cb = o.chunk_bytes
        payload = o.snapshot_bytes - O.HEADER_BYTES
        nchunks = (payload + cb - 1) // cb
        for j, h in enumerate(self.place[r], 1):
            if not self.alive[h]:
                continue
            dst = self.recv[(h, r)][slot]
            stop = None if abort_after_chunks is None else abort_after_chunks.get(j)
            dst[:O.HEADER_BYTES] = 0
            for c in range(nchunks):
                if stop is not None and c >= stop:
                    break
                lo = O.HEADER_BYTES + c * cb
                hi = min(lo + cb, o.snapshot_bytes)
                dst[lo:hi] = src[lo:hi]
            if stop is None:
                dst[:O.HEADER_BYTES] = src[:O.HEADER_BYTES]

    # -- failures (R16 on a whole node: live state, local replica and every buffer it holds) ---
    def fail(self, ranks: Iterable[int]):
        for r in ranks:
            self.alive[r] = False
            o = self.shards[r]
            o.drop_live()
            for s in range(2):
                o.replica[s][:] = 0
            for (h, _), bufs in self.recv.items():
                if h == r:
                    for s in range(2):
                        bufs[s][:] = 0xA5

    # -- recovery stage 3 for one lost shard (R28) ---------------------
    def newest_replica_of(self, r: int) -> Optional[Tuple[int, int, int, dict]]:
        """(holder, j, slot, header) of the valid, identity-matching slot with the largest step
        among surviving holders of rank r's shard (j = the holder's 1-based number), or None."""
        o = self.shards[r]
        best = None
        for j, h in enumerate(self.place[r], 1):
            if not self.alive[h]:
                continue
            for s in range(2):
                hd = O.parse_header(self.recv[(h, r)][s][:O.HEADER_BYTES].tobytes())
                if hd is None:
                    continue
                if (hd["layout_hash"] != o.layout_hash or hd["dp"] != o.dp or hd["tp"] != o.tp
                        or hd["pp"] != o.pp or hd["n"] != o.n or hd["n_padded"] != o.n_padded):
                    continue
                if best is None or hd["step"] > best[3]["step"]:
                    best = (h, j, s, hd)
        return best

    def recover(self, r: int) -> int:
        """A replacement node assumes rank r's role: pull the newest replica from a
        surviving holder into the live shard; the rank is alive again, its local replica and the
        buffers it holds start empty."""
        best = self.newest_replica_of(r)
        if best is None:
            raise O.OracleError("shard lost: owner and all holders failed (PAPER.md:175)")
        h, j, s, hd = best
        o = self.shards[r]
        o.replica[hd["step"] % 2][:] = self.recv[(h, r)][s]   # same bytes, then the plain restore
        o.replica[1 - hd["step"] % 2][:] = 0
        step = o.restore()
        for (hh, _), bufs in self.recv.items():
            if hh == r:
                for ss in range(2):
                    bufs[ss][:] = 0
        self.alive[r] = True
        return step


# ---- model-parameter publication and reconstruction ---------------------------
#
# In a ZeRO-2 distributed optimizer every DP rank of one TP/PP coordinate holds the SAME
# model parameters for that partition; after the step each rank has updated only its 1/D range of the
# flat space and the ranges are all-gathered.  Readings:
#   R29  the model-parameter buffer W of a TP/PP partition is the flat padded space of a0 in the model
#        dtype: W[r*L : (r+1)*L] = rank r's model-parameter copy (bf16: RNE_bf16(p_r); all-FP32 precision:
#        p_r itself), L = n_padded.  Publication = concatenation in rank order (an all-gather).
#   R30  on a permanent failure the replacement "can reconstruct its parameter shard from healthy ranks
#        at the same TP/PP coordinate via a targeted collective" (171, 248): W is copied
#        whole from any surviving DP rank of the same partition — they are byte-identical (I2).


def publish(shards) -> np.ndarray:
    """R29: the model-parameter buffer every DP rank holds after the step (uint16 bf16 bits, or float32)."""
    if shards[0].precision == "fp32":
        return np.concatenate([o.p for o in shards])
    return np.concatenate([o.p16 for o in shards])


def reconstruct_params(buffers, alive, r: int) -> np.ndarray:
    """R30: rank r's replacement takes W from the first surviving rank of the partition (ring order)."""
    D = len(buffers)
    for j in range(1, D):
        h = (r + j) % D
        if alive[h]:
            return buffers[h].copy()
    raise O.OracleError("no surviving rank holds the partition's parameters")


def p_loss_exact(dp_size: int, k: int, p):
    """Exact probability (any numeric type, e.g. Fraction) that some shard is unrecoverable when every
    rank fails independently with probability p within a step — brute force over all failure subsets."""
    total = 0
    for mask in range(1 << dp_size):
        failed = [r for r in range(dp_size) if mask >> r & 1]
        if not recoverable(dp_size, k, failed):
            total = total + p ** len(failed) * (1 - p) ** (dp_size - len(failed))
    return total
