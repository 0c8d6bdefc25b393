"""Peer replication plumbing: received buffers, CUDA IPC handle exchange around
the data-parallel ring, binding.  Marshalling only — every byte is moved by libphx's copy-engine
flush (phx_snapshot_flush_peers_async) or restore (phx_restore_from); ring arithmetic is
phx_ring_peer.  torch.distributed is used for ONE control-plane exchange of 64-byte IPC handles at
set-up (the paper's control plane is a TCPStore); the data path has no collective.

One process per GPU (the ring peer is "the rank sharing the same tensor-parallel and
pipeline-parallel positions but with a different data-parallel index"):
    ring = PeerRing(shard, k, group=dp_group)      # allocates what this rank holds for its k
                                                   # predecessors, exchanges handles, opens and
                                                   # binds its k successors' buffers
    shard.step_and_snapshot(...); ring.flush_async(peer_stream); ...; ring.wait(step)
Single process (tests, the 1-GPU bench stand-in): connect_in_process([shard_0, .., shard_{D-1}], k)
wires D logical ranks living on one device to each other without IPC.
"""
from __future__ import annotations

from typing import List, Optional, Sequence

from . import binding as B


def successors(dp_size: int, dp_rank: int, k: int) -> List[int]:
    """Ranks that hold this rank's replicas: ring peers j = 1..k (phx_ring_peer)."""
    return [B.phx_ring_peer(dp_size, dp_rank, j) for j in range(1, k + 1)]


def predecessors(dp_size: int, dp_rank: int, k: int) -> List[int]:
    """Ranks whose replicas this rank holds: ring peers j = -1..-k."""
    return [B.phx_ring_peer(dp_size, dp_rank, -j) for j in range(1, k + 1)]


def placement(dp_size: int, k: int, domains: Optional[Sequence[int]] = None) -> List[List[int]]:
    """place[r] = the ranks that hold rank r's replicas: the plain ring (phx_ring_peer), or — `domains[q]` = the
    failure domain of rank q — the topology-aware placement of PAPER.md:187 (phx_ring_peers_topology_aware)."""
    if domains is None:
        return [successors(dp_size, r, k) for r in range(dp_size)]
    assert len(domains) == dp_size
    return [B.phx_ring_peers_topology_aware(dp_size, r, k, domains) for r in range(dp_size)]


def held_for(place: Sequence[Sequence[int]], h: int) -> List[int]:
    """The owners whose replicas rank h holds, in the order of h's received buffers: by ring distance from the
    owner to h (on the plain ring: predecessor 1, 2, .. k — buffer j-1 belongs to the j-th predecessor)."""
    D = len(place)
    return sorted((r for r in range(D) if h in place[r]), key=lambda r: (h - r) % D)


def route_handles(table: Sequence[Sequence[bytes]], place: Sequence[Sequence[int]], dp_rank: int) -> List[bytes]:
    """table[h][i] = handle of the buffer rank h keeps for held_for(place, h)[i] (gathered from all ranks).
    Returns the handles this rank must open, one per holder in place[dp_rank]."""
    return [table[h][held_for(place, h).index(dp_rank)] for h in place[dp_rank]]


class _Raw:
    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def device_view(ptr: int, nbytes: int):
    """Zero-copy uint8 torch view of a raw device address (memory owned by libphx allocations)."""
    import torch
    return torch.as_tensor(_Raw(ptr, nbytes), device="cuda")


class ReceivedBuffers:
    """The received buffers (two snapshot slots each) a rank keeps for the owners whose replicas it holds: its k ring
    predecessors, or held_for(place, rank) under a topology-aware placement (possibly none, possibly more than k)."""

    def __init__(self, slot_stride: int, k: int):
        self.slot_stride, self.k = slot_stride, k
        self.ptrs = [B.phx_peer_buffer_alloc(2 * slot_stride) for _ in range(k)]

    def handles(self) -> List[bytes]:
        return [B.phx_ipc_export(p) for p in self.ptrs]

    def view(self, j: int):
        """Zero-copy uint8 torch view of the buffer kept for predecessor j (1-based), for inspection."""
        return device_view(self.ptrs[j - 1], 2 * self.slot_stride)

    def inspect(self, j: int):
        """[(header, valid)] of the buffer kept for predecessor j (1-based)."""
        return B.phx_replica_inspect(self.ptrs[j - 1], self.slot_stride)

    def free(self):
        for p in self.ptrs:
            B.phx_peer_buffer_free(p)
        self.ptrs = []


class PeerRing:
    """One rank's end of the ring: its received buffers + its successors' buffers opened over IPC."""

    def __init__(self, shard, k: int, group=None, ring_size: Optional[int] = None, ring_rank: Optional[int] = None,
                 domains: Optional[Sequence[int]] = None):
        """group: the DP group of this shard.  ring_size / ring_rank override the ring the handles are routed
        on when only some of the D data-parallel ranks are present (e.g. N < D GPUs of one node in a
        benchmark): the ring then closes among the ranks of `group`.  domains[q] = failure domain of ring
        position q: the replicas go to the topology-aware placement instead of the ring successors."""
        import torch.distributed as dist
        self.shard, self.k = shard, k
        D = shard.info.dp_size if ring_size is None else ring_size
        r = shard.info.dp_rank if ring_rank is None else ring_rank
        assert dist.is_initialized() and dist.get_world_size(group) == D and dist.get_rank(group) == r, \
            "PeerRing needs one process per ring position"
        assert 1 <= k <= D - 1
        # every rank reaches both exchanges whatever happens locally, then all ranks agree on the outcome:
        # a rank whose allocation / IPC open failed must not leave the others waiting
        self.received, self.opened, err = None, [], None
        try:
            self.place = placement(D, k, domains)          # same inputs on every rank => the same table everywhere
            self.holds = held_for(self.place, r)
            self.received = ReceivedBuffers(shard.info.slot_stride, len(self.holds))
            mine = self.received.handles()
        except Exception as e:  # noqa: BLE001
            mine, err = None, repr(e)
        table: List[Optional[List[bytes]]] = [None] * D
        dist.all_gather_object(table, mine, group=group)
        if err is None and all(t is not None for t in table):
            try:
                self.opened = [B.phx_ipc_open(h) for h in route_handles(table, self.place, r)]
                B.phx_shard_bind_peers(shard.h, self.opened)
            except Exception as e:  # noqa: BLE001
                err = repr(e)
        elif err is None:
            err = "a peer could not allocate its received buffers"
        status: List[Optional[str]] = [None] * D
        dist.all_gather_object(status, err, group=group)
        if any(x is not None for x in status):
            self.close()
            raise RuntimeError("PeerRing set-up failed: " + "; ".join(f"rank {i}: {x}" for i, x in enumerate(status) if x))

    def flush_async(self, peer_stream):
        B.phx_snapshot_flush_peers_async(self.shard.h, peer_stream)

    def wait(self, step: int):
        B.phx_snapshot_wait_peers(self.shard.h, step)

    def close(self):
        if self.opened:
            B.phx_shard_bind_peers(self.shard.h, [])
        for p in self.opened:
            B.phx_ipc_close(p)
        self.opened = []
        if self.received is not None:
            self.received.free()
            self.received = None


class ParamBuffer:
    """A rank's model-parameter buffer W (dp_size * n_padded model-dtype elements), allocated so that it can be
    exported over CUDA IPC.  Allocate it BEFORE the Shard and hand `own_range()` to the Shard as its bf16 copy
    (`Shard(wl, p16=buf.own_range())`): the fused kernel then keeps the rank's own range of W current through
    d_p_bf16 and the rank's own buffer need not be bound as a publication target."""

    def __init__(self, wl):
        h = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank),
                               pp=(wl.pp_size, wl.pp_rank), flags=wl.flags(),
                               precision=B.PHX_PRECISION_FP32 if wl.precision == "fp32" else B.PHX_PRECISION_BF16_GRADS)
        info = B.phx_shard_info(h)
        B.phx_shard_destroy(h)
        self.fp32 = wl.precision == "fp32"
        self.n_padded, self.dp_size, self.dp_rank = info.n_padded, info.dp_size, info.dp_rank
        self.nbytes = info.param_bytes
        self.ptr = B.phx_peer_buffer_alloc(self.nbytes)

    def view(self):
        """Zero-copy torch view (model dtype) of W."""
        import torch
        return device_view(self.ptr, self.nbytes).view(torch.float32 if self.fp32 else torch.bfloat16)

    def own_range(self):
        """The rank's own range of W (for Shard(p16=...) in the bf16 precision)."""
        return self.view()[self.dp_rank * self.n_padded:(self.dp_rank + 1) * self.n_padded]

    def free(self):
        if self.ptr is not None:
            B.phx_peer_buffer_free(self.ptr)
            self.ptr = None


class ParamGroup:
    """one rank's end of the model-parameter publication.  Every rank of the DP group owns
    a model-parameter buffer W (dp_size * n_padded model-dtype elements, IPC-exportable); the others' buffers
    are opened over CUDA IPC and bound, so that the fused step kernel (PHX_PUBLISH_FUSED) or the copy engine
    (PHX_PUBLISH_COPY_ENGINE) writes this rank's range into all of them — the all-gather.

    `own`: a ParamBuffer the shard was built on (Shard(p16=own.own_range())): only the D-1 OTHER buffers are
    bound (D <= PHX_MAX_PARAM_PEERS + 1 = 16, no redundant local stores).  Without it (or in the all-FP32
    precision, where the kernel has no model-param copy of its own) the rank's W is allocated here and bound
    like a peer: D targets, D <= PHX_MAX_PARAM_PEERS."""

    def __init__(self, shard, mode=B.PHX_PUBLISH_FUSED, group=None, ring_size: Optional[int] = None,
                 ring_rank: Optional[int] = None, own: Optional[ParamBuffer] = None):
        import torch.distributed as dist
        self.shard = shard
        D = shard.info.dp_size if ring_size is None else ring_size
        r = shard.info.dp_rank if ring_rank is None else ring_rank
        assert dist.is_initialized() and dist.get_world_size(group) == D and dist.get_rank(group) == r
        elem = 4 if shard.fp32 else 2
        self.nbytes = shard.info.dp_size * shard.info.n_padded * elem
        self.own, self.opened, err = None, [], None
        self.owns_buffer = own is None
        in_place = (own is not None and not shard.fp32 and shard.p16 is not None
                    and shard.p16.data_ptr() == own.ptr + shard.info.dp_rank * shard.info.n_padded * 2)
        n_targets = (D - 1) if in_place else D
        if n_targets > B.PHX_MAX_PARAM_PEERS:
            err = (f"publication to {n_targets} buffers exceeds PHX_MAX_PARAM_PEERS = {B.PHX_MAX_PARAM_PEERS}"
                   + ("" if in_place else "; build the Shard on a ParamBuffer (own=) to need only dp_size - 1"))
        mine = None
        if err is None:
            try:
                self.own = own.ptr if own is not None else B.phx_peer_buffer_alloc(self.nbytes)
                mine = B.phx_ipc_export(self.own)
            except Exception as e:  # noqa: BLE001
                mine, err = None, repr(e)
        table: List[Optional[bytes]] = [None] * D
        dist.all_gather_object(table, mine, group=group)
        if err is None and all(t is not None for t in table):
            try:
                self.opened = [B.phx_ipc_open(table[j]) for j in range(D) if j != r]
                B.phx_shard_bind_param_peers(shard.h, ([] if in_place else [self.own]) + self.opened, mode)
            except Exception as e:  # noqa: BLE001
                err = repr(e)
        elif err is None:
            err = "a peer could not allocate its parameter buffer"
        status: List[Optional[str]] = [None] * D
        dist.all_gather_object(status, err, group=group)
        if any(x is not None for x in status):
            self.close()
            raise RuntimeError("ParamGroup set-up failed: " + "; ".join(f"rank {i}: {x}" for i, x in enumerate(status) if x))

    def publish_async(self, stream):
        B.phx_publish_params_async(self.shard.h, stream)

    def view(self):
        """Zero-copy torch view (model dtype) of this rank's parameter buffer W."""
        import torch
        t = device_view(self.own, self.nbytes)
        return t.view(torch.float32 if self.shard.fp32 else torch.bfloat16)

    def close(self):
        if self.opened:
            B.phx_shard_bind_param_peers(self.shard.h, [])
        for p in self.opened:
            B.phx_ipc_close(p)
        self.opened = []
        if self.own is not None and self.owns_buffer:
            B.phx_peer_buffer_free(self.own)
        self.own = None


def connect_in_process(shards: Sequence, k: int, domains: Optional[Sequence[int]] = None) -> List[ReceivedBuffers]:
    """D logical ranks in one process on one device: every rank gets a received buffer per owner it holds replicas
    for (held_for order; on the plain ring buffer j-1 belongs to the j-th predecessor), bound by plain device
    pointer (no IPC inside one process)."""
    D = len(shards)
    assert all(s.info.dp_size == D and s.info.dp_rank == r for r, s in enumerate(shards))
    place = placement(D, k, domains)
    holds = [held_for(place, h) for h in range(D)]
    recv = [ReceivedBuffers(s.info.slot_stride, len(holds[h])) for h, s in enumerate(shards)]
    for r, s in enumerate(shards):
        B.phx_shard_bind_peers(s.h, [recv[h].ptrs[holds[h].index(r)] for h in place[r]])
    return recv
