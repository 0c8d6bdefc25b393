"""CPU tier for the peer-replication plumbing: phx_ring_peer against the ring
oracle, argument errors of the peer entry points without a GPU, and the handle exchange on a
world_size-2 (and 3) gloo group with stand-in handles."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import ring as R
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import ring as PR


def test_ring_peer_matches_the_oracle_and_rejects_bad_arguments():
    for D in range(2, 10):
        for r in range(D):
            for j in list(range(1, D)) + [-x for x in range(1, D)]:
                assert B.phx_ring_peer(D, r, j) == R.ring_peer(D, r, j)
            for k in range(1, D):
                assert PR.successors(D, r, k) == R.holders(D, r, k)
                # rank r is the j-th successor of its j-th predecessor
                assert [PR.successors(D, h, k)[j] for j, h in enumerate(PR.predecessors(D, r, k))] == [r] * k
    L = B.lib()
    import ctypes as C
    out = C.c_uint32()
    for args in ((0, 0, 1), (4, 4, 1), (4, 0, 0), (4, 0, 4), (4, 0, -4), (1, 0, 1)):
        assert L.phx_ring_peer(*args, C.byref(out)) == B.PHX_ERR_INVALID_ARG, args
    assert L.phx_ring_peer(4, 0, 1, None) == B.PHX_ERR_INVALID_ARG


def test_peer_entry_points_fail_loudly_without_binding_or_gpu():
    L = B.lib()
    h = B.phx_shard_create([(100, 0)], 4, 0)
    import ctypes as C
    arr = (C.c_void_p * 1)(256)
    assert L.phx_shard_bind_peers(h, arr, 1) == B.PHX_ERR_NOT_BOUND
    assert L.phx_shard_bind_peers(h, arr, 5) == B.PHX_ERR_INVALID_ARG
    assert L.phx_snapshot_flush_peers_async(h, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_snapshot_wait_peers(h, 1) == B.PHX_ERR_NOT_BOUND
    assert L.phx_restore_from(h, None, None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_restore_from(h, 256, None, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_fault_inject_torn_peer_flush(h, 0, 1) == B.PHX_ERR_INVALID_ARG
    assert L.phx_fault_inject_torn_peer_flush(h, 5, 1) == B.PHX_ERR_INVALID_ARG
    assert L.phx_fault_inject_torn_peer_flush(h, 2, 1) == B.PHX_OK
    assert L.phx_replica_inspect(None, 512, None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_peer_buffer_alloc(0, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_ipc_export(None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_ipc_open(None, None) == B.PHX_ERR_INVALID_ARG
    if not torch.cuda.is_available():
        p = C.c_void_p()
        assert L.phx_peer_buffer_alloc(4096, C.byref(p)) in (B.PHX_ERR_NOMEM, B.PHX_ERR_CUDA)   # never a host stand-in
    B.phx_shard_destroy(h)


def test_topology_aware_placement_matches_the_oracle_on_every_domain_map():
    import ctypes as C
    import itertools
    from oracle import oracle as O
    L = B.lib()
    for D in range(2, 7):
        for domains in itertools.product(range(min(D, 4)), repeat=D):
            for k in range(1, min(D, 5)):
                for r in range(D):
                    try:
                        want = R.holders_topology_aware(domains, r, k)
                    except O.OracleError:
                        want = None
                    if want is None:
                        dom = (C.c_uint32 * D)(*domains)
                        out = (C.c_uint32 * k)()
                        assert L.phx_ring_peers_topology_aware(D, r, k, dom, out) == B.PHX_ERR_INVALID_ARG
                    else:
                        assert B.phx_ring_peers_topology_aware(D, r, k, domains) == want, (domains, r, k)
    # one rank per domain: the plain ring; held_for on the plain ring: predecessor 1, 2, .. k
    for D, k in ((3, 1), (5, 2), (6, 4)):
        assert PR.placement(D, k, list(range(D))) == PR.placement(D, k) == R.placement(D, k)
        for h in range(D):
            assert PR.held_for(PR.placement(D, k), h) == PR.predecessors(D, h, k)
    dom = (C.c_uint32 * 4)(0, 0, 1, 1)
    out = (C.c_uint32 * 4)()
    for args in ((0, 0, 1, dom, out), (4, 4, 1, dom, out), (4, 0, 4, dom, out), (4, 0, 1, None, out), (4, 0, 1, dom, None)):
        assert L.phx_ring_peers_topology_aware(*args) == B.PHX_ERR_INVALID_ARG, args[:3]
    assert L.phx_ring_peers_topology_aware(4, 0, 0, dom, None) == B.PHX_OK


def _worker(rank, world, k, port, q, domains=None):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo")
    place = PR.placement(world, k, domains)
    # stand-in handles: 64 bytes that name (holder, buffer index); one buffer per owner this rank holds replicas for
    mine = [bytes([rank, j]) + b"\0" * 62 for j in range(len(PR.held_for(place, rank)))]
    table = [None] * world
    dist.all_gather_object(table, mine)
    got = PR.route_handles(table, place, rank)
    q.put((rank, [(h[0], h[1]) for h in got]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,k", [(2, 1), (3, 2)])
def test_handle_exchange_on_gloo(world, k):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29800 + (os.getpid() + 7 * world) % 150
    ps = [ctx.Process(target=_worker, args=(r, world, k, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        # rank r must open, for j = 1..k, the buffer number j-1 of its j-th ring successor — exactly the
        # buffers the ring oracle's replicate() writes
        assert res[r] == [(R.ring_peer(world, r, j), j - 1) for j in range(1, k + 1)]


def test_handle_exchange_with_a_topology_aware_placement_on_gloo():
    world, k, domains = 4, 1, [0, 0, 1, 1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29960 + os.getpid() % 30
    ps = [ctx.Process(target=_worker, args=(r, world, k, port, q, domains)) for r in range(world)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    place = R.placement(world, k, domains)
    assert place == [[2], [2], [0], [0]]
    # rank 2 holds for owners 1 (distance 1) and 0 (distance 2) in that order; rank 0 for owners 3 and 2
    assert res == {0: [(2, 1)], 1: [(2, 0)], 2: [(0, 1)], 3: [(0, 0)]}
