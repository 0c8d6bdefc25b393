"""GPU parity for SURVEY.md §8(f1): peer replication around the DP ring through the C ABI against
the ring oracle — received buffers byte-identical, recovery from a surviving holder bit-exact,
torn peer transfers never chosen.  One GPU: D logical ranks live in one process (their kernels
never wait on one another; each rank's work is plain stream-ordered), and a two-process test
exercises the CUDA IPC path on the same device."""
import os

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from oracle import oracle as O
from oracle import ring as R
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import ring as PR
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, assert_state_equal, bits16, grad_record, hp_of

pytestmark = pytest.mark.gpu


def build_ring(numels, D, k, *, chunk=8192, domains=None, **shard_kw):
    """D Shards (one per DP rank) wired in process + the ring oracle, equal initial state, per-rank grads."""
    wls = [W.tiny_workload(numels, dp_size=D, dp_rank=r) for r in range(D)]
    shards = [Shard(wl, device=DEV, chunk_bytes=chunk, **shard_kw) for wl in wls]
    recv = PR.connect_in_process(shards, k, domains)
    oring = R.OracleRing(wls[0].layout(), D, k, chunk_bytes=(chunk + 255) & ~255, domains=domains)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        p0 = W.init_params(s.n, s.n_padded, seed=100 + r)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
    return wls, shards, recv, oring


def grads_for(wls, shards, t):
    return [W.gen_grads(wl, s.segments, s.n_padded, t, seed=7 + r) for r, (wl, s) in enumerate(zip(wls, shards))]


def step_all(wls, shards, oring, t, streams, flush_host=True, flush_peers=True):
    gs = grads_for(wls, shards, t)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        s.step_and_snapshot(gs[r].to(DEV), t)
        if flush_host:
            s.flush_async(streams[0])
        if flush_peers:
            B.phx_snapshot_flush_peers_async(s.h, streams[1])
        o.step(grad_record(gs[r]), **hp_of(wls[r]), step=t)
        o.snapshot()
        if flush_peers:
            oring.replicate(r)
    return gs


def received_bytes(recv, h, j, slot, shard):
    st, nb = shard.info.slot_stride, shard.info.snapshot_bytes
    return recv[h].view(j)[slot * st: slot * st + nb].cpu().numpy()


@pytest.mark.parametrize("D,k", [(2, 1), (3, 2), (5, 4)])
@pytest.mark.parametrize("numels", [[64], [5000, 77, 2048 * 3]])
def test_received_buffers_equal_the_oracle_rings(D, k, numels):
    wls, shards, recv, oring = build_ring(numels, D, k)
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    for t in range(1, 4):
        step_all(wls, shards, oring, t, streams)
    for s in shards:
        B.phx_snapshot_wait_peers(s.h, 3)
        s.wait(3)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        assert_state_equal(s, o, f"rank {r}")
        for j in range(1, k + 1):
            h = B.phx_ring_peer(D, r, j)
            for slot in (0, 1):
                assert np.array_equal(received_bytes(recv, h, j, slot, s), oring.received[h][j - 1][slot]), (r, j, slot)
            assert np.array_equal(received_bytes(recv, h, j, 1, s), s.replica_slot(3).numpy())       # R26
            (h0, v0), (h1, v1) = recv[h].inspect(j)
            assert v0 and v1 and (h0.step, h1.step) == (2, 3) and h1.dp_rank == r and h1.layout_hash == s.info.layout_hash
    for s in shards:
        s.close()
    for rb in recv:
        rb.free()


@pytest.mark.parametrize("rmode", [B.PHX_RESTORE_COPY_ENGINE, B.PHX_RESTORE_BULK_KERNEL])
@pytest.mark.parametrize("failed", [(1,), (0, 1), (3, 0)])
def test_recovery_from_a_surviving_holder_resumes_bit_exactly(failed, rmode):
    D, k = 4, 2
    wls, shards, recv, oring = build_ring([30_000, 123], D, k, restore_mode=rmode)
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    for t in range(1, 6):
        step_all(wls, shards, oring, t, streams)
    g6 = grads_for(wls, shards, 6)
    for r in failed:                                     # step 6 in flight on the nodes that die
        shards[r].step_and_snapshot(g6[r].to(DEV), 6)
        oring.shards[r].step(grad_record(g6[r]), **hp_of(wls[r]), step=6)
    torch.cuda.synchronize()
    oring.fail(failed)
    for r in failed:                                     # the node is gone: live state, local replica, what it held
        shards[r].close()
        for j in range(1, k + 1):
            recv[r].view(j).fill_(0xA5)
    for r in failed:
        # a replacement node assumes rank r's role: fresh handle, fresh memory, no local replica
        fresh = Shard(wls[r], device=DEV, chunk_bytes=8192, restore_mode=rmode)
        holder, j, slot, hd = oring.newest_replica_of(r)
        (ha, va), (hb, vb) = recv[holder].inspect(j)
        assert (va and ha.step == hd["step"]) or (vb and hb.step == hd["step"])
        assert B.phx_restore_from(fresh.h, recv[holder].ptrs[j - 1]) == 5 == oring.recover(r)
        shards[r] = fresh
        assert_state_equal(fresh, oring.shards[r], f"restored rank {r}")
    recv2 = PR.connect_in_process(shards, k)             # topology re-established (PAPER.md:171 stage 2)
    for t in (6, 7):
        gs = grads_for(wls, shards, t)
        for r, (s, o) in enumerate(zip(shards, oring.shards)):
            if o.last_step == t - 1:
                s.step_and_snapshot(gs[r].to(DEV), t)
                B.phx_snapshot_flush_peers_async(s.h, streams[1])
                o.step(grad_record(gs[r]), **hp_of(wls[r]), step=t)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        assert_state_equal(s, o, f"resumed rank {r}")
        B.phx_snapshot_wait_peers(s.h, 7)
        s.close()
    for rb in recv + recv2:
        rb.free()


@pytest.mark.parametrize("D,k,domains,dead", [(4, 1, [0, 0, 1, 1], 0), (6, 2, [0, 0, 1, 1, 2, 2], 1),
                                              (5, 2, [7, 3, 3, 7, 9], 3)])
def test_topology_aware_placement_survives_a_whole_failed_domain(D, k, domains, dead):
    """PAPER.md:187 (R38): the k + 1 copies of every shard sit under distinct failure domains; the received
    buffers — irregular now: some ranks hold for several owners, some for none — are byte-identical to the oracle's,
    and after ALL ranks of one domain die every lost shard comes back from a surviving holder and resumes bit-exactly."""
    wls, shards, recv, oring = build_ring([20_000, 77], D, k, domains=domains)
    place = PR.placement(D, k, domains)
    assert place == oring.place and R.max_copies_in_one_domain(domains, place) == 1
    holds = [PR.held_for(place, h) for h in range(D)]
    assert [len(rb.ptrs) for rb in recv] == [len(x) for x in holds]
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    for t in range(1, 5):
        step_all(wls, shards, oring, t, streams)
    for s in shards:
        B.phx_snapshot_wait_peers(s.h, 4)
    for r, s in enumerate(shards):
        for h in place[r]:
            j = holds[h].index(r) + 1
            for slot in (0, 1):
                assert np.array_equal(received_bytes(recv, h, j, slot, s), oring.recv[(h, r)][slot]), (r, h, slot)
    failed = [q for q in range(D) if domains[q] == domains[dead]]
    g5 = grads_for(wls, shards, 5)
    for r in failed:                                     # step 5 in flight on the nodes that die with their switch
        shards[r].step_and_snapshot(g5[r].to(DEV), 5)
        oring.shards[r].step(grad_record(g5[r]), **hp_of(wls[r]), step=5)
    torch.cuda.synchronize()
    oring.fail(failed)
    for r in failed:
        shards[r].close()
        for j in range(1, len(holds[r]) + 1):
            recv[r].view(j).fill_(0xA5)
    for r in failed:
        fresh = Shard(wls[r], device=DEV, chunk_bytes=8192)
        holder, _, _, hd = oring.newest_replica_of(r)
        assert holder not in failed
        assert B.phx_restore_from(fresh.h, recv[holder].ptrs[holds[holder].index(r)]) == 4 == oring.recover(r)
        shards[r] = fresh
        assert_state_equal(fresh, oring.shards[r], f"restored rank {r}")
    recv2 = PR.connect_in_process(shards, k, domains)    # topology re-established (PAPER.md:171 stage 2)
    for t in (5, 6):
        gs = grads_for(wls, shards, t)
        for r, (s, o) in enumerate(zip(shards, oring.shards)):
            if o.last_step == t - 1:
                s.step_and_snapshot(gs[r].to(DEV), t)
                B.phx_snapshot_flush_peers_async(s.h, streams[1])
                o.step(grad_record(gs[r]), **hp_of(wls[r]), step=t)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        assert_state_equal(s, o, f"resumed rank {r}")
        B.phx_snapshot_wait_peers(s.h, 6)
        s.close()
    for rb in recv + recv2:
        rb.free()


def test_torn_peer_transfer_is_never_chosen_and_other_holder_has_the_newer_step():
    D, k = 3, 2
    wls, shards, recv, oring = build_ring([20_000], D, k, chunk=4096)
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    step_all(wls, shards, oring, 1, streams)
    gs = grads_for(wls, shards, 2)
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        s.step_and_snapshot(gs[r].to(DEV), 2)
        o.step(grad_record(gs[r]), **hp_of(wls[r]), step=2)
        o.snapshot()
    B.phx_fault_inject_torn_peer_flush(shards[0].h, 1, 2)       # rank 0 -> peer 1 torn after 2 chunks
    oring.replicate(0, abort_after_chunks={1: 2})
    for r in (1, 2):
        oring.replicate(r)
    for s in shards:
        B.phx_snapshot_flush_peers_async(s.h, streams[1])
    with pytest.raises(B.PhxError) as e:
        B.phx_snapshot_wait_peers(shards[0].h, 2)
    assert e.value.code == B.PHX_ERR_CORRUPT_SLOT
    B.phx_snapshot_wait_peers(shards[1].h, 2)
    for j in (1, 2):
        h = B.phx_ring_peer(D, 0, j)
        for slot in (0, 1):
            assert np.array_equal(received_bytes(recv, h, j, slot, shards[0]), oring.received[h][j - 1][slot]), (j, slot)
    (h0, v0), (h1, v1) = recv[1].inspect(1)
    assert not v0 and v1 and h1.step == 1                       # slot 0 (step 2) is torn on holder 1
    fresh = Shard(wls[0], device=DEV, chunk_bytes=4096)
    assert B.phx_restore_from(fresh.h, recv[1].ptrs[0]) == 1    # torn buffer: falls back to step 1
    assert B.phx_restore_from(fresh.h, recv[2].ptrs[1]) == 2    # the other holder has step 2
    oring.fail((0,))
    assert oring.recover(0) == 2
    assert_state_equal(fresh, oring.shards[0], "restored from holder 2")
    fresh.close()
    for s in shards:
        s.close()
    for rb in recv:
        rb.free()


def test_restore_from_refuses_foreign_and_empty_replicas():
    wls, shards, recv, oring = build_ring([4096], 2, 1)
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    empty = Shard(wls[0], device=DEV)
    with pytest.raises(B.PhxError) as e:
        B.phx_restore_from(empty.h, recv[1].ptrs[0])
    assert e.value.code == B.PHX_ERR_NO_COMMITTED_SNAPSHOT
    step_all(wls, shards, oring, 1, streams)
    B.phx_snapshot_wait_peers(shards[0].h, 1)
    # rank 1's handle must not accept rank 0's replica (logical shard identity)
    other = Shard(wls[1], device=DEV)
    with pytest.raises(B.PhxError) as e:
        B.phx_restore_from(other.h, recv[1].ptrs[0])
    assert e.value.code == B.PHX_ERR_LAYOUT_MISMATCH
    assert B.phx_restore_from(empty.h, recv[1].ptrs[0]) == 1
    # pinned host replicas are accepted as well (the local replica of the owner)
    shards[0].wait(1)
    again = Shard(wls[0], device=DEV)
    assert B.phx_restore_from(again.h, shards[0].replica) == 1
    assert_state_equal(again, oring.shards[0], "from pinned host memory")
    with pytest.raises(B.PhxError) as e:
        B.phx_restore_from(again.h, torch.zeros(1 << 20, dtype=torch.uint8).data_ptr() // 256 * 256 + 256)
    assert e.value.code == B.PHX_ERR_INVALID_ARG                  # pageable host memory
    for s in shards + [empty, other, again]:
        s.close()
    for rb in recv:
        rb.free()


def test_direct_source_peer_flush_and_sync_point():
    """PHX_SNAPSHOT_DIRECT + peers: the peer DMA reads the live planes, so step k+1 must wait for the
    peer commit.  Back-to-back steps with a slow many-chunk peer flush in between."""
    D, k = 2, 1
    wls, shards, recv, oring = build_ring([1_200_000], D, k, chunk=16 << 10, snapshot_source=B.PHX_SNAPSHOT_DIRECT)
    streams = (torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV))
    snaps = {}
    for t in range(1, 7):
        step_all(wls, shards, oring, t, streams, flush_host=(t % 2 == 0))
        snaps[t] = [oring.received[B.phx_ring_peer(D, r, 1)][0][t % 2].copy() for r in range(D)]
    for s in shards:
        B.phx_snapshot_wait_peers(s.h, 6)
    torch.cuda.synchronize()
    for r, s in enumerate(shards):
        h = B.phx_ring_peer(D, r, 1)
        assert np.array_equal(received_bytes(recv, h, 1, 0, s), snaps[6][r])
        assert np.array_equal(received_bytes(recv, h, 1, 1, s), snaps[5][r])
        assert_state_equal(s, oring.shards[r], "direct + peers")
        s.close()
    for rb in recv:
        rb.free()


# ------------------------------------------------------------------------------------------------
# CUDA IPC: the holder and the owner are different processes (one process per GPU in production;
# here both use the only GPU of the box).  Host-side hand-shakes only; no kernel waits on another.
# ------------------------------------------------------------------------------------------------


def _holder(q_out, q_in):
    """Rank 1: allocates the received buffer for its predecessor (rank 0), exports it, and later serves it to
    a replacement of rank 0 by re-exporting the same buffer."""
    torch.cuda.set_device(0)
    wl = W.tiny_workload([50_000, 333], dp_size=2, dp_rank=1)
    s = Shard(wl, device=DEV)
    rb = PR.ReceivedBuffers(s.info.slot_stride, 1)
    q_out.put(rb.handles()[0])
    assert q_in.get(timeout=120) == "replicated"
    (h0, v0), (h1, v1) = rb.inspect(1)
    q_out.put(((v0, h0.step, h0.dp_rank), (v1, h1.step, h1.dp_rank)))
    assert q_in.get(timeout=120) == "done"
    s.close()
    rb.free()


def test_two_process_ipc_replication_and_recovery():
    ctx = mp.get_context("spawn")
    q_h2o, q_o2h = ctx.Queue(), ctx.Queue()
    child = ctx.Process(target=_holder, args=(q_h2o, q_o2h))
    child.start()
    try:
        handle = q_h2o.get(timeout=180)
        wl = W.tiny_workload([50_000, 333], dp_size=2, dp_rank=0)
        s = Shard(wl, device=DEV, chunk_bytes=64 << 10)
        o = O.OracleShard(wl.layout(), 2, 0, chunk_bytes=64 << 10)
        p0 = W.init_params(s.n, s.n_padded, 5)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
        peer = B.phx_ipc_open(handle)                       # the holder's HBM, mapped into this process
        B.phx_shard_bind_peers(s.h, [peer])
        st = torch.cuda.Stream(device=DEV)
        for t in range(1, 4):
            g = W.gen_grads(wl, s.segments, s.n_padded, t, 5)
            s.step_and_snapshot(g.to(DEV), t)
            B.phx_snapshot_flush_peers_async(s.h, st)
            o.step(grad_record(g), **hp_of(wl), step=t)
            o.snapshot()
        B.phx_snapshot_wait_peers(s.h, 3)
        q_o2h.put("replicated")
        seen = q_h2o.get(timeout=120)                       # what the HOLDER process reads in its own buffer
        assert seen == ((True, 2, 0), (True, 3, 0))
        # the owner dies; a replacement restores from the holder's buffer over IPC
        s.drop_live()
        B.phx_shard_bind_peers(s.h, [])
        s.close()
        fresh = Shard(wl, device=DEV)
        assert B.phx_restore_from(fresh.h, peer) == 3
        assert_state_equal(fresh, o, "restored over IPC")
        fresh.close()
        B.phx_ipc_close(peer)
        q_o2h.put("done")
    finally:
        child.join(timeout=120)
    assert child.exitcode == 0


def _ring_rank(rank, world, port, q):
    """One process per ring position (both on the only GPU of the box; control plane on gloo)."""
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo")
    wl = W.tiny_workload([40_000, 77], dp_size=world, dp_rank=rank)
    s = Shard(wl, device=DEV, chunk_bytes=32 << 10)
    o = O.OracleShard(wl.layout(), world, rank, chunk_bytes=32 << 10)
    p0 = W.init_params(s.n, s.n_padded, 50 + rank)
    s.p.copy_(p0)
    s.set_state(0)
    o.set_state(p0.numpy())
    ring = PR.PeerRing(s, 1)
    st = torch.cuda.Stream(device=DEV)
    for t in range(1, 4):
        g = W.gen_grads(wl, s.segments, s.n_padded, t, 50 + rank)
        s.step_and_snapshot(g.to(DEV), t)
        ring.flush_async(st)
        o.step(grad_record(g), **hp_of(wl), step=t)
        o.snapshot()
    ring.wait(3)
    dist.barrier()
    # what I hold for my predecessor: its dp_rank, steps 2 and 3, valid
    (h0, v0), (h1, v1) = ring.received.inspect(1)
    pred = B.phx_ring_peer(world, rank, -1)
    held = (v0 and v1, (h0.step, h1.step), (h0.dp_rank, h1.dp_rank))
    # my own replica, read back from my successor's HBM through the IPC mapping, equals the oracle's snapshot bytes
    view = torch.as_tensor(type("R", (), {"__cuda_array_interface__": {
        "shape": (2 * s.info.slot_stride,), "typestr": "|u1", "data": (ring.opened[0], False), "version": 2}})(),
        device="cuda")
    same = bool(np.array_equal(view[s.info.slot_stride: s.info.slot_stride + s.info.snapshot_bytes].cpu().numpy(),
                               o.replica[1]))
    # every rank loses its live shard and pulls it back from its successor
    s.drop_live()
    back = B.phx_restore_from(s.h, ring.opened[0])
    torch.cuda.synchronize()
    ok = all(np.array_equal(a.cpu().numpy().view(np.uint32), b.view(np.uint32))
             for a, b in ((s.p, o.p), (s.m, o.m), (s.v, o.v))) and np.array_equal(bits16(s.p16), o.p16)
    q.put((rank, held, pred, same, back, bool(ok)))
    dist.barrier()
    ring.close()
    s.close()
    dist.destroy_process_group()


def test_peer_ring_class_two_processes_over_ipc():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29950 + os.getpid() % 40
    ps = [ctx.Process(target=_ring_rank, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=300) for _ in ps)
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, held, pred, same, back, ok in res:
        assert held == (True, (2, 3), (pred, pred)), (rank, held)
        assert same and back == 3 and ok


# ------------------------------------------------------------------------------------------------
# §8(f3): model-parameter publication (the all-gather fused into the step, or by copy engine) and
# reconstruction from a surviving DP rank
# ------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("mode", [B.PHX_PUBLISH_FUSED, B.PHX_PUBLISH_COPY_ENGINE])
@pytest.mark.parametrize("D,numels", [(2, [64]), (3, [5000, 77, 2048 * 3]), (4, [100_000, 12_345])])
def test_parameter_publication_equals_the_oracle_all_gather(D, numels, mode, precision):
    wls = [W.tiny_workload(numels, dp_size=D, dp_rank=r, precision=precision) for r in range(D)]
    probe = B.phx_shard_create(wls[0].layout(), D, 0)
    L = B.phx_shard_info(probe).n_padded
    B.phx_shard_destroy(probe)
    mdt = torch.float32 if precision == "fp32" else torch.bfloat16
    Wbuf = [torch.zeros(D * L, dtype=mdt, device=DEV) for _ in range(D)]          # every rank's model-parameter buffer
    shards, oshards = [], []
    for r, wl in enumerate(wls):
        kw = {} if precision == "fp32" else dict(p16=Wbuf[r][r * L:(r + 1) * L])
        s = Shard(wl, device=DEV, chunk_bytes=8192, **kw)
        o = O.OracleShard(wl.layout(), D, r, chunk_bytes=8192, precision=precision)
        p0 = W.init_params(s.n, s.n_padded, 30 + r)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
        others = [Wbuf[j] for j in range(D) if j != r] + ([Wbuf[r]] if precision == "fp32" else [])
        B.phx_shard_bind_param_peers(s.h, others, mode)
        shards.append(s)
        oshards.append(o)
    st = torch.cuda.Stream(device=DEV)
    gdt = torch.float32 if precision == "fp32" else torch.bfloat16
    for t in range(1, 4):
        for r, (s, o) in enumerate(zip(shards, oshards)):
            g = W.gen_grads(wls[r], s.segments, s.n_padded, t, 30 + r, dtype=gdt)
            s.step_and_snapshot(g.to(DEV), t)
            if mode == B.PHX_PUBLISH_COPY_ENGINE:
                B.phx_publish_params_async(s.h, st)
            o.step(grad_record(g), **hp_of(wls[r]), step=t)
        torch.cuda.synchronize()
        want = R.publish(oshards)
        for j in range(D):                                                        # every rank holds the same W
            got = Wbuf[j].cpu().numpy() if precision == "fp32" else bits16(Wbuf[j])
            assert np.array_equal(got.view(np.uint8), want.view(np.uint8)), (t, j)
    for r, (s, o) in enumerate(zip(shards, oshards)):
        assert_state_equal(s, o, f"rank {r}")
    # R30: a replacement of rank 1 (or 0) reconstructs W from a surviving rank, then its optimizer shard
    lost = min(1, D - 1)
    fresh_W = torch.zeros_like(Wbuf[lost])
    src = Wbuf[(lost + 1) % D]
    B.phx_params_restore_from(shards[lost].h, src, fresh_W)
    torch.cuda.synchronize()
    assert torch.equal(fresh_W.view(torch.uint8), src.view(torch.uint8))
    for s in shards:
        B.phx_shard_bind_param_peers(s.h, [])
        s.close()


def test_publication_argument_errors():
    wl = W.tiny_workload([4096], dp_size=2, dp_rank=0)
    s = Shard(wl, device=DEV)
    buf = torch.zeros(2 * s.n_padded, dtype=torch.bfloat16, device=DEV)
    L = B.lib()
    import ctypes as C
    arr = (C.c_void_p * 16)(*[buf.data_ptr()] * 16)
    assert L.phx_shard_bind_param_peers(s.h, arr, 16, 0) == B.PHX_ERR_INVALID_ARG
    assert L.phx_shard_bind_param_peers(s.h, arr, 1, 2) == B.PHX_ERR_INVALID_ARG
    assert L.phx_publish_params_async(s.h, None) == B.PHX_ERR_NOT_BOUND
    arr2 = (C.c_void_p * 1)(buf.data_ptr() + 2)
    assert L.phx_shard_bind_param_peers(s.h, arr2, 1, 0) == B.PHX_ERR_ALIGNMENT
    B.phx_shard_bind_param_peers(s.h, [buf])
    s.close()


def _param_rank(rank, world, port, mode, q, in_place=False):
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo")
    wl = W.tiny_workload([40_000, 77], dp_size=world, dp_rank=rank)
    # in_place: the shard's bf16 copy IS the rank's own range of W, only the other D-1 buffers are bound
    own = PR.ParamBuffer(wl) if in_place else None
    s = Shard(wl, device=DEV, p16=own.own_range() if in_place else None)
    o = O.OracleShard(wl.layout(), world, rank)
    p0 = W.init_params(s.n, s.n_padded, 70 + rank)
    s.p.copy_(p0)
    s.set_state(0)
    o.set_state(p0.numpy())
    pg = PR.ParamGroup(s, mode, own=own)
    st = torch.cuda.Stream(device=DEV)
    for t in range(1, 3):
        g = W.gen_grads(wl, s.segments, s.n_padded, t, 70 + rank)
        s.step_and_snapshot(g.to(DEV), t)
        if mode == B.PHX_PUBLISH_COPY_ENGINE:
            pg.publish_async(st)
        o.step(grad_record(g), **hp_of(wl), step=t)
    torch.cuda.synchronize()
    dist.barrier()                      # every rank's stores into my W have completed
    mine = bits16(pg.view())
    gathered = [None] * world
    dist.all_gather_object(gathered, o.p16.tobytes())           # the oracle's all-gather (control plane, gloo)
    want = np.frombuffer(b"".join(gathered), np.uint16)
    q.put((rank, bool(np.array_equal(mine, want)), bool(np.array_equal(bits16(s.p16), o.p16))))
    dist.barrier()
    pg.close()
    s.close()
    if own is not None:
        own.free()
    dist.destroy_process_group()


@pytest.mark.parametrize("in_place", [False, True])
@pytest.mark.parametrize("mode", [B.PHX_PUBLISH_FUSED, B.PHX_PUBLISH_COPY_ENGINE])
def test_param_group_two_processes_over_ipc(mode, in_place):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29900 + (os.getpid() + mode + 2 * int(in_place)) % 40
    ps = [ctx.Process(target=_param_rank, args=(r, world, port, mode, q, in_place)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=300) for _ in ps)
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert res == [(0, True, True), (1, True, True)]
