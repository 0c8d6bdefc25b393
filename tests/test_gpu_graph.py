"""GPU parity for the graph-capturable form (include/phx.h "graph"): the device-side derivation
of the per-step scalars equals the oracle's bitwise, and a CAPTURED (compute window + flush + step) graph
replayed for many iterations leaves exactly the oracle's state, staging bytes and committed host slots."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

from gpu_util import DEV, assert_state_equal, hp_of, make_pair

pytestmark = pytest.mark.gpu


def test_device_derived_scalars_equal_the_oracle_for_steps_up_to_a_million():
    rng = np.random.default_rng(3)
    steps = sorted(set([1, 2, 3, 4, 5, 7, 10, 100, 1000, 65535, 65536, 10**6, 2**40 + 3]
                       + [int(x) for x in rng.integers(1, 10**6, 4000)]))
    for lr, b1, b2, wd in ((3e-4, 0.9, 0.95, 0.1), (1e-3, 0.9, 0.999, 0.01), (6e-4, 0.8, 0.98, 0.0)):
        got = np.array(B.phx_derived_scalars_device(lr, b1, b2, wd, steps), np.float32).view(np.uint32)
        for i, t in enumerate(steps):
            exp = O.scalars(lr, b1, b2, 1e-8, wd, t).view(np.uint32)
            assert np.array_equal(got[i], exp), (lr, b1, b2, wd, t)
            host = np.array(B.phx_derived_scalars_host(lr, b1, b2, wd, t), np.float32).view(np.uint32)
            assert np.array_equal(host, exp)


@pytest.mark.parametrize("source", [B.PHX_SNAPSHOT_STAGED, B.PHX_SNAPSHOT_DIRECT])
@pytest.mark.parametrize("clip", [0.0, 0.02])
def test_eager_calls_of_the_graph_form_match_the_oracle(source, clip):
    wl = W.tiny_workload([300_000, 77, 12_345], dp_size=1, hyper=W.Hyper(max_grad_norm=clip))
    s, o, gdev, gbits = make_pair(wl, steps=6, chunk_bytes=256 << 10, snapshot_source=source, user=b"graph-user")
    side = torch.cuda.Stream(device=DEV)
    hp = hp_of(wl)
    s.step_and_snapshot(gdev[0], 1)                   # eager step; its snapshot becomes the graph form's first flush
    o.step(gbits[0], **hp, step=1); o.snapshot()
    s.graph_begin()
    with pytest.raises(B.PhxError) as e:
        s.step_and_snapshot(gdev[1], 2)
    assert e.value.code == B.PHX_ERR_GRAPH_MODE
    snaps = {1: o.replica[1].copy()}
    for t in range(2, 6):
        s.graph_flush(side)                           # flush of snapshot t-1
        s.graph_step(gdev[t - 1])
        o.step(gbits[t - 1], **hp, step=t); o.snapshot()
        snaps[t] = o.replica[t % 2].copy()
    assert s.graph_end() == 5
    assert_state_equal(s, o, "graph form, eager")
    assert np.array_equal(s.replica_slot(4).numpy(), snaps[4])
    assert np.array_equal(s.replica_slot(3).numpy(), snaps[3])         # slot 1 holds step 3 (step 5 not flushed yet)
    if source == B.PHX_SNAPSHOT_STAGED:
        assert np.array_equal(s.staging_slot(5).cpu().numpy(), o.packed_snapshot())
    s.flush_async(side)                               # back in the eager form: the still-staged newest snapshot
    s.wait(5)
    assert np.array_equal(s.replica_slot(5).numpy(), o.replica[1])
    s.step_and_snapshot(gdev[5], 6)                   # and the eager step continues at last_step + 1
    o.step(gbits[5], **hp, step=6)
    assert_state_equal(s, o, "eager after graph_end")
    s.drop_live()
    assert s.restore() == 5 and B.phx_restored_user_metadata(s.h) == b"graph-user"
    s.close()


@pytest.mark.parametrize("mode,depth", [(B.PHX_SYNC_STRICT, 2), (B.PHX_SYNC_RELAXED, 2), (B.PHX_SYNC_STRICT, 1),
                                        (B.PHX_SYNC_RELAXED, 4)])
def test_captured_graph_replayed_ten_iterations_is_bit_exact(mode, depth):
    """a captured (GEMM window + flush(k-1) + step k) x L graph, L = lcm(depth, 2) iterations,
    replayed until 10+ iterations have run, against the oracle stepping 10+ times."""
    wl = W.CONFIGS["c1"]
    L = {1: 2, 2: 2, 4: 4}[depth]
    reps = (10 + L - 1) // L
    s, o, _, _ = make_pair(wl, steps=0, chunk_bytes=1 << 20, staging_depth=depth, sync_mode=mode)
    hp = hp_of(wl)
    # the graph reads the gradients of iteration i from a fixed buffer: L buffers, refilled between replays
    gbuf = [torch.zeros(s.n_padded, dtype=torch.bfloat16, device=DEV) for _ in range(L)]
    a = torch.randn(512, 512, device=DEV, dtype=torch.bfloat16)
    c = torch.empty_like(a)
    cap = torch.cuda.Stream(device=DEV)
    side = torch.cuda.Stream(device=DEV)
    with torch.cuda.stream(cap):
        torch.matmul(a, a, out=c)                      # cuBLAS must be initialised on this stream before a capture
    torch.cuda.synchronize()
    # one eager step of the graph form first, so that the first captured flush has a snapshot to send
    osegs = [(tid, off, ln) for tid, _, off, ln in o.segments]
    g1 = W.gen_grads(wl, osegs, s.n_padded, 1, wl.seed)
    s.graph_begin(stream=cap)
    gbuf[1 % L].copy_(g1)
    torch.cuda.synchronize()
    s.graph_step(gbuf[1 % L], stream=cap)
    o.step(g1.view(torch.int16).numpy().view(np.uint16).copy(), **hp, step=1); o.snapshot()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(L):
            t = 2 + i                                  # issue index at capture: 2 .. L+1
            side.wait_stream(cap)                      # fork: the flush of snapshot t-1 runs beside the window
            s.graph_flush(side)
            for _ in range(4):
                torch.matmul(a, a, out=c)              # the stand-in compute window
            s.graph_step(gbuf[t % L], stream=cap)      # a2 joins the side stream back, then prologue + fused kernel
        cap.wait_stream(side)                          # relaxed mode: the last flush may not be joined by any a2
    t = 1
    for _ in range(reps):
        for i in range(L):
            t += 1
            g = W.gen_grads(wl, osegs, s.n_padded, t, wl.seed)
            gbuf[t % L].copy_(g)
            o.step(g.view(torch.int16).numpy().view(np.uint16).copy(), **hp, step=t)
            o.snapshot()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        assert_state_equal_live(s, o, f"after replay ending at step {t}")
    assert s.graph_end() == t and t >= 11
    assert_state_equal(s, o, "graph replays")
    # every flush inside the graph committed: host slots hold steps t-1 (newest flushed) and t-2
    assert np.array_equal(s.replica_slot(t - 1).numpy(), o_slot_of(o, wl, hp, t - 1))
    s.flush_async(side)
    s.wait(t)
    assert np.array_equal(s.replica_slot(t).numpy(), o.replica[t % 2])
    s.close()


def assert_state_equal_live(s, o, what):
    for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v)):
        assert np.array_equal(dev.cpu().numpy().view(np.uint32), ref.view(np.uint32)), (what, name)


def o_slot_of(o, wl, hp, step):
    """The oracle's replica slot of `step` — still intact in slot step % 2 because the oracle snapshotted every step
    and only step+1 (other parity) came after it."""
    h = O.parse_header(o.replica[step % 2][:256].tobytes())
    assert h is not None and h["step"] == step
    return o.replica[step % 2]


def test_misaligned_replay_is_reported():
    wl = W.tiny_workload([8192], dp_size=1)
    s, o, gdev, _ = make_pair(wl, steps=3)
    cap = torch.cuda.Stream(device=DEV)
    s.graph_begin(stream=cap)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        s.graph_step(gdev[0], stream=cap)              # ONE step captured with depth 2: every second replay is misaligned
    graph.replay(); graph.replay()
    with pytest.raises(B.PhxError) as e:
        s.graph_end()
    assert e.value.code == B.PHX_ERR_STEP_ORDER
    assert B.phx_last_step(s.h) == 2                   # the device counter is still the truth
    s.close()


@pytest.mark.parametrize("depth,captured,replays,ok", [(1, 1, 2, False), (3, 3, 2, False), (1, 2, 3, True),
                                                       (3, 6, 2, True), (2, 2, 3, True)])
def test_replay_alignment_covers_the_host_ping_pong_parity(depth, captured, replays, ok):
    """a captured sequence of `depth` steps keeps the STAGING slot aligned on every replay, but with an odd
    depth it flips the host ping-pong parity baked into the captured flush (step & 1): every second replay would
    invalidate and rewrite the newest committed host slot.  phx.h asks for a multiple of lcm(depth, 2) steps; the
    device check must report anything else (PHX_ERR_STEP_ORDER at phx_graph_end)."""
    wl = W.tiny_workload([8192], dp_size=1)
    s, o, gdev, _ = make_pair(wl, steps=6, staging_depth=depth)
    cap, side = torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV)
    s.graph_begin(stream=cap)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(captured):
            s.graph_step(gdev[i], stream=cap)
            side.wait_stream(cap)
            s.graph_flush(side)
            cap.wait_stream(side)
    for _ in range(replays):
        graph.replay()
    torch.cuda.synchronize()
    if ok:
        assert s.graph_end() == captured * replays
    else:
        with pytest.raises(B.PhxError) as e:
            s.graph_end()
        assert e.value.code == B.PHX_ERR_STEP_ORDER
        assert B.phx_last_step(s.h) == captured * replays
    s.close()


def test_user_metadata_changed_between_replays_reaches_the_committed_envelope():
    """the caller blob (RNG states) changes every iteration, but the graph form's envelope
    template was frozen at phx_graph_begin, so every replayed snapshot committed the blob of begin and a restore
    handed back stale RNG state.  phx_graph_set_user_metadata updates the device-resident template in stream order;
    the eager setter refuses in graph mode instead of silently doing nothing.  Replica slots vs the oracle's, byte
    for byte, and the restored blob."""
    wl = W.tiny_workload([50_000, 77], dp_size=1)
    blob0, blob1, blob2 = b"rng-state-at-begin", bytes(range(1, 129)), b"x"
    s, o, gdev, gbits = make_pair(wl, steps=7, chunk_bytes=64 << 10, user=blob0)
    hp = hp_of(wl)
    cap, side = torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV)
    gbuf = [torch.zeros_like(gdev[0]) for _ in range(2)]
    s.graph_begin(stream=cap)
    assert B.lib().phx_set_user_metadata(s.h, blob1, len(blob1)) == B.PHX_ERR_GRAPH_MODE
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(2):
            s.graph_step(gbuf[(1 + i) % 2], stream=cap)     # issue indices 1, 2
            side.wait_stream(cap)
            s.graph_flush(side)
            cap.wait_stream(side)
        assert B.lib().phx_graph_set_user_metadata(s.h, blob1, len(blob1), cap.cuda_stream) == B.PHX_ERR_INVALID_ARG
        assert B.lib().phx_graph_set_hyper(s.h, 1e-3, 0.9, 0.95, 1e-8, 0.0, cap.cuda_stream) == B.PHX_ERR_INVALID_ARG
    t = 0
    for blob in (None, blob1, blob2):                       # replay 1 keeps the blob of begin
        if blob is not None:
            B.phx_graph_set_user_metadata(s.h, blob, cap)
            o.user = blob
        for i in range(2):
            t += 1
            with torch.cuda.stream(cap):
                gbuf[t % 2].copy_(gdev[t - 1])
            o.step(gbits[t - 1], **hp, step=t)
            o.snapshot()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        for k in (t - 1, t):
            assert np.array_equal(s.replica_slot(k).numpy(), o.replica[k % 2]), (t, k)
        hdr = O.parse_header(s.replica_slot(t).numpy()[:256].tobytes())
        assert hdr["user"] == (blob0 if blob is None else blob)
    assert s.graph_end() == 6
    # the eager calls carry the last blob on, and a restore hands it back
    s.step_and_snapshot(gdev[6], 7); s.flush_async(side); s.wait(7)
    o.step(gbits[6], **hp, step=7); o.snapshot()
    assert np.array_equal(s.replica_slot(7).numpy(), o.replica[1])
    s.drop_live()
    assert s.restore() == 7
    assert B.phx_restored_user_metadata(s.h) == blob2
    s.close()


def test_graph_form_protocol_errors():
    wl = W.tiny_workload([8192], dp_size=1)
    s, _, gdev, _ = make_pair(wl, steps=1)
    L = B.lib()
    assert L.phx_graph_step_and_snapshot(s.h, gdev[0].data_ptr(), None) == B.PHX_ERR_GRAPH_MODE
    assert L.phx_graph_flush_async(s.h, None) == B.PHX_ERR_GRAPH_MODE
    assert L.phx_graph_end(s.h, None) == B.PHX_ERR_GRAPH_MODE
    s.graph_begin()
    assert L.phx_graph_begin(s.h, 1e-3, 0.9, 0.95, 1e-8, 0.0, None) == B.PHX_ERR_GRAPH_MODE
    assert L.phx_graph_flush_async(s.h, None) == B.PHX_ERR_NO_FLUSH_PENDING
    assert L.phx_restore(s.h, None, None) == B.PHX_ERR_GRAPH_MODE
    assert L.phx_graph_step_and_snapshot(s.h, gdev[0].data_ptr() + 2, None) == B.PHX_ERR_ALIGNMENT
    assert s.graph_end() == 0
    s.close()
    full = B.phx_shard_create([(8192, 0)], 1, 0, payload=B.PHX_PAYLOAD_FULL_RANK_STATE)
    assert L.phx_graph_begin(full, 1e-3, 0.9, 0.95, 1e-8, 0.0, None) == B.PHX_ERR_NOT_BOUND
    B.phx_shard_destroy(full)


@pytest.mark.parametrize("k", [1, 2])
def test_captured_graph_with_host_flush_and_ring_peer_flush(k):
    """The graph form covers §8(f1) too: [flush(k-1) to the host ‖ flush(k-1) to the k ring peers ‖ window] -> step k,
    captured once, replayed; the peers' received slots are byte-identical to the host slots and to the oracle's."""
    from paper_2607_01646_b200 import ring as PR
    wl = W.tiny_workload([200_000, 77], dp_size=3, dp_rank=0)
    s, o, _, _ = make_pair(wl, steps=0, chunk_bytes=256 << 10)
    recv = PR.ReceivedBuffers(s.info.slot_stride, k)
    B.phx_shard_bind_peers(s.h, recv.ptrs)
    hp = hp_of(wl)
    osegs = [(tid, off, ln) for tid, _, off, ln in o.segments]
    gbuf = [torch.zeros(s.n_padded, dtype=torch.bfloat16, device=DEV) for _ in range(2)]
    a = torch.randn(256, 256, device=DEV, dtype=torch.bfloat16)
    c = torch.empty_like(a)
    cap, side, peer = (torch.cuda.Stream(device=DEV) for _ in range(3))
    with torch.cuda.stream(cap):
        torch.matmul(a, a, out=c)
    torch.cuda.synchronize()

    def grads_of(t):
        return W.gen_grads(wl, osegs, s.n_padded, t, wl.seed)

    s.graph_begin(stream=cap)
    g1 = grads_of(1)
    gbuf[1].copy_(g1)
    torch.cuda.synchronize()
    s.graph_step(gbuf[1], stream=cap)
    o.step(g1.view(torch.int16).numpy().view(np.uint16).copy(), **hp, step=1); o.snapshot()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(2):
            side.wait_stream(cap); s.graph_flush(side)
            peer.wait_stream(cap); B.phx_graph_flush_peers_async(s.h, peer)
            torch.matmul(a, a, out=c)
            s.graph_step(gbuf[i & 1], stream=cap)
        cap.wait_stream(side); cap.wait_stream(peer)
    t = 1
    snaps = {}
    for _ in range(3):
        for i in range(2):
            t += 1
            g = grads_of(t)
            gbuf[t & 1].copy_(g)
            o.step(g.view(torch.int16).numpy().view(np.uint16).copy(), **hp, step=t); o.snapshot()
            snaps[t] = o.replica[t % 2].copy()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
    assert s.graph_end() == t == 7
    assert_state_equal(s, o, "graph with peers")
    for step in (5, 6):
        host = s.replica_slot(step).numpy()
        assert np.array_equal(host, snaps[step]), step
        for j in range(1, k + 1):
            got = recv.view(j)[(step % 2) * s.info.slot_stride:(step % 2) * s.info.slot_stride + s.info.snapshot_bytes]
            assert np.array_equal(got.cpu().numpy(), snaps[step]), (step, j)
    # back in the eager form: the newest snapshot is still pending for both destinations
    s.flush_async(side)
    B.phx_snapshot_flush_peers_async(s.h, peer)
    s.wait(7)
    B.phx_snapshot_wait_peers(s.h, 7)
    for j in range(1, k + 1):
        got = recv.view(j)[s.info.slot_stride:s.info.slot_stride + s.info.snapshot_bytes]
        assert np.array_equal(got.cpu().numpy(), snaps[7])
    s.drop_live()
    assert B.phx_restore_from(s.h, recv.ptrs[0], torch.cuda.current_stream()) == 7
    assert_state_equal(s, o, "restored from the ring peer after graph replays")
    B.phx_shard_bind_peers(s.h, [])
    recv.free()
    s.close()
