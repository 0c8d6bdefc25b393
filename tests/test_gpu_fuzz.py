"""Model-based protocol fuzz: random sequences of the library's calls — step, flush, torn flush, drop + restore in one
or two phases (issued while flushes are still in flight), stretches through the graph-capturable form — on small ragged
shards in every staging depth / sync mode / snapshot source / restore mode, with the CPU oracle driven through the
same sequence.  At random points and at the end (the comparison synchronises, so not after every call) the live state must equal the oracle's bit for bit, errors must agree (a restore with
nothing committed fails on both sides), and at the end both host slots must hold the oracle's bytes — torn slots
included.  What it guards: the slot / event bookkeeping of phx_api.cu (which snapshot is pending, which slot is in flight,
torn or committed, what a restore may trust), not the arithmetic."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

from gpu_util import DEV, assert_state_equal, hp_of, make_pair

pytestmark = pytest.mark.gpu

CONFIGS = [(depth, sync, "staged", rmode) for depth in (1, 2, 3, 4) for sync in ("strict", "relaxed")
           for rmode in ("copy", "bulk")] + [(2, "strict", "direct", "copy"), (2, "strict", "direct", "bulk")]


@pytest.mark.parametrize("round_", [0, 1])
@pytest.mark.parametrize("depth,sync,source,rmode", CONFIGS)
def test_random_call_sequences_track_the_oracle(depth, sync, source, rmode, round_):
    import zlib
    seed = zlib.crc32(repr((depth, sync, source, rmode, round_)).encode()) & 0xFFFF
    rng = np.random.default_rng(seed)
    n = int(rng.integers(3_000, 120_000))
    clip = float(rng.choice([0.0, 0.02]))
    wl = W.tiny_workload([n, 77, 1], dp_size=2, dp_rank=int(rng.integers(0, 2)), grad_kind="heavy_tail",
                         hyper=W.Hyper(max_grad_norm=clip))
    chunk = int(rng.choice([16, 64, 256])) << 10
    s, o, gdev, gbits = make_pair(
        wl, steps=8, chunk_bytes=chunk, staging_depth=depth,
        sync_mode=B.PHX_SYNC_STRICT if sync == "strict" else B.PHX_SYNC_RELAXED,
        snapshot_source=B.PHX_SNAPSHOT_DIRECT if source == "direct" else B.PHX_SNAPSHOT_STAGED,
        restore_mode=B.PHX_RESTORE_COPY_ENGINE if rmode == "copy" else B.PHX_RESTORE_BULK_KERNEL)
    hp = hp_of(wl)
    cur, side = torch.cuda.current_stream(), torch.cuda.Stream(device=DEV)
    nchunks = (o.snapshot_bytes - O.HEADER_BYTES + o.chunk_bytes - 1) // o.chunk_bytes
    pending = False                     # the newest step's snapshot has not been flushed
    log = []

    def step():
        nonlocal pending
        t = o.last_step + 1
        s.step_and_snapshot(gdev[t % 8], t)
        o.step(gbits[t % 8], **hp, step=t)
        pending = True

    def flush(torn=None):
        nonlocal pending
        if torn is not None:
            B.phx_fault_inject_torn_flush(s.h, torn)
        s.flush_async(side)
        o.snapshot(abort_after_chunks=torn)
        pending = False

    def restore(two_phase):
        nonlocal pending
        try:
            want = o.restore()
        except O.OracleError:
            want = None
        if want is None:
            rc = (B.lib().phx_restore_async if two_phase else B.lib().phx_restore)(s.h, None, None)
            assert rc == B.PHX_ERR_NO_COMMITTED_SNAPSHOT, (log, rc)
            return
        if two_phase:
            side.wait_stream(cur)
            assert s.restore_async(side) == want, log
            if rng.random() < 0.5:
                s.restore_wait_params(cur)
        else:
            assert s.restore(cur) == want, log
        pending = False

    for _ in range(60):
        r = rng.random()
        if r < 0.40:
            op = "step"
            step()
        elif r < 0.65 and pending:
            op = "flush"
            flush()
        elif r < 0.72 and pending:
            j = int(rng.integers(0, nchunks + 1))
            op = f"torn{j}"
            flush(torn=j)
        elif r < 0.86:
            two = bool(rng.random() < 0.5)
            if rng.random() < 0.7:      # a real fault: the live state is gone (issued on the compute stream, no host
                if source == "direct":  # sync; a direct-source flush READS the live planes, so the fault follows it)
                    cur.wait_stream(side)
                for x in (s.p, s.m, s.v, s.p16):
                    x.zero_()
                o.drop_live()
                op = "drop+restore" + ("_async" if two else "")
            else:                       # a rollback of a healthy rank
                op = "restore" + ("_async" if two else "")
            log.append(op)
            restore(two)
            step()                      # recompute of the in-flight step (waits for the moments by itself); after a
                                        # restore that found nothing committed both sides go on from the same (lost) state
            log.append("step")
            if rng.random() < 0.5:      # (the comparison synchronises: not after every call, so that the next calls
                assert_state_equal(s, o, f"seed {seed} after {log[-12:]}")   # find flushes and restores in flight)
            continue
        elif r < 0.93:
            k = int(rng.integers(1, 4))
            op = f"graph{k}"
            s.graph_begin()
            for _i in range(k):
                if pending:
                    s.graph_flush(side)
                    o.snapshot()
                t = o.last_step + 1
                s.graph_step(gdev[t % 8])
                o.step(gbits[t % 8], **hp, step=t)
                pending = True
            assert s.graph_end() == o.last_step, log
        else:
            op = "sync"
            torch.cuda.synchronize()
        log.append(op)
        if rng.random() < 0.3:
            assert_state_equal(s, o, f"seed {seed} after {log[-12:]}")
    assert_state_equal(s, o, f"seed {seed} at the end of {log}")
    if pending:
        flush()
    torch.cuda.synchronize()
    stride = s.info.host_slot_stride
    for k in (0, 1):
        got = s.replica[k * stride: k * stride + s.info.host_snapshot_bytes].numpy()
        assert np.array_equal(got, o.replica[k]), f"seed {seed}: host slot {k} after {log[-12:]}"
    host_dropped, _ = B.phx_dropped_snapshots(s.h)
    assert host_dropped >= 0
    s.close()


RING_CASES = [(3, 1, None), (4, 2, None), (4, 1, [0, 0, 1, 1]), (5, 2, [7, 3, 3, 7, 9]), (6, 2, [0, 0, 1, 1, 2, 2]),
              (6, 3, [0, 1, 2, 3, 0, 1])]


@pytest.mark.parametrize("D,k,domains", RING_CASES)
def test_random_ring_histories_with_failures_track_the_ring_oracle(D, k, domains):
    """f1 under fuzz: D logical ranks, each at its own step, replicate to their k holders (plain ring or the
    topology-aware placement), skip or tear transfers at random; whole failure domains (or random ranks) die with a step
    in flight and are rebuilt from whichever holder the ring oracle names; the history goes on over the SAME received
    buffers.  At the end every rank's state and every received slot — torn ones included — equal the oracle's."""
    import zlib
    from oracle import ring as R
    from paper_2607_01646_b200 import ring as PR
    from paper_2607_01646_b200.shard import Shard
    from gpu_util import grad_record
    rng = np.random.default_rng(zlib.crc32(repr((D, k, domains)).encode()))
    chunk = 8192
    n0 = int(rng.integers(2_000, 40_000))
    wls = [W.tiny_workload([n0, 77], dp_size=D, dp_rank=r) for r in range(D)]
    shards = [Shard(wl, device=DEV, chunk_bytes=chunk) for wl in wls]
    recv = PR.connect_in_process(shards, k, domains)
    oring = R.OracleRing(wls[0].layout(), D, k, chunk_bytes=chunk, domains=domains)
    place = PR.placement(D, k, domains)
    assert place == oring.place
    holds = [PR.held_for(place, h) for h in range(D)]
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        p0 = W.init_params(s.n, s.n_padded, seed=200 + r)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
    peer_stream = torch.cuda.Stream(device=DEV)
    nchunks = (oring.shards[0].snapshot_bytes - O.HEADER_BYTES + chunk - 1) // chunk
    hp = hp_of(wls[0])

    def step(r, flush=True):
        s, o = shards[r], oring.shards[r]
        t = o.last_step + 1
        g = W.gen_grads(wls[r], s.segments, s.n_padded, t, seed=7 + r)
        s.step_and_snapshot(g.to(DEV), t)
        o.step(grad_record(g), **hp, step=t)
        if not flush:
            return
        u = rng.random()
        if u < 0.75:
            B.phx_snapshot_flush_peers_async(s.h, peer_stream)
            oring.replicate(r)
        elif u < 0.9:
            j, c = int(rng.integers(1, k + 1)), int(rng.integers(0, nchunks + 1))
            B.phx_fault_inject_torn_peer_flush(s.h, j, c)
            B.phx_snapshot_flush_peers_async(s.h, peer_stream)
            oring.replicate(r, abort_after_chunks={j: c})
        # else: this snapshot never reaches the peers

    n_failures = 0
    for _round in range(10):
        for r in rng.permutation(D):
            for _ in range(int(rng.integers(0, 3))):
                step(int(r))
        if rng.random() < 0.5:
            if domains is not None:
                d = domains[int(rng.integers(0, D))]
                failed = [q for q in range(D) if domains[q] == d]
            else:
                failed = [int(x) for x in rng.choice(D, size=int(rng.integers(1, k + 1)), replace=False)]
            if not R.recoverable_with(place, failed):
                continue
            for q in failed:                             # would every lost shard still have a valid replica on a survivor?
                oring.alive[q] = False
            covered = all(oring.newest_replica_of(r) is not None for r in failed)
            for q in failed:
                oring.alive[q] = True
            if not covered:
                continue                                 # nothing committed on a survivor yet: not a history I3 covers
            for r in failed:
                step(r, flush=False)                     # a step in flight on the nodes that die
            torch.cuda.synchronize()
            oring.fail(failed)
            for r in failed:
                shards[r].close()
                for j in range(1, len(holds[r]) + 1):
                    recv[r].view(j).fill_(0xA5)
            for r in failed:
                fresh = Shard(wls[r], device=DEV, chunk_bytes=chunk)
                holder, _, _, hd = oring.newest_replica_of(r)
                got = B.phx_restore_from(fresh.h, recv[holder].ptrs[holds[holder].index(r)])
                assert got == hd["step"] == oring.recover(r)
                for j in range(1, len(holds[r]) + 1):    # "the buffers it holds start empty"
                    recv[r].view(j).zero_()
                B.phx_shard_bind_peers(fresh.h, [recv[h].ptrs[holds[h].index(r)] for h in place[r]])
                shards[r] = fresh
                assert_state_equal(fresh, oring.shards[r], f"rank {r} rebuilt from holder {holder}")
            n_failures += 1
    torch.cuda.synchronize()
    st, nb = shards[0].info.slot_stride, shards[0].info.snapshot_bytes
    for r, (s, o) in enumerate(zip(shards, oring.shards)):
        assert_state_equal(s, o, f"rank {r} at the end")
        for h in place[r]:
            buf = recv[h].view(holds[h].index(r) + 1)
            for slot in (0, 1):
                assert np.array_equal(buf[slot * st: slot * st + nb].cpu().numpy(), oring.recv[(h, r)][slot]), (r, h, slot)
    assert n_failures >= 1, "the seeded history must contain at least one recovered failure"
    for s in shards:
        B.phx_shard_bind_peers(s.h, [])
        s.close()
    for rb in recv:
        rb.free()
