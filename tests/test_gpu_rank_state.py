"""GPU parity for SURVEY.md §8(f4): the full rank-state local snapshot (optimizer shard + model-parameter
buffer W + envelope) and the in-place recovery it enables, through the
C ABI against oracle/rank_state.py — host slot bytes identical, W part equal to the oracle all-gather,
restore bit-exact with nothing read from other ranks, torn flushes never chosen, protocol errors.
One GPU: the D logical ranks of a DP group live in one process and publish into each other's W with the
fused kernel (P2P stores) or the copy engine."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from oracle import rank_state as RS
from oracle import ring as R
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import ring as PR
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, assert_state_equal, bits16, grad_record, hp_of

pytestmark = pytest.mark.gpu
FULL = B.PHX_PAYLOAD_FULL_RANK_STATE


def build_group(numels, D, *, precision="bf16", chunk=8192, mode=B.PHX_PUBLISH_FUSED, user=b"", **kw):
    """D Shards with full-rank-state local slots, every rank's W wired to every other rank's publication,
    and the oracle twin of each."""
    wls = [W.tiny_workload(numels, dp_size=D, dp_rank=r, precision=precision) for r in range(D)]
    shards = [Shard(wl, device=DEV, chunk_bytes=chunk, payload=FULL, **kw) for wl in wls]
    ranks = []
    for r, (wl, s) in enumerate(zip(wls, shards)):
        o = O.OracleShard(wl.layout(), D, r, chunk_bytes=(chunk + 255) & ~255, precision=precision, user=user)
        p0 = W.init_params(s.n, s.n_padded, seed=60 + r)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
        if user:
            B.phx_set_user_metadata(s.h, user)
        ranks.append(RS.FullRankState(o))
    for r, s in enumerate(shards):
        others = [shards[j].W for j in range(D) if j != r] + ([s.W] if precision == "fp32" else [])
        s.has_pub = bool(others)
        if others:
            B.phx_shard_bind_param_peers(s.h, others, mode)
    return wls, shards, ranks


def iteration(wls, shards, ranks, t, streams, mode=B.PHX_PUBLISH_FUSED, flush=True, torn=None):
    """step on every rank (+ publication), all ranks' W complete, then the full-rank-state flush."""
    gdt = torch.float32 if wls[0].precision == "fp32" else torch.bfloat16
    cur = torch.cuda.current_stream()
    for r, (wl, s, fr) in enumerate(zip(wls, shards, ranks)):
        g = W.gen_grads(wl, s.segments, s.n_padded, t, seed=11 + r, dtype=gdt)
        s.params_guard()                                  # R32: nobody overwrites W while a flush still reads it
        s.step_and_snapshot(g.to(DEV), t)
        if mode == B.PHX_PUBLISH_COPY_ENGINE and s.has_pub:
            B.phx_publish_params_async(s.h, streams[1])
        fr.o.step(grad_record(g), **hp_of(wl), step=t)
    cur.wait_stream(streams[1])                           # every publication of step t has landed (one process)
    Wo = R.publish([fr.o for fr in ranks])
    for r, (s, fr) in enumerate(zip(shards, ranks)):
        fr.W[:] = Wo
        s.params_ready()
        if flush:
            if torn is not None and r == 0:
                B.phx_fault_inject_torn_flush(s.h, torn)
                fr.snapshot(abort_after_chunks=torn)
            else:
                fr.snapshot()
            s.flush_async(streams[0])


def w_bits(s):
    return s.W.cpu().numpy().view(np.uint8) if s.fp32 else bits16(s.W).view(np.uint8)


def close_all(shards):
    for s in shards:
        B.phx_shard_bind_param_peers(s.h, [])
        s.close()


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("mode", [B.PHX_PUBLISH_FUSED, B.PHX_PUBLISH_COPY_ENGINE])
@pytest.mark.parametrize("D,numels", [(1, [64]), (2, [5000, 77]), (3, [100_000, 12_345, 2048 * 3])])
def test_host_slots_hold_the_oracles_full_rank_state(D, numels, mode, precision):
    wls, shards, ranks = build_group(numels, D, precision=precision, mode=mode, user=b"rng-state-blob")
    streams = [torch.cuda.Stream(device=DEV) for _ in range(2)]
    for t in range(1, 5):
        iteration(wls, shards, ranks, t, streams, mode)
        for s, fr in zip(shards, ranks):
            s.wait(t)
            got = s.replica_slot(t).numpy()
            assert got.size == fr.snapshot_bytes
            assert np.array_equal(got, fr.slots[t % 2]), (t, fr.r)
            assert np.array_equal(w_bits(s), fr.W.view(np.uint8))
    for s, fr in zip(shards, ranks):
        assert_state_equal(s, fr.o, f"rank {fr.r}")
        hdrs = B.phx_replica_inspect(s.replica, s.info.host_slot_stride)
        assert all(v for _, v in hdrs) and {h.step for h, _ in hdrs} == {3, 4}
        assert all(h.payload == RS.payload_word(4 if s.fp32 else 2) for h, _ in hdrs)
    close_all(shards)


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("rmode", [B.PHX_RESTORE_COPY_ENGINE, B.PHX_RESTORE_BULK_KERNEL])
def test_in_place_recovery_is_bit_exact_and_reads_no_other_rank(rmode, precision):
    D, numels = 3, [30_000, 4097, 64]
    wls, shards, ranks = build_group(numels, D, precision=precision, restore_mode=rmode, user=b"rng")
    wls2, ref, ref_ranks = build_group(numels, D, precision=precision)
    streams = [torch.cuda.Stream(device=DEV) for _ in range(2)]
    for t in range(1, 8):
        iteration(wls2, ref, ref_ranks, t, streams, flush=False)
    for t in range(1, 5):
        iteration(wls, shards, ranks, t, streams)
    victim, vfr = shards[1], ranks[1]
    victim.wait(4)
    # step 5 is in flight on the victim when the transient fault hits; its partial work is discarded (I4)
    gdt = torch.float32 if precision == "fp32" else torch.bfloat16
    g5 = W.gen_grads(wls[1], victim.segments, victim.n_padded, 5, seed=12, dtype=gdt).to(DEV)
    victim.step_and_snapshot(g5, 5)
    torch.cuda.synchronize()
    victim.drop_live()
    for j in (0, 2):                                       # poison everything that is not the victim's own host memory
        shards[j].replica.fill_(0xEE)
        shards[j].W.fill_(7.0)
        shards[j].p.fill_(float("nan"))
    torch.cuda.synchronize()
    assert victim.restore() == 4
    vfr.o.step(grad_record(g5), **hp_of(wls[1]), step=5)
    vfr.drop_live()
    assert vfr.restore_in_place() == 4
    assert_state_equal(victim, vfr.o, "victim after in-place recovery")
    assert np.array_equal(w_bits(victim), vfr.W.view(np.uint8))
    assert B.phx_restored_user_metadata(victim.h) == b"rng"
    # R33: the rank's own range of W is its model-param copy again
    N = victim.n_padded
    own = victim.W[N:2 * N]
    if precision == "bf16":
        assert np.array_equal(bits16(own), O.rne_bf16(victim.p.cpu().numpy()))
    else:
        assert torch.equal(own, victim.p)
    # the victim alone replays 5..7 and lands on the uninterrupted trajectory (its grads do not depend on the others)
    for t in range(5, 8):
        g = W.gen_grads(wls[1], victim.segments, victim.n_padded, t, seed=12, dtype=gdt)
        victim.step_and_snapshot(g.to(DEV), t)
    torch.cuda.synchronize()
    for a, b in ((victim.p, ref[1].p), (victim.m, ref[1].m), (victim.v, ref[1].v)):
        assert torch.equal(a.view(torch.int32), b.view(torch.int32))
    if precision == "bf16":
        assert torch.equal(victim.p16.view(torch.int16), ref[1].p16.view(torch.int16))
    close_all(shards)
    close_all(ref)


def test_torn_flush_in_either_region_is_never_chosen_and_slot_bytes_match():
    D, numels, chunk = 2, [3000], 2048
    wls, shards, ranks = build_group(numels, D, chunk=chunk)
    streams = [torch.cuda.Stream(device=DEV) for _ in range(2)]
    s, fr = shards[0], ranks[0]
    N = s.n_padded
    n_w, n_o = -(-D * N * 2 // chunk), -(-12 * N // chunk)
    iteration(wls, shards, ranks, 1, streams)
    t = 1
    for stop in (0, 1, n_w, n_w + 1, n_w + n_o - 1, n_w + n_o):
        t += 1
        iteration(wls, shards, ranks, t, streams, torn=stop)
        torch.cuda.synchronize()
        with pytest.raises(B.PhxError) as e:
            s.wait(t)
        assert e.value.code == B.PHX_ERR_CORRUPT_SLOT
        assert np.array_equal(s.replica_slot(t).numpy(), fr.slots[t % 2]), stop     # same torn bytes, R32 order
        assert B.phx_snapshot_query(s.h) == (t - 1, (t - 1) % 2)
        # a fault now: in-place recovery goes back to t-1 on both sides, then the step is redone and commits
        s.drop_live()
        fr.drop_live()
        assert s.restore() == t - 1 == fr.restore_in_place()
        assert_state_equal(s, fr.o, f"stop {stop}")
        assert np.array_equal(w_bits(s), fr.W.view(np.uint8))
        shards[1].drop_live(); ranks[1].drop_live()
        assert shards[1].restore() == t == ranks[1].restore_in_place()                # rank 1 committed step t
        # bring rank 1 back to t-1 as the group rolls back to the last step EVERY rank completed
        t -= 1
        for x, xr in ((shards[1], ranks[1]),):
            x.replica_slot(t + 1)[:256].zero_(); xr.slots[(t + 1) % 2][:256] = 0
            x.drop_live(); xr.drop_live()
            assert x.restore() == t == xr.restore_in_place()
        t += 1
        iteration(wls, shards, ranks, t, streams)
        s.wait(t)
        assert np.array_equal(s.replica_slot(t).numpy(), fr.slots[t % 2])
    close_all(shards)


def test_protocol_errors():
    wl = W.tiny_workload([5000], dp_size=2, dp_rank=1)
    s = Shard(wl, device=DEV, payload=FULL)
    st = torch.cuda.Stream(device=DEV)
    g = W.gen_grads(wl, s.segments, s.n_padded, 1, seed=0).to(DEV)
    s.set_state(0)
    s.step_and_snapshot(g, 1)
    with pytest.raises(B.PhxError) as e:                   # W not declared complete for step 1
        s.flush_async(st)
    assert e.value.code == B.PHX_ERR_PARAMS_NOT_READY
    s.params_ready()
    s.flush_async(st)
    s.wait(1)
    s.step_and_snapshot(g, 2)
    with pytest.raises(B.PhxError) as e:                   # the declaration of step 1 does not carry over
        s.flush_async(st)
    assert e.value.code == B.PHX_ERR_PARAMS_NOT_READY
    s.params_ready()
    s.flush_async(st)
    s.wait(2)
    # bf16: d_p_bf16 must be the rank's own range of W
    other = torch.zeros(2 * s.n_padded, dtype=torch.bfloat16, device=DEV)
    assert B.lib().phx_shard_bind_params(s.h, other.data_ptr()) == B.PHX_ERR_INVALID_ARG
    assert B.lib().phx_shard_bind_params(s.h, s.W.data_ptr() + 2) == B.PHX_ERR_ALIGNMENT
    # an optimizer-only shard of the same identity refuses the full-rank-state slot and vice versa
    s2 = Shard(wl, device=DEV, replica=s.replica)
    with pytest.raises(B.PhxError) as e:
        s2.restore()
    assert e.value.code == B.PHX_ERR_LAYOUT_MISMATCH
    s2.close()
    s.close()


def test_ring_peers_still_receive_the_optimizer_only_payload():
    # asymmetric payloads: local slot = full rank state, received buffer = envelope ‖ p ‖ m ‖ v
    D, numels = 2, [5000, 77]
    wls, shards, ranks = build_group(numels, D)
    recv = PR.connect_in_process(shards, 1)
    streams = [torch.cuda.Stream(device=DEV) for _ in range(3)]
    for t in range(1, 4):
        iteration(wls, shards, ranks, t, streams)
        for s in shards:
            B.phx_snapshot_flush_peers_async(s.h, streams[2])
    torch.cuda.synchronize()
    for r, (s, fr) in enumerate(zip(shards, ranks)):
        h = (r + 1) % D
        st, nb = s.info.slot_stride, s.info.snapshot_bytes
        got = recv[h].view(1)[1 * st: 1 * st + nb].cpu().numpy()
        assert np.array_equal(got, fr.o.packed_snapshot())              # payload word 0, no W
        assert np.array_equal(s.replica_slot(3).numpy(), fr.slots[1])
    # permanent failure of rank 0: optimizer shard from the holder, W from the surviving rank (R30)
    shards[0].drop_live()
    assert B.phx_restore_from(shards[0].h, recv[1].ptrs[0]) == 3
    B.phx_params_restore_from(shards[0].h, shards[1].W, shards[0].W)
    assert_state_equal(shards[0], ranks[0].o, "rank 0 from its holder")
    assert np.array_equal(w_bits(shards[0]), ranks[0].W.view(np.uint8))
    for s in shards:
        B.phx_shard_bind_peers(s.h, [])
    for rb in recv:
        rb.free()
    close_all(shards)


def test_full_payload_under_relaxed_sync_never_commits_a_W_of_the_next_step():
    """the full-rank-state flush reads the LIVE W, and the rank's own range of W is d_p_bf16,
    which step k+1's kernel rewrites.  Under PHX_SYNC_RELAXED (depth 3) with a slow flush (4 KiB chunks) and steps
    issued back to back WITHOUT phx_params_guard, every committed host slot must still hold the W of exactly its
    own step: the step waits until the newest flush has finished reading W."""
    wls, shards, ranks = build_group([600_000, 77], 1, chunk=4096, sync_mode=B.PHX_SYNC_RELAXED, staging_depth=3)
    wl, s, fr = wls[0], shards[0], ranks[0]
    side = torch.cuda.Stream(device=DEV)
    snaps = {}
    grads = [W.gen_grads(wl, s.segments, s.n_padded, t, seed=11).to(DEV) for t in range(1, 7)]
    torch.cuda.synchronize()
    for t in range(1, 7):
        s.step_and_snapshot(grads[t - 1], t)          # no guard, no host sync: the hazard window is wide open
        s.params_ready()
        s.flush_async(side)                           # ~2300 small copies, W first
        fr.o.step(grad_record(grads[t - 1]), **hp_of(wl), step=t)
        fr.W[:] = R.publish([fr.o])
        fr.snapshot()
        snaps[t] = fr.slots[t % 2].copy()
    s.wait(6)
    torch.cuda.synchronize()
    for t in (5, 6):
        assert np.array_equal(s.replica_slot(t).numpy(), snaps[t]), t
    assert_state_equal(s, fr.o, "full + relaxed")
    close_all(shards)


@pytest.mark.parametrize("sync", [B.PHX_SYNC_STRICT, B.PHX_SYNC_RELAXED])
def test_graph_form_with_full_rank_state_payload(sync):
    """The graph-capturable form covers §8(f4) too: per iteration, for the D ranks of one DP group,
    [params_ready -> full-rank-state flush(k-1) ‖ window] -> params_guard -> step k (fused publication), captured
    once (two iterations per graph) and replayed; host slots byte-identical to oracle/rank_state.py, then an
    in-place recovery from them back in the eager form."""
    D, numels = 2, [60_000, 4097, 64]
    wls, shards, ranks = build_group(numels, D, chunk=64 << 10, sync_mode=sync)
    cap, side = torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV)
    a = torch.randn(256, 256, device=DEV, dtype=torch.bfloat16)
    c = torch.empty_like(a)
    with torch.cuda.stream(cap):
        torch.matmul(a, a, out=c)
    torch.cuda.synchronize()
    gbuf = [[torch.zeros(s.n_padded, dtype=torch.bfloat16, device=DEV) for _ in range(2)] for s in shards]

    def load_grads(t):
        for r, (wl, s, fr) in enumerate(zip(wls, shards, ranks)):
            g = W.gen_grads(wl, s.segments, s.n_padded, t, seed=11 + r)
            gbuf[r][t & 1].copy_(g)
            fr.o.step(grad_record(g), **hp_of(wl), step=t)
        Wo = R.publish([fr.o for fr in ranks])
        for fr in ranks:
            fr.W[:] = Wo
            fr.snapshot()

    for s in shards:
        s.graph_begin(stream=cap)
    # a full payload flush without the declaration is refused in the graph form as well
    load_grads(1)
    torch.cuda.synchronize()
    for r, s in enumerate(shards):
        s.graph_step(gbuf[r][1], stream=cap)
    torch.cuda.synchronize()
    assert B.lib().phx_graph_flush_async(shards[0].h, side.cuda_stream) == B.PHX_ERR_PARAMS_NOT_READY
    snaps = {1: [fr.slots[1].copy() for fr in ranks]}
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(2):
            for s in shards:
                s.params_ready(cap)                 # every rank's step k-1 (same capture stream) has published into W
            side.wait_stream(cap)
            for s in shards:
                s.graph_flush(side)
            torch.matmul(a, a, out=c)
            for s in shards:
                s.params_guard(cap)                 # no rank publishes step k into a W a flush still reads
            for r, s in enumerate(shards):
                s.graph_step(gbuf[r][i & 1], stream=cap)
        cap.wait_stream(side)
    t = 1
    for _ in range(3):
        for i in range(2):
            t += 1
            load_grads(t)
            snaps[t] = [fr.slots[t % 2].copy() for fr in ranks]
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
    assert t == 7
    for r, (s, fr) in enumerate(zip(shards, ranks)):
        assert s.graph_end() == 7
        assert_state_equal(s, fr.o, f"rank {r} after graph replays")
        assert np.array_equal(w_bits(s), fr.W.view(np.uint8))
        for step in (5, 6):
            assert np.array_equal(s.replica_slot(step).numpy(), snaps[step][r]), (r, step)
    # eager again: the newest snapshot (7) is still pending; declare, flush, then recover rank 1 in place
    for s in shards:
        s.params_ready()
        s.flush_async(side)
    for r, s in enumerate(shards):
        s.wait(7)
        assert np.array_equal(s.replica_slot(7).numpy(), snaps[7][r])
    victim, vfr = shards[1], ranks[1]
    victim.drop_live()
    victim.W.zero_()
    assert victim.restore() == 7
    torch.cuda.synchronize()
    assert_state_equal(victim, vfr.o, "in-place recovery after the graph form")
    assert np.array_equal(w_bits(victim), vfr.W.view(np.uint8))
    close_all(shards)
