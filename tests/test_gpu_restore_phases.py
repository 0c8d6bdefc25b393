"""GPU parity for the TWO-PHASE restore (include/phx.h phx_restore_async / phx_restore_wait_params; DESIGN.md
reading R37): on a side stream the parameters come back first (p, the bf16 copy, W of a full rank state), the
moments behind them; the recomputed iteration's forward/backward may start at "parameters ready" and the next
optimizer step waits for the moments by itself.  Compared with the oracle's two phases (oracle.restore_params_first /
restore_finish, rank_state.restore_in_place_*) bit for bit, with the side stream artificially held back so that a
missing wait would be seen."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

from gpu_util import DEV, assert_state_equal, bits16, hp_of, make_pair
from test_gpu_rank_state import build_group, close_all, iteration, w_bits

pytestmark = pytest.mark.gpu
RMODES = [B.PHX_RESTORE_COPY_ENGINE, B.PHX_RESTORE_BULK_KERNEL]
HOLD = 60_000_000     # cycles the side stream is held back before the restore may start (~30 ms)


def run_with_flushes(s, o, gdev, gbits, hp, steps, side, torn_last=None):
    for t in range(1, steps + 1):
        s.step_and_snapshot(gdev[t - 1], t)
        o.step(gbits[t - 1], **hp, step=t)
        if t == steps and torn_last is not None:
            B.phx_fault_inject_torn_flush(s.h, torn_last)
        s.flush_async(side)
        o.snapshot(abort_after_chunks=torn_last if t == steps else None)


@pytest.mark.parametrize("rmode", RMODES)
@pytest.mark.parametrize("numels,precision", [([300_000, 1234, 77], "bf16"), ([2048 * 5 + 64], "bf16"), ([64], "bf16"),
                                              ([70_001, 3], "fp32")])
def test_parameters_first_then_moments_bit_exact(rmode, numels, precision):
    wl = W.tiny_workload(numels, dp_size=2, dp_rank=1, precision=precision, grad_kind="heavy_tail",
                         hyper=W.Hyper(max_grad_norm=0.05))
    s, o, gdev, gbits = make_pair(wl, steps=6, chunk_bytes=64 << 10, restore_mode=rmode)
    hp = hp_of(wl)
    cur, side = torch.cuda.current_stream(), torch.cuda.Stream(device=DEV)
    run_with_flushes(s, o, gdev, gbits, hp, 4, side)
    s.step_and_snapshot(gdev[4], 5)                  # in flight when the fault hits; its work is discarded (I4)
    s.drop_live()
    o.drop_live()
    s.m.fill_(123.0)                                 # sentinels: a step that did not wait for the moments would use them
    s.v.fill_(0.5)
    side.wait_stream(cur)                            # the fault (test code on `cur`) precedes the recovery
    with torch.cuda.stream(side):
        torch.cuda._sleep(HOLD)                      # the whole restore starts late ...
    assert s.restore_async(side) == 4                # ... but the call only enqueues
    assert B.phx_last_step(s.h) == 4
    s.restore_wait_params(cur)
    p_then = s.p.clone()                             # enqueued on the compute stream right behind "parameters ready"
    p16_then = None if s.p16 is None else s.p16.clone()
    s.step_and_snapshot(gdev[4], 5)                  # recompute of the in-flight step: waits for m and v by itself
    assert o.restore_params_first() == 4
    torch.cuda.synchronize()
    assert np.array_equal(p_then.cpu().numpy().view(np.uint32), o.p.view(np.uint32))
    if p16_then is not None:
        assert np.array_equal(bits16(p16_then), o.p16)
    assert o.restore_finish() == 4
    o.step(gbits[4], **hp, step=5)
    assert_state_equal(s, o, "recompute after the two-phase restore")
    s.flush_async(side)
    o.snapshot()
    s.step_and_snapshot(gdev[5], 6)
    o.step(gbits[5], **hp, step=6)
    assert_state_equal(s, o, "step 6")
    s.wait(5)
    assert np.array_equal(s.replica_slot(5).numpy(), o.replica[1])
    s.close()


@pytest.mark.parametrize("rmode", RMODES)
@pytest.mark.parametrize("torn", [0, 1, 5])
def test_torn_newest_flush_falls_back_in_both_phases(rmode, torn):
    wl = W.tiny_workload([200_000, 77], dp_size=1)
    s, o, gdev, gbits = make_pair(wl, steps=5, chunk_bytes=64 << 10, restore_mode=rmode)
    hp = hp_of(wl)
    side = torch.cuda.Stream(device=DEV)
    run_with_flushes(s, o, gdev, gbits, hp, 4, side, torn_last=torn)
    s.drop_live()
    o.drop_live()
    assert s.restore_async(side) == 3
    assert o.restore_params_first() == 3 and o.restore_finish() == 3
    for t in (4, 5):
        s.step_and_snapshot(gdev[t - 1], t)
        o.step(gbits[t - 1], **hp, step=t)
    assert_state_equal(s, o, "resumed after a torn flush")
    s.close()


@pytest.mark.parametrize("rmode", RMODES)
def test_one_phase_restore_and_graph_form_order_behind_an_outstanding_two_phase_restore(rmode):
    wl = W.tiny_workload([150_000, 4097], dp_size=1)
    s, o, gdev, gbits = make_pair(wl, steps=6, chunk_bytes=64 << 10, restore_mode=rmode)
    hp = hp_of(wl)
    cur, side = torch.cuda.current_stream(), torch.cuda.Stream(device=DEV)
    run_with_flushes(s, o, gdev, gbits, hp, 3, side)
    s.drop_live()
    side.wait_stream(cur)                            # the fault (test code on `cur`) precedes the recovery
    with torch.cuda.stream(side):
        torch.cuda._sleep(HOLD)
    assert s.restore_async(side) == 3
    s.p.fill_(9.0)                                   # on `cur`, not ordered against the side stream: lost or overwritten
    assert s.restore(cur) == 3                       # the one-phase restore orders itself behind the outstanding one
    o.restore()
    assert_state_equal(s, o, "restore after restore_async")
    # graph form right after a two-phase restore: phx_graph_begin settles it
    s.drop_live()
    side.wait_stream(cur)                            # the fault (test code on `cur`) precedes the recovery
    with torch.cuda.stream(side):
        torch.cuda._sleep(HOLD)
    assert s.restore_async(side) == 3
    s.graph_begin()
    for t in (4, 5):
        s.graph_step(gdev[t - 1])
        o.step(gbits[t - 1], **hp, step=t)
    assert s.graph_end() == 5
    assert_state_equal(s, o, "graph-form steps after the two-phase restore")
    B.phx_restore_wait_params(s.h, cur)              # nothing outstanding: a no-op
    s.close()


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("rmode", RMODES)
def test_full_rank_state_brings_W_back_with_the_parameters(rmode, precision):
    D, numels = 3, [30_000, 4097, 64]
    wls, shards, ranks = build_group(numels, D, precision=precision, restore_mode=rmode)
    streams = [torch.cuda.Stream(device=DEV) for _ in range(2)]
    for t in range(1, 4):
        iteration(wls, shards, ranks, t, streams)
    victim, vfr = shards[1], ranks[1]
    victim.wait(3)
    victim.drop_live()
    vfr.drop_live()
    cur, side = torch.cuda.current_stream(), streams[0]
    side.wait_stream(cur)                            # the fault (test code on `cur`) precedes the recovery
    with torch.cuda.stream(side):
        torch.cuda._sleep(HOLD)
    assert victim.restore_async(side) == 3
    victim.restore_wait_params(cur)
    W_then = victim.W.clone()
    assert vfr.restore_in_place_params_first() == 3
    torch.cuda.synchronize()
    got = W_then.cpu().numpy().view(np.uint8) if victim.fp32 else bits16(W_then).view(np.uint8)
    assert np.array_equal(got, vfr.W.view(np.uint8))
    assert vfr.restore_in_place_finish() == 3
    assert_state_equal(victim, vfr.o, "full rank state, two phases")
    assert np.array_equal(w_bits(victim), vfr.W.view(np.uint8))
    for t in (4, 5):                                 # the group goes on; the recovered rank is indistinguishable
        iteration(wls, shards, ranks, t, streams)
    for s, fr in zip(shards, ranks):
        s.wait(5)
        assert_state_equal(s, fr.o, f"rank {fr.r} after recovery")
        assert np.array_equal(s.replica_slot(5).numpy(), fr.slots[1])
    close_all(shards)


def test_protocol_errors():
    wl = W.tiny_workload([1000], dp_size=1)
    s, o, gdev, gbits = make_pair(wl, steps=1)
    L = B.lib()
    assert L.phx_restore_async(None, None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_restore_wait_params(None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_restore_async(s.h, None, None) == B.PHX_ERR_NO_COMMITTED_SNAPSHOT
    s.graph_begin()
    assert L.phx_restore_async(s.h, None, None) == B.PHX_ERR_GRAPH_MODE
    s.graph_end()
    s.close()
