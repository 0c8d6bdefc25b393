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
