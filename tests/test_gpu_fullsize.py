"""Whole-array parity at FULL size, in the launch configuration bench.py times: for every
BASELINE.json config of bandwidth size — c2, c3 (with the clip), c4a, c4b, c5 — and for c2 in the paper's own
precision with decay groups, three steps are run on the GPU and by the oracle (all host cores) on the same
seeded inputs, and EVERY element of p, m, v, the bf16 copy and the committed replica slot is compared, bit for
bit.  No sampling: the oracle does ~3.5 G elements/s on the box's cores.  c3 then takes a fourth step through the
gradient producer's epilogue (clip_source = producer), also compared whole.

Also here: a real in-flight fault (the drop is issued from a SECOND stream, unsynchronised, while step k+1's
kernel and the flush of snapshot k are running at c2 size).  (The > 2^32-element shard with its dense block
straddling element 2^32 is tests/test_gpu_huge.py.)"""
import os

import numpy as np
import pytest
import torch

from oracle import grad_finalize as GF
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, bits16, hp_of

pytestmark = pytest.mark.gpu
CORES = len(os.sched_getaffinity(0))


def i32(t: torch.Tensor) -> torch.Tensor:
    return t.detach().view(torch.int32).cpu()


def assert_whole_equal(dev: torch.Tensor, ref: np.ndarray, what):
    """Bit compare of a whole device plane with the oracle's array (int views: -0.0 != 0.0, NaN == NaN)."""
    if dev.dtype == torch.bfloat16:
        got, exp = dev.detach().view(torch.int16).cpu(), torch.from_numpy(ref.view(np.int16))
    else:
        got, exp = i32(dev), torch.from_numpy(ref.view(np.int32))
    if not torch.equal(got, exp):
        bad = torch.nonzero(got != exp).flatten()
        raise AssertionError(f"{what}: {bad.numel()} of {exp.numel()} lanes differ, first {bad[:5].tolist()}")


def assert_replica_is_oracle_snapshot(s: Shard, o: O.OracleShard, step: int, what):
    """Committed host slot == the oracle's packed snapshot header ‖ p ‖ m ‖ v, all bytes."""
    rep = s.replica_slot(step)
    N4 = 4 * s.n_padded
    assert bytes(rep[:256].numpy().tobytes()) == o._header(True), what
    for k, plane in enumerate((o.p, o.m, o.v)):
        got = rep[256 + k * N4:256 + (k + 1) * N4].view(torch.int32)
        assert torch.equal(got, torch.from_numpy(plane.view(np.int32))), (what, "pmv"[k])


def run_config(wl, steps=3, **shard_kw):
    fp32 = wl.precision == "fp32"
    s = Shard(wl, device=DEV, **shard_kw)              # library defaults = the launch configuration bench.py times
    N = s.n_padded
    o = O.OracleShard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank), (wl.pp_size, wl.pp_rank),
                      chunk_bytes=32 << 20, max_grad_norm=wl.hyper.max_grad_norm, flags=wl.flags(),
                      precision=wl.precision)
    assert (o.n, o.n_padded) == (s.n, N) and o.n == wl.n_expected
    p0 = W.init_params(s.n, N, wl.seed, device=DEV)
    s.p.copy_(p0)
    s.set_state(0)
    o.set_state(p0.cpu().numpy())
    del p0
    side = torch.cuda.Stream(device=DEV)
    hp = hp_of(wl)
    for t in range(1, steps + 1):
        g = W.gen_grads(wl, s.segments, N, t, wl.seed, device=DEV, dtype=torch.float32 if fp32 else torch.bfloat16)
        s.step_and_snapshot(g, t)
        s.flush_async(side)
        grec = g.cpu().numpy() if fp32 else bits16(g)
        o.step(grec, **hp, step=t, nthreads=CORES)
        if wl.hyper.max_grad_norm > 0:
            coef, S = B.phx_last_clip(s.h)
            assert np.float32(coef) == o.last_coef, (t, coef, o.last_coef)      # bitwise
            assert abs(S - O.sumsq(grec)) <= 1e-13 * S
        for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v)):
            assert_whole_equal(dev, ref, f"{wl.key} step {t} {name}")
        if not fp32:
            assert_whole_equal(s.p16, o.p16, f"{wl.key} step {t} p16")
        s.wait(t)
        assert_replica_is_oracle_snapshot(s, o, t, f"{wl.key} replica of step {t}")
        del g, grec
    return s, o, side


@pytest.mark.parametrize("key", ["c2", "c3", "c4a", "c4b", "c5"])
def test_whole_array_parity_full_size(key):
    wl = W.CONFIGS[key]
    s, o, side = run_config(wl)
    N = s.n_padded
    hp = hp_of(wl)
    if key == "c3":
        # step 4 through the gradient producer's epilogue: fp32 main gradients -> bf16 + sum of squares, one pass,
        # and a step with no a1 pass of its own (clip_source = producer)
        g32 = W.gen_grads(wl, s.segments, N, 4, wl.seed, device=DEV, dtype=torch.float32)
        g16 = torch.empty(N, dtype=torch.bfloat16, device=DEV)
        S = torch.zeros(1, dtype=torch.float64, device=DEV)
        s.grads_finalize(g32, 1.0, g16, S)
        B.phx_set_clip_partials(s.h, S, 1)
        l0 = B.phx_kernel_launches(s.h)
        s.step_and_snapshot(g16, 4)
        assert B.phx_kernel_launches(s.h) - l0 == 2
        s.flush_async(side)
        bits, So = GF.grads_finalize(g32.cpu().numpy(), 1.0)
        assert torch.equal(g16.view(torch.int16).cpu(), torch.from_numpy(bits.view(np.int16)))
        coef, Sg = B.phx_last_clip(s.h)
        assert abs(Sg - So) <= 4 * np.spacing(So)
        o.step(bits, **hp, step=4, nthreads=CORES)
        assert np.float32(coef) == o.last_coef
        for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v), ("p16", s.p16, o.p16)):
            assert_whole_equal(dev, ref, f"c3 producer step {name}")
        s.wait(4)
        assert_replica_is_oracle_snapshot(s, o, 4, "c3 replica of the producer step")
        del g32, g16
    # restore(snapshot(s)) == s on every element
    last = o.last_step
    s.drop_live()
    assert s.restore() == last
    for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v), ("p16", s.p16, o.p16)):
        assert_whole_equal(dev, ref, f"{key} restored {name}")
    # ... and through the two-phase restore (parameters first on the side stream, moments behind them)
    s.drop_live()
    side.wait_stream(torch.cuda.current_stream())
    assert s.restore_async(side) == last
    s.restore_wait_params()
    assert_whole_equal(s.p16, o.p16, f"{key} two-phase restore, p16 at 'parameters ready'")
    torch.cuda.synchronize()
    for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v), ("p16", s.p16, o.p16)):
        assert_whole_equal(dev, ref, f"{key} two-phase restored {name}")
    s.close()


def test_whole_array_parity_c2_paper_precision_with_decay_groups():
    import dataclasses
    wl = dataclasses.replace(W.CONFIGS["c2"], precision="fp32", decay_groups=True)
    s, o, _ = run_config(wl)
    assert s.p16 is None and o.no_decay is not None and o.no_decay.any()
    s.close()


# ------------------------------------------------------------------------------------------------------------
# a real in-flight fault at c2 size (SURVEY.md:241 fault phases; I3/I4 PAPER.md:168-169)
# ------------------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("mode,depth,torn", [(B.PHX_SYNC_STRICT, 2, None), (B.PHX_SYNC_RELAXED, 3, None),
                                             (B.PHX_SYNC_RELAXED, 3, 40), (B.PHX_SYNC_RELAXED, 4, 0)])
def test_drop_from_a_second_stream_while_kernel_and_flush_are_in_flight(mode, depth, torn):
    """The fault lands with NO host synchronisation, on a second stream that only waits for step k's kernel: at
    that moment flush(k) (and, relaxed, earlier flushes) is being DMA'd and step k+1's kernel is queued behind the
    sync point (strict) or running beside the flushes (relaxed); the fault zeroes the live planes and scribbles
    the staging slot of step k+1, racing all of it.  Restore must return k — or k-1 when flush(k) was torn —
    with every element equal to the oracle's state of that step, and the replay must rejoin the trajectory."""
    wl = W.CONFIGS["c2"]
    hp = hp_of(wl)
    s = Shard(wl, device=DEV, staging_depth=depth, sync_mode=mode, chunk_bytes=4 << 20)
    N = s.n_padded
    o = O.OracleShard(wl.layout(), wl.dp_size, wl.dp_rank, chunk_bytes=4 << 20)
    p0 = W.init_params(s.n, N, wl.seed, device=DEV)
    s.p.copy_(p0); s.set_state(0); o.set_state(p0.cpu().numpy())
    del p0
    grads = [W.gen_grads(wl, s.segments, N, t, wl.seed, device=DEV) for t in (1, 2, 3, 4)]
    gbits = [bits16(g) for g in grads]
    cur = torch.cuda.current_stream()
    side, fault = torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV)
    k = 3
    states = {}
    for t in range(1, k + 1):
        o.step(gbits[t - 1], **hp, step=t, nthreads=CORES)
        states[t] = (o.p.copy(), o.m.copy(), o.v.copy(), o.p16.copy())
    torch.cuda.synchronize()
    after_k = torch.cuda.Event()
    for t in range(1, k + 1):
        s.step_and_snapshot(grads[t - 1], t)
        if t == k:
            after_k.record(cur)
            if torn is not None:
                B.phx_fault_inject_torn_flush(s.h, torn)  # flush(k) dies after `torn` payload chunks
        s.flush_async(side)                               # ~36 ms of DMA each; nothing waits on the host
    s.step_and_snapshot(grads[k], k + 1)                  # step k+1: launched, in flight
    fault.wait_event(after_k)                             # the fault lands once step k's kernel has finished, i.e. WHILE
    with torch.cuda.stream(fault):                        # flush(k) is being DMA'd and step k+1 is queued / running; no host sync
        for x in (s.p, s.m, s.v, s.p16):
            x.zero_()
        s.staging_slot(k + 1).fill_(0xA5)
    cur.wait_stream(fault)                                # recovery starts after the fault (device-side order only)
    back = s.restore()
    want = k if torn is None else k - 1
    assert back == want
    ref = states[want]
    for name, dev, r in (("p", s.p, ref[0]), ("m", s.m, ref[1]), ("v", s.v, ref[2]), ("p16", s.p16, ref[3])):
        got = dev.view(torch.int16 if dev.dtype == torch.bfloat16 else torch.int32).cpu()
        exp = torch.from_numpy(r.view(np.int16 if dev.dtype == torch.bfloat16 else np.int32))
        assert torch.equal(got, exp), (mode, depth, torn, name)
    # replay rejoins the uninterrupted trajectory (GPU vs oracle, whole arrays)
    o.step(gbits[k], **hp, step=k + 1, nthreads=CORES)
    for t in range(want + 1, k + 2):
        s.step_and_snapshot(grads[t - 1], t)
        s.flush_async(side)
    s.wait(k + 1)
    for name, dev, r in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v), ("p16", s.p16, o.p16)):
        assert_whole_equal(dev, r, f"replayed {name}")
    assert_replica_is_oracle_snapshot(s, o, k + 1, "replica after the replay")
    s.close()
