"""Pins of the ring oracle against the paper: the loss condition of
PAPER.md:175, Eq. (1) P_loss <= D p^(k+1) and the value the paper prints for
D = 128, k = 1; plus the byte-level invariants of the H2H phase.  CPU only."""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O
from oracle import ring as R

HP = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "ploss_pins.txt")


def test_ring_peers_are_distinct_successors():
    for D in range(2, 9):
        for r in range(D):
            for k in range(1, D):
                hs = R.holders(D, r, k)
                assert len(set(hs)) == k and r not in hs
                assert hs == [(r + j) % D for j in range(1, k + 1)]
                # predecessor j of the holder is the owner
                assert all(R.ring_peer(D, h, -(j + 1)) == r for j, h in enumerate(hs))
    with pytest.raises(AssertionError):
        R.holders(4, 0, 4)          # k distinct peers need k <= D - 1


def test_loss_condition_brute_force_matches_the_papers_statement():
    # lost only if the owner AND all k holders fail within the same step
    for D, k in ((4, 1), (5, 2), (6, 1), (6, 3), (7, 2)):
        for m in range(D + 1):
            for failed in itertools.combinations(range(D), m):
                f = set(failed)
                lost = any(all(((r + j) % D) in f for j in range(1, k + 1)) for r in f)
                assert R.recoverable(D, k, failed) == (not lost)
        # the smallest unrecoverable sets are exactly the D runs of k+1 consecutive ranks
        bad = [c for c in itertools.combinations(range(D), k + 1) if not R.recoverable(D, k, c)]
        assert len(bad) == D
        assert all(R.recoverable(D, k, c) for m in range(k + 1) for c in itertools.combinations(range(D), m))


def test_equation_1_union_bound_in_exact_rationals():
    # Eq. (1): P_loss <= D * p^(k+1); tight to first order for small p
    for D, k in ((4, 1), (5, 2), (6, 1), (8, 2), (8, 3)):
        for p in (Fraction(1, 10), Fraction(1, 1000), Fraction(1, 10 ** 6)):
            exact = R.p_loss_exact(D, k, p)
            bound = D * p ** (k + 1)
            assert 0 < exact <= bound
            if p <= Fraction(1, 1000):
                assert exact >= bound * (1 - (D + 1) * p)      # the bound is the leading term


def test_papers_printed_loss_probabilities():
    # tests/golden/ploss_pins.txt: values printed at PAPER.md:181 and PAPER.md:189
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for D, k, p, steps, printed in rows:
        D, k, steps = int(D), int(k), int(steps)
        p, printed = Fraction(p), float(printed)
        bound = float(D * p ** (k + 1) * steps)
        assert abs(bound - printed) <= 5e-3 * printed, (D, k, bound, printed)


def _ring(D=4, k=2, numels=(1000, 333, 77), chunk=1024, seed=0, **kw):
    layout = [(n, i) for i, n in enumerate(numels)]
    ring = R.OracleRing(layout, D, k, chunk_bytes=chunk, **kw)
    rng = np.random.default_rng(seed)
    for o in ring.shards:
        p0 = np.zeros(o.n_padded, np.float32)
        p0[:o.n] = rng.normal(0, 0.02, o.n)
        o.set_state(p0)
    return ring, rng


def _grads(ring, rng, fp32=False):
    out = []
    for o in ring.shards:
        g = np.zeros(o.n_padded, np.float32)
        g[:o.n] = rng.normal(0, 1e-3, o.n)
        out.append(g if fp32 else (g.view(np.uint32) >> 16).astype(np.uint16))
    return out


def _step_all(ring, gs, t, replicate=True):
    for r, o in enumerate(ring.shards):
        if ring.alive[r]:
            o.step(gs[r], **HP, step=t)
            o.snapshot()
            if replicate:
                ring.replicate(r)


def test_received_slots_are_byte_identical_to_the_owners_local_slots():
    ring, rng = _ring()
    for t in range(1, 4):
        _step_all(ring, _grads(ring, rng), t)
        for r, o in enumerate(ring.shards):
            for j in range(1, ring.k + 1):
                h = R.ring_peer(ring.D, r, j)
                assert np.array_equal(ring.received[h][j - 1][t % 2], o.replica[t % 2])     # R26
                assert np.array_equal(ring.received[h][j - 1][t % 2], o.packed_snapshot())
    # what a holder keeps for two different predecessors differs (their shards differ)
    assert not np.array_equal(ring.received[2][0][1], ring.received[2][1][1])


@pytest.mark.parametrize("failed", [(1,), (0, 1), (1, 3), (3, 0)])
def test_recovery_from_surviving_holder_resumes_the_uninterrupted_trajectory(failed):
    D, k = 4, 2
    ring, rng = _ring(D, k, seed=3)
    ref, _ = _ring(D, k, seed=3)
    gs_all = [_grads(ring, rng) for _ in range(8)]
    for t in range(1, 9):
        _step_all(ref, gs_all[t - 1], t, replicate=False)
    for t in range(1, 6):
        _step_all(ring, gs_all[t - 1], t)
    # step 6 is in flight on the failing ranks when they die: partial work is discarded (I4)
    for r in failed:
        ring.shards[r].step(gs_all[5][r], **HP, step=6)
    ring.fail(failed)
    assert R.recoverable(D, k, failed)
    for r in failed:
        assert ring.recover(r) == 5
    for r in range(D):
        if r not in failed:                                   # survivors had not started step 6
            ring.shards[r].step(gs_all[5][r], **HP, step=6)
    for r in failed:
        ring.shards[r].step(gs_all[5][r], **HP, step=6)       # recompute of the in-flight step
    for t in (7, 8):
        for r, o in enumerate(ring.shards):
            o.step(gs_all[t - 1][r], **HP, step=t)
    for a, b in zip(ring.shards, ref.shards):
        for x, y in ((a.p, b.p), (a.m, b.m), (a.v, b.v), (a.p16, b.p16)):
            assert np.array_equal(x.view(np.uint8), y.view(np.uint8))


def test_owner_and_all_holders_failing_loses_the_shard():
    ring, rng = _ring(4, 1)
    _step_all(ring, _grads(ring, rng), 1)
    ring.fail((1, 2))                       # rank 1's only holder is rank 2
    assert not R.recoverable(4, 1, (1, 2))
    with pytest.raises(O.OracleError):
        ring.recover(1)
    assert ring.recover(2) == 1             # rank 2's holder (rank 3) survived


def test_torn_peer_transfer_leaves_the_previous_received_slot_usable():
    ring, rng = _ring(3, 2, numels=(5000,), chunk=4096)
    _step_all(ring, _grads(ring, rng), 1)
    gs = _grads(ring, rng)
    for r, o in enumerate(ring.shards):
        o.step(gs[r], **HP, step=2)
        o.snapshot()
    ring.replicate(0, abort_after_chunks={1: 1, 2: 0})     # both transfers of rank 0's step 2 are torn
    ring.replicate(1)
    ring.replicate(2)
    ring.fail((0,))
    h, j, s, hd = ring.newest_replica_of(0)
    assert hd["step"] == 1 and s == 1                       # the torn slot (step 2 -> slot 0) is never chosen
    assert ring.recover(0) == 1
    # a torn transfer to ONE peer only: the other holder has the newer step
    ring2, rng2 = _ring(3, 2, numels=(5000,), chunk=4096)
    _step_all(ring2, _grads(ring2, rng2), 1)
    gs = _grads(ring2, rng2)
    for r, o in enumerate(ring2.shards):
        o.step(gs[r], **HP, step=2)
        o.snapshot()
        ring2.replicate(r, abort_after_chunks={1: 2} if r == 0 else None)
    ring2.fail((0,))
    assert ring2.newest_replica_of(0)[:2] == (2, 2) and ring2.recover(0) == 2


def test_holder_refuses_a_foreign_layout():
    ring, rng = _ring(3, 1)
    _step_all(ring, _grads(ring, rng), 1)
    ring.fail((0,))
    ring.shards[0] = O.OracleShard([(1000, 0), (333, 1), (78, 2)], 3, 0)     # a different logical shard
    with pytest.raises(O.OracleError):
        ring.recover(0)


# ---------------------------------------------------------------------------- §8(f3) publication


def test_publication_is_the_rounded_flat_master_in_rank_order():
    import torch
    D = 3
    ring, rng = _ring(D, 1, numels=(1000, 333, 77), seed=5)
    for t in range(1, 4):
        _step_all(ring, _grads(ring, rng), t)
    W = R.publish(ring.shards)
    L = ring.shards[0].n_padded
    assert W.dtype == np.uint16 and W.size == D * L
    flat = np.concatenate([o.p for o in ring.shards])                      # the flat padded master space of a0
    want = torch.from_numpy(flat).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(W, want)                                         # library cast (torch, RNE)
    # element i of tensor t sits where a0 says: rank = flat // L, offset = flat % L
    total = ring.shards[0].total_numel
    assert not W[total:].any()                                             # padding of the flat space stays zero
    for r, o in enumerate(ring.shards):
        for tid, off_t, off_s, ln in o.segments:
            start = sum(n for n, i in o.layout if i < tid) + off_t         # flat index of the segment's first element
            assert np.array_equal(W[start:start + ln], o.p16[off_s:off_s + ln])
            assert start == r * L + off_s


def test_publication_fp32_precision_is_the_master_itself():
    ring, rng = _ring(2, 1, numels=(500, 70), precision="fp32")
    _step_all(ring, _grads(ring, rng, fp32=True), 1)
    W = R.publish(ring.shards)
    assert W.dtype == np.float32
    assert np.array_equal(W.view(np.uint32), np.concatenate([o.p for o in ring.shards]).view(np.uint32))


def test_parameter_reconstruction_from_a_surviving_rank():
    D = 4
    ring, rng = _ring(D, 2, seed=6)
    _step_all(ring, _grads(ring, rng), 1)
    W = R.publish(ring.shards)
    bufs = [W.copy() for _ in range(D)]                                    # every DP rank holds the same bytes (I2)
    ring.fail((1, 2))
    bufs[1][:] = 0
    bufs[2][:] = 0
    got = R.reconstruct_params(bufs, ring.alive, 1)                        # successors 2 (dead), 3 (alive)
    assert np.array_equal(got, W)
    assert ring.recover(1) == 1
    L = ring.shards[1].n_padded
    assert np.array_equal(got[L:2 * L], ring.shards[1].p16)                # consistent with the restored optimizer shard
    with pytest.raises(O.OracleError):
        R.reconstruct_params(bufs, [False] * D, 0)
