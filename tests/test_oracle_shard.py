"""Pins of the oracle's shard definition (a0), envelope, snapshot (a4/a5), restore (a6)
and resume (a7): brute force on tiny inputs, architecture arithmetic of the configs, and the
invariants BASELINE.json:north_star lists — restore(snapshot(s)) == s bit-exactly; training
resumed from a restored shard reproduces the uninterrupted trajectory bit-exactly; the
snapshot bytes equal the live shard bit-exactly.  CPU only.
"""
import itertools

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import workloads as W

HP = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)


def tbits(t: torch.Tensor) -> np.ndarray:
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def make(wl, **kw):
    return O.OracleShard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank),
                         (wl.pp_size, wl.pp_rank), **kw)


def seeded(wl, steps, **kw):
    s = make(wl, **kw)
    s.set_state(W.init_params(s.n, s.n_padded, wl.seed).numpy())
    segs = [(tid, off, ln) for tid, _, off, ln in s.segments]
    gs = [tbits(W.gen_grads(wl, segs, s.n_padded, t, wl.seed)) for t in range(1, steps + 1)]
    return s, gs


def state_bytes(s):
    return b"".join(a.tobytes() for a in (s.p, s.m, s.v, s.p16)) + bytes([s.last_step % 256])


# ---------------------------------------------------------------------------- a0


@pytest.mark.parametrize("numels,dp", [([5], 1), ([100, 3, 64, 1], 3), ([63, 1, 64, 129], 2),
                                       ([1000, 24, 7], 4), ([64 * 4], 4), ([1], 5)])
def test_partition_brute_force(numels, dp):
    layout = [(n, 10 + i) for i, n in enumerate(numels)]
    total = sum(numels)
    # brute force: element e of the flat space belongs to tensor owner[e] at offset within[e]
    owner = np.concatenate([np.full(n, 10 + i) for i, n in enumerate(numels)])
    within = np.concatenate([np.arange(n) for n in numels])
    seen = np.zeros(total, int)
    Ls = set()
    n_sum = 0
    for r in range(dp):
        d = O.define_shard(layout, dp, r)
        L = d["n_padded"]
        Ls.add(L)
        assert L % 64 == 0 and d["shard_begin"] == r * L and d["total_numel"] == total
        assert L * dp >= total and (L - 64) * dp < total  # smallest multiple of 64 that covers
        assert d["n"] == min(max(total - r * L, 0), L)
        n_sum += d["n"]
        cover = 0
        for tid, off_t, off_s, ln in d["segments"]:
            lo = d["shard_begin"] + off_s
            assert np.all(owner[lo:lo + ln] == tid)
            assert np.array_equal(within[lo:lo + ln], np.arange(off_t, off_t + ln))
            seen[lo:lo + ln] += 1
            assert off_s == cover  # segments are contiguous from 0 and ordered
            cover += ln
        assert cover == d["n"]
    assert len(Ls) == 1 and n_sum == total and np.all(seen == 1)


def test_layout_hash_separates_layouts():
    base = O.define_shard([(100, 0), (28, 1)], 2, 0)["layout_hash"]
    assert O.define_shard([(100, 0), (28, 1)], 2, 1)["layout_hash"] == base  # rank is a coordinate
    others = [O.define_shard([(28, 0), (100, 1)], 2, 0), O.define_shard([(100, 0), (28, 2)], 2, 0),
              O.define_shard([(128, 0)], 2, 0), O.define_shard([(100, 0), (28, 1)], 4, 0),
              O.define_shard([(100, 0), (28, 1)], 2, 0, tp=(2, 0)),
              O.define_shard([(100, 0), (28, 1)], 2, 0, pp=(2, 1))]
    hs = {o["layout_hash"] for o in others}
    assert base not in hs and len(hs) == len(others)
    assert O.fnv1a64(b"") == 0xCBF29CE484222325 and O.fnv1a64(b"a") == 0xAF63DC4C8601EC8C  # published FNV-1a vectors


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4a", "c4b", "c5"])
def test_config_shard_sizes_match_the_configs(key):
    wl = W.CONFIGS[key]
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank)
    assert d["n"] == wl.n_expected == d["n_padded"]
    totals = dict(c1=5_289_472, c2=1_315_819_520, c3=6_738_415_616, c4a=3_254_067_200,
                  c4b=3_254_067_200, c5=1_044_807_680)  # SURVEY.md Appendix C arithmetic
    assert wl.total_numel == totals[key]


# ---------------------------------------------------------------------------- envelope


def test_header_roundtrip_and_rejection():
    kw = dict(step=7, n=100, n_padded=128, total_numel=500, shard_begin=128, layout_hash=0x1234,
              dp=(4, 1), tp=(2, 0), pp=(2, 1), chunk_bytes=1 << 22, user=b"rng-state-\x00\x01\x02")
    raw = O.pack_header(**kw)
    assert len(raw) == 256 and raw[:8] == b"PHXSNAP1"
    h = O.parse_header(raw)
    assert h["step"] == 7 and h["dp"] == (4, 1) and h["tp"] == (2, 0) and h["pp"] == (2, 1)
    assert h["user"] == kw["user"] and h["layout_hash"] == 0x1234 and h["n"] == 100
    assert O.parse_header(O.pack_header(**kw, committed=False)) is None   # seq_end != seq_begin
    assert O.parse_header(bytes(256)) is None
    for pos in (0, 9, 17, 40, 100, 130, 241, 250):
        bad = bytearray(raw)
        bad[pos] ^= 0x40
        assert O.parse_header(bytes(bad)) is None, pos


# ---------------------------------------------------------------------------- snapshot / restore


def test_snapshot_bytes_equal_live_and_restore_roundtrip():
    wl = W.tiny_workload([1000, 37, 2048, 5], dp_size=2, dp_rank=1)
    s, gs = seeded(wl, 4, chunk_bytes=4096, user=b"envelope")
    for t, g in enumerate(gs, 1):
        s.step(g, **HP, step=t)
        slot = s.snapshot()
        assert slot == t % 2
        raw = s.replica[slot]
        N4 = 4 * s.n_padded
        assert raw[256:256 + N4].tobytes() == s.p.tobytes()
        assert raw[256 + N4:256 + 2 * N4].tobytes() == s.m.tobytes()
        assert raw[256 + 2 * N4:].tobytes() == s.v.tobytes()
        assert raw.tobytes() == s.packed_snapshot().tobytes()
        before = state_bytes(s)
        s.drop_live()
        assert s.restore() == t and s.restored_user == b"envelope"
        assert state_bytes(s) == before  # incl. regenerated p16 == p16 before the fault


def test_torn_slot_is_never_chosen_and_previous_slot_survives():
    wl = W.tiny_workload([5000], dp_size=1)
    s, gs = seeded(wl, 3, chunk_bytes=2048)
    s.step(gs[0], **HP, step=1); s.snapshot()
    s.step(gs[1], **HP, step=2); s.snapshot()
    after2 = state_bytes(s)
    s.step(gs[2], **HP, step=3)
    nchunks = -(-12 * s.n_padded // 2048)
    for j in (0, 1, nchunks // 2, nchunks):          # interrupted after j of N chunks
        s.snapshot(abort_after_chunks=j)             # targets slot 1 (held step 1)
        assert O.parse_header(s.replica[1][:256].tobytes()) is None
        got = s.newest_committed()
        assert got is not None and got[0] == 0 and got[1]["step"] == 2
    s.drop_live()
    assert s.restore() == 2 and state_bytes(s) == after2


def test_restore_refuses_foreign_replica_and_empty_replica():
    a = W.tiny_workload([1000, 24], dp_size=2, dp_rank=0)
    s, gs = seeded(a, 1)
    with pytest.raises(O.OracleError):
        s.restore()                                   # nothing committed yet
    s.step(gs[0], **HP, step=1); s.snapshot()
    for other in (W.tiny_workload([1000, 24], dp_size=2, dp_rank=1),
                  W.tiny_workload([24, 1000], dp_size=2, dp_rank=0)):
        o = make(other)
        assert o.snapshot_bytes == s.snapshot_bytes
        o.replica = s.replica
        with pytest.raises(O.OracleError):
            o.restore()                               # logical identity differs


def test_step_order_is_enforced():
    s, gs = seeded(W.tiny_workload([100], 1), 2)
    with pytest.raises(O.OracleError):
        s.step(gs[0], **HP, step=2)
    s.step(gs[0], **HP, step=1)
    with pytest.raises(O.OracleError):
        s.step(gs[1], **HP, step=1)


@pytest.mark.parametrize("fault_at,torn", [(1, False), (5, False), (5, True), (9, False)])
def test_resume_equals_uninterrupted(fault_at, torn):
    wl = W.tiny_workload([3000, 100, 977], dp_size=2, dp_rank=0,
                         hyper=W.Hyper(max_grad_norm=0.05))
    T = 10
    ref, gs = seeded(wl, T, chunk_bytes=4096, max_grad_norm=0.05)
    for t in range(1, T + 1):
        ref.step(gs[t - 1], **HP, step=t)
    s, _ = seeded(wl, 0, chunk_bytes=4096, max_grad_norm=0.05)
    t = 1
    faulted = False
    while t <= T:
        s.step(gs[t - 1], **HP, step=t)
        if t == fault_at and not faulted:
            # fault while step t is in flight: live state partly mutated, nothing of t committed
            faulted = True
            s.p[::3] = 7.0
            s.drop_live()
            if fault_at == 1 and not torn:
                with pytest.raises(O.OracleError):
                    s.restore()
                # no replica yet: restart from the initial state (outside the hot path)
                s.set_state(W.init_params(s.n, s.n_padded, wl.seed).numpy())
                t = 1
                continue
            back = s.restore()
            assert back == (t - 2 if torn else t - 1)   # replay <= 1 step, 2 if flush(t-1) tore
            t = back + 1
            continue
        if torn and t == fault_at - 1 and not faulted:
            s.snapshot(abort_after_chunks=2)            # flush(t) interrupted at chunk 2 (R17 variant)
        else:
            s.snapshot()
        t += 1
    assert state_bytes(s) == state_bytes(ref)


def test_pad_lanes_stay_zero():
    wl = W.tiny_workload([70], dp_size=1)               # n = 70, n_padded = 128
    s, gs = seeded(wl, 10)
    assert s.n == 70 and s.n_padded == 128
    for t, g in enumerate(gs, 1):
        assert not g[70:].any()
        s.step(g, **HP, step=t)
        for a in (s.p, s.m, s.v, s.p16):
            assert not a[70:].view(np.uint8).any()
            assert a[:70].view(np.uint8).any()


def test_c1_ten_steps_snapshot_restore_resume():
    """BASELINE.json:configs[0] on the oracle alone: 10 steps, snapshot after every step,
    restore-and-compare, then fault at step 5 and resume to 10."""
    wl = W.CONFIGS["c1"]
    ref, gs = seeded(wl, 10)
    for t in range(1, 11):
        ref.step(gs[t - 1], **HP, step=t, nthreads=4)
        ref.snapshot()
        b = state_bytes(ref)
        ref.drop_live(); ref.restore()
        assert state_bytes(ref) == b
    s, _ = seeded(wl, 0)
    for t in range(1, 6):
        s.step(gs[t - 1], **HP, step=t, nthreads=4)
        if t < 5:
            s.snapshot()
    s.drop_live()
    assert s.restore() == 4
    for t in range(5, 11):
        s.step(gs[t - 1], **HP, step=t, nthreads=4)
        s.snapshot()
    assert state_bytes(s) == state_bytes(ref)


# ---------------------------------------------------------------------------- generators


def test_generators_are_seeded_and_shaped():
    wl = W.CONFIGS["c1"]
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank)
    segs = [(tid, off, ln) for tid, _, off, ln in d["segments"]]
    g1 = W.gen_grads(wl, segs, d["n_padded"], 1, 0)
    assert torch.equal(g1, W.gen_grads(wl, segs, d["n_padded"], 1, 0))
    assert not torch.equal(g1, W.gen_grads(wl, segs, d["n_padded"], 2, 0))
    p = W.init_params(d["n"], d["n_padded"], 0)
    assert abs(float(p.std()) - 0.02) < 2e-4 and g1.dtype == torch.bfloat16
    sc = W.group_scales(wl, 0)
    assert all(0.5 <= x <= 2.0 for x in sc)
    tid, off, ln = max(segs, key=lambda s: s[2])
    assert abs(float(g1[off:off + ln].float().std()) / (1e-3 * sc[tid]) - 1) < 0.02
    ht = W.tiny_workload([400_000], 1, grad_kind="heavy_tail")
    gh = W.gen_grads(ht, [(0, 0, 400_000)], 400_000, 1, 0).float() / (1e-3 * W.group_scales(ht, 0)[0])
    frac_big = float((gh.abs() > 6).float().mean())      # N(0,1) never; 1% Student-t(3) sometimes
    assert 1e-5 < frac_big < 1e-3
