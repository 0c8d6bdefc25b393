"""Pins of the full-rank-state oracle (oracle/rank_state.py) — the D2H payload
of PAPER.md:145 and the in-place recovery of PAPER.md:160/230.  CPU only.

What fixes it from outside the oracle: the model-parameter part against torch's bf16 cast of the
flat master space in rank order; the byte layout against offsets computed here by hand; the
optimizer part against the optimizer-only snapshot (oracle.py, itself pinned); restore against the
state before the fault with every other rank's memory poisoned; FNV-1a of the header against a
hash computed here."""
import struct

import numpy as np
import pytest

from oracle import oracle as O
from oracle import rank_state as RS
from oracle import ring as R

HP = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)


def _group(D=3, numels=(1000, 333, 77), chunk=1024, seed=0, precision="bf16", user=b""):
    layout = [(n, i) for i, n in enumerate(numels)]
    rng = np.random.default_rng(seed)
    ranks = []
    for r in range(D):
        o = O.OracleShard(layout, D, r, chunk_bytes=chunk, precision=precision, user=user)
        p0 = np.zeros(o.n_padded, np.float32)
        p0[:o.n] = rng.normal(0, 0.02, o.n)
        o.set_state(p0)
        ranks.append(RS.FullRankState(o))
    return ranks, rng


def _grads(ranks, rng, fp32=False):
    out = []
    for fr in ranks:
        g = np.zeros(fr.o.n_padded, np.float32)
        g[:fr.o.n] = rng.normal(0, 1e-3, fr.o.n)
        out.append(g if fp32 else (g.view(np.uint32) >> 16).astype(np.uint16))
    return out


def _iteration(ranks, gs, t, snapshot=True):
    """step on every rank, all-gather (R29), full-rank-state flush (R31/R32)."""
    for fr, g in zip(ranks, gs):
        fr.o.step(g, **HP, step=t)
    W = R.publish([fr.o for fr in ranks])
    for fr in ranks:
        fr.W[:] = W
        if snapshot:
            fr.snapshot()


def _bits(a):
    return a.view(np.uint8)


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
def test_layout_by_hand_and_parameter_part_against_the_library_cast(precision):
    import torch
    D = 3
    ranks, rng = _group(D, precision=precision, user=b"rng-state")
    for t in (1, 2):
        _iteration(ranks, _grads(ranks, rng, precision == "fp32"), t)
    N = ranks[0].o.n_padded
    eb = 4 if precision == "fp32" else 2
    flat = np.concatenate([fr.o.p for fr in ranks])                 # the flat padded master space of a0
    if precision == "bf16":
        want_w = torch.from_numpy(flat).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    else:
        want_w = flat
    for fr in ranks:
        buf = fr.packed()
        assert buf.size == 256 + 12 * N + D * N * eb == fr.snapshot_bytes
        assert np.array_equal(buf[256:256 + 4 * N], _bits(fr.o.p))
        assert np.array_equal(buf[256 + 4 * N:256 + 8 * N], _bits(fr.o.m))
        assert np.array_equal(buf[256 + 8 * N:256 + 12 * N], _bits(fr.o.v))
        assert np.array_equal(buf[256 + 12 * N:], _bits(want_w))   # W = rank-order all-gather of the cast
        # the rank's own range of W is its own model-param copy
        own = buf[256 + 12 * N + fr.r * N * eb:256 + 12 * N + (fr.r + 1) * N * eb]
        assert np.array_equal(own, _bits(want_w[fr.r * N:(fr.r + 1) * N]))
        # committed local slot == the packed buffer
        assert np.array_equal(fr.slots[2 % 2], buf)


def test_optimizer_part_and_header_against_the_optimizer_only_snapshot():
    ranks, rng = _group(2, user=b"\x01\x02\x03")
    _iteration(ranks, _grads(ranks, rng), 1)
    fr = ranks[1]
    full, opt = fr.packed(), fr.o.packed_snapshot()
    N = fr.o.n_padded
    assert np.array_equal(full[256:256 + 12 * N], opt[256:])        # same bytes at the same offsets
    hf, ho = full[:256].tobytes(), opt[:256].tobytes()
    # payload word: byte offset 8+4+4+7*8+6*4+8+4 = 108 (little-endian u32), hand-counted from R10
    assert struct.unpack_from("<I", ho, 108)[0] == 0
    assert struct.unpack_from("<I", hf, 108)[0] == 1 | (2 << 8)
    assert hf[:108] == ho[:108] and hf[112:240] == ho[112:240]      # nothing else differs before the hash
    h = 0xCBF29CE484222325
    for b in hf[:240]:
        h = ((h ^ b) * 0x100000001B3) & ((1 << 64) - 1)
    assert struct.unpack_from("<Q", hf, 240)[0] == h                # FNV-1a 64 recomputed here
    assert struct.unpack_from("<Q", hf, 248)[0] == 1                # seq_end == step: committed
    # an optimizer-only reader still parses it and sees the payload word
    assert O.parse_header(hf)["payload"] == RS.payload_word(2) and O.parse_header(ho)["payload"] == 0


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
def test_in_place_recovery_reads_nothing_from_other_ranks_and_resumes_bit_exactly(precision):
    D, fp32 = 3, precision == "fp32"
    ranks, rng = _group(D, seed=7, precision=precision, user=b"rng")
    ref, _ = _group(D, seed=7, precision=precision, user=b"rng")
    gs_all = [_grads(ranks, rng, fp32) for _ in range(6)]
    for t in range(1, 7):
        _iteration(ref, gs_all[t - 1], t, snapshot=False)
    for t in range(1, 5):
        _iteration(ranks, gs_all[t - 1], t)
    victim = ranks[1]
    before = [x.copy() for x in (victim.o.p, victim.o.m, victim.o.v, victim.o.p16, victim.W)]
    # step 5 is in flight on the victim when the transient fault hits: partial work is discarded (I4)
    victim.o.step(gs_all[4][1], **HP, step=5)
    victim.drop_live()
    for fr in ranks:                                                # poison everything that is not the victim's host
        if fr is not victim:
            for s in fr.slots:
                s[:] = 0xEE
    assert victim.restore_in_place() == 4
    after = (victim.o.p, victim.o.m, victim.o.v, victim.o.p16, victim.W)
    for a, b in zip(after, before):
        assert np.array_equal(_bits(a), _bits(b))
    assert victim.o.restored_user == b"rng"
    own = victim.o.p if fp32 else O.rne_bf16(victim.o.p)
    assert np.array_equal(_bits(victim.own_range()), _bits(own))    # R33: own range of W == the model-param copy
    for t in (5, 6):
        _iteration(ranks, gs_all[t - 1], t, snapshot=False)
    for a, b in zip(ranks, ref):
        for x, y in ((a.o.p, b.o.p), (a.o.m, b.o.m), (a.o.v, b.o.v), (a.o.p16, b.o.p16), (a.W, b.W)):
            assert np.array_equal(_bits(x), _bits(y))


def test_torn_flush_in_either_region_is_never_chosen():
    ranks, rng = _group(2, numels=(3000,), chunk=2048)
    fr = ranks[0]
    N = fr.o.n_padded
    n_w = -(-2 * N * 2 // 2048)                                     # chunks of the W region (D * N * 2 bytes)
    n_o = -(-12 * N // 2048)
    _iteration(ranks, _grads(ranks, rng), 1)
    for stop in (0, 1, n_w, n_w + 1, n_w + n_o - 1, n_w + n_o):     # torn in W, at the boundary, in p‖m‖v, before commit
        gs = _grads(ranks, rng)
        t = fr.o.last_step + 1
        for x, g in zip(ranks, gs):
            x.o.step(g, **HP, step=t)
        W = R.publish([x.o for x in ranks])
        for x in ranks:
            x.W[:] = W
        slot = fr.snapshot(abort_after_chunks=stop)
        assert O.parse_header(fr.slots[slot][:256].tobytes()) is None
        # R32 transfer order: the first `stop` chunks landed, W region first
        src = fr.packed()
        w0 = 256 + 12 * N
        landed_w = min(stop, n_w) * 2048
        assert np.array_equal(fr.slots[slot][w0:min(w0 + landed_w, fr.snapshot_bytes)],
                              src[w0:min(w0 + landed_w, fr.snapshot_bytes)])
        s, h = fr.newest_committed()
        assert s == 1 - slot and h["step"] == t - 1
        ranks[1].snapshot()
        fr.snapshot()                                               # the retry commits
        assert fr.newest_committed()[1]["step"] == t


def test_slot_of_another_identity_or_payload_kind_is_refused():
    ranks, rng = _group(2)
    _iteration(ranks, _grads(ranks, rng), 1)
    a, b = ranks
    a.slots[1][:] = b.slots[1]                                      # rank 1's state in rank 0's slot
    a.drop_live()
    with pytest.raises(O.OracleError):
        a.restore_in_place()
    # an optimizer-only snapshot (the H2H payload) in a full-rank-state slot is refused as well
    b.slots[1][:256 + 12 * b.o.n_padded] = b.o.packed_snapshot()
    with pytest.raises(O.OracleError):
        b.restore_in_place()
