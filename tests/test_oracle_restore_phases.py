"""Pins of the oracle's TWO-PHASE restore (reading R37; "execution resumes from the last
completed step"): phase 1 brings back the parameters (p, the bf16 copy, W for a full rank state), phase 2 the
moments.  Pinned against the already pinned one-phase restore (byte identity of the final state, incl. the choice
of slot under a torn flush), against torch's bf16 cast, and by sentinels that show WHAT each phase may touch.  CPU only.
"""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from oracle import rank_state as RS
from paper_2607_01646_b200 import workloads as W

from test_oracle_shard import HP, seeded, state_bytes


def run_to(wl, steps, torn_last=None, **kw):
    s, gs = seeded(wl, steps, **kw)
    for t in range(1, steps + 1):
        s.step(gs[t - 1], **HP, step=t)
        s.snapshot(abort_after_chunks=torn_last if t == steps else None)
    return s, gs


@pytest.mark.parametrize("torn_last", [None, 0, 1, 3])
def test_two_phases_equal_the_one_phase_restore(torn_last):
    wl = W.tiny_workload([3000, 77, 1], dp_size=2, dp_rank=1)
    a, gs = run_to(wl, 5, torn_last, chunk_bytes=4096)
    b, _ = run_to(wl, 5, torn_last, chunk_bytes=4096)
    for s in (a, b):
        s.drop_live()
    want = a.restore()
    assert want == (5 if torn_last is None else 4)
    assert b.restore_params_first() == want
    assert b.restore_finish() == want
    assert state_bytes(a) == state_bytes(b) and a.restored_user == b.restored_user
    # and the resumed trajectories stay equal
    for t in range(want + 1, 6):
        a.step(gs[t - 1], **HP, step=t)
        b.step(gs[t - 1], **HP, step=t)
    assert state_bytes(a) == state_bytes(b)


def test_phase_one_touches_the_parameters_only_and_blocks_the_optimizer_step():
    wl = W.tiny_workload([1000, 24, 7], dp_size=1)
    s, gs = run_to(wl, 3, chunk_bytes=1024)
    slot = s.replica[3 % 2]
    N4 = 4 * s.n_padded
    s.p[:] = 7.0
    s.p16[:] = 0x1234
    s.m[:] = -3.0      # sentinels: phase 1 must not touch the moments
    s.v[:] = 5.0
    assert s.restore_params_first() == 3
    assert s.p.tobytes() == slot[O.HEADER_BYTES:O.HEADER_BYTES + N4].tobytes()
    want16 = torch.from_numpy(s.p.copy()).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(s.p16, want16)
    assert np.all(s.m == -3.0) and np.all(s.v == 5.0)
    with pytest.raises(O.OracleError):
        s.step(gs[0], **HP, step=4)                      # the moments are not back yet
    assert s.restore_finish() == 3
    assert s.m.tobytes() == slot[O.HEADER_BYTES + N4:O.HEADER_BYTES + 2 * N4].tobytes()
    assert s.v.tobytes() == slot[O.HEADER_BYTES + 2 * N4:].tobytes()


def test_no_committed_snapshot_and_wrong_identity():
    wl = W.tiny_workload([500], dp_size=2, dp_rank=0)
    s, _ = seeded(wl, 1)
    with pytest.raises(O.OracleError):
        s.restore_params_first()
    a, _ = run_to(wl, 2)
    other = O.OracleShard(wl.layout(), 2, 1)             # another dp_rank reads rank 0's replica
    other.replica = a.replica
    with pytest.raises(O.OracleError):
        other.restore_params_first()


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("torn", [None, 0, 2])
def test_full_rank_state_two_phases(precision, torn):
    D = 2
    wl = W.tiny_workload([2000, 65], dp_size=D, dp_rank=1, precision=precision)

    def build():
        o = O.OracleShard(wl.layout(), D, 1, chunk_bytes=2048, precision=precision)
        o.set_state(W.init_params(o.n, o.n_padded, 3).numpy())
        return RS.FullRankState(o)
    a, b = build(), build()
    segs = [(tid, off, ln) for tid, _, off, ln in a.o.segments]
    rng = np.random.default_rng(0)
    for t in (1, 2, 3):
        g = W.gen_grads(wl, segs, a.o.n_padded, t, 0, dtype=torch.float32 if precision == "fp32" else torch.bfloat16)
        gb = g.numpy().copy() if precision == "fp32" else g.view(torch.int16).numpy().view(np.uint16).copy()
        other = rng.integers(0, 60000, a.o.n_padded).astype(a.wdtype)      # the other rank's published range
        for f in (a, b):
            f.o.step(gb, **HP, step=t)
            f.write_own_range()
            f.W[:f.o.n_padded] = other
            f.snapshot(abort_after_chunks=torn if t == 3 else None)
    for f in (a, b):
        f.drop_live()
    want = a.restore_in_place()
    assert want == (3 if torn is None else 2)
    b.o.m[:] = 9.0
    b.o.p[:] = -7.0
    assert b.restore_in_place_params_first() == want
    # for a full rank state the parameters ARE W: phase 1 brings back W alone (the own range of it = the model-param
    # copy, which must equal torch's bf16 cast of the p that arrives in phase 2)
    assert np.array_equal(b.W, a.W) and np.array_equal(b.o.p16, a.o.p16)
    assert np.all(b.o.m == 9.0) and np.all(b.o.p == -7.0)          # phase 1 left p and the moments alone
    assert b.restore_in_place_finish() == want
    assert state_bytes(a.o) == state_bytes(b.o) and np.array_equal(a.W, b.W)
    if precision == "bf16":
        cast = torch.from_numpy(b.o.p.copy()).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
        assert np.array_equal(b.own_range(), cast)       # R31: the own range of the restored W == RNE_bf16(restored p)
    else:
        assert np.array_equal(b.own_range(), b.o.p)
