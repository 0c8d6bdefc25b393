"""Pins of the DP-global gradient-norm clip oracle (oracle/global_clip.py; SURVEY.md §8(e),
BASELINE.json:configs[2], reading R7b) against things other than itself: partition
invariance against the already pinned dp_size=1 shard-local clip, a hand-computable norm re-derived
with exact rationals, math.fsum, monotonicity, and a demonstration that the plausible mistake
("every rank clips by its own norm") fails the pins.  CPU only."""
import math
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import global_clip as GC
from oracle import oracle as O

HP = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)
f32 = np.float32


def bf16_bits_of(x):
    t = torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def widen(bits):
    return (bits.astype(np.uint32) << 16).view(np.float32)


def cut(flat, shard):
    """Rank-local slice of a flat (unpadded) array, zero-padded to n_padded."""
    out = np.zeros(shard.n_padded, flat.dtype)
    out[:shard.n] = flat[shard.shard_begin:shard.shard_begin + shard.n]
    return out


def flat_problem(numels, seed, heavy=True):
    rng = np.random.default_rng(seed)
    total = sum(numels)
    p = rng.normal(0, 0.02, total).astype(f32)
    gs = []
    for t in range(3):
        z = rng.standard_t(3, total) if heavy else rng.normal(0, 1, total)
        # uneven norms across the flat space, so that the ranks' local norms differ a lot
        z *= np.linspace(0.2, 5.0, total)
        gs.append(bf16_bits_of(z * 1e-3))
    return p, gs


@pytest.mark.parametrize("D", [1, 2, 3, 4])
def test_partition_invariance_against_the_dp1_local_clip(D):
    """The global norm does not depend on how the flat space is cut: D shards under the global clip
    reproduce, bit for bit, the ONE-shard run whose clip is the (pinned) shard-local rule R7."""
    numels = [1000, 37, 2048, 5, 700]
    layout = [(n, i) for i, n in enumerate(numels)]
    max_norm = 0.05
    p0, gs = flat_problem(numels, 5)
    one = O.OracleShard(layout, 1, 0, max_grad_norm=max_norm)
    one.set_state(cut(p0, one))
    grp = GC.OracleDPGroup(layout, D, max_norm)
    for s in grp.shards:
        s.set_state(cut(p0, s))
    for t, g in enumerate(gs, start=1):
        one.step(cut(g, one), **HP, step=t)
        coef = grp.step([cut(g, s) for s in grp.shards], **HP, step=t)
        assert coef.view(np.uint32) == one.last_coef.view(np.uint32)
        assert float(coef) < 1.0          # the clip is active, otherwise this pins nothing
        for s in grp.shards:
            lo, n = s.shard_begin, s.n
            for a, b in ((s.p, one.p), (s.m, one.m), (s.v, one.v), (s.p16, one.p16)):
                assert np.array_equal(a[:n], b[lo:lo + n]), (D, t)
            # pad lanes stay exactly zero
            assert not s.p[n:].any() and not s.m[n:].any() and not s.v[n:].any()


def test_hand_computable_global_norm_and_exact_rational_coefficient():
    # rank 0: 16 x 2^-3 -> S0 = 16 * 2^-6 = 1/4 ; rank 1: 12 x 2^-2 -> S1 = 12 * 2^-4 = 3/4 ; S = 1
    g0 = bf16_bits_of(np.full(16, 2.0 ** -3))
    g1 = bf16_bits_of(np.concatenate([np.full(12, 2.0 ** -2), np.zeros(4)]))
    assert GC.global_sumsq([g0, g1]) == 1.0
    max_norm = f32(0.5)
    want = Fraction(float(max_norm)) / (Fraction(1) + Fraction(1e-6))   # double 1e-6, as the C literal
    got = GC.global_clip_coef([g0, g1], float(max_norm))
    # fp32(double(x)) — the double division is within half an ulp(double) of the rational, far from an fp32 tie
    assert got == f32(float(want))
    assert abs(float(got) - 0.4999995) < 1e-7
    # the local rule would have given different numbers on each rank: 0.5/(0.5+1e-6) -> 1 (clamped), 0.5/(0.866+1e-6)
    assert O.clip_coef(O.sumsq(g0), 0.5) == f32(float(Fraction(0.5) / (Fraction(0.5) + Fraction(1e-6))))
    assert float(O.clip_coef(O.sumsq(g1), 0.5)) == pytest.approx(0.5 / math.sqrt(0.75), rel=1e-5)


def test_global_sumsq_is_the_exactly_rounded_sum_over_all_ranks():
    rng = np.random.default_rng(21)
    for D, n, scale in ((2, 1000, 1e-3), (5, 70_001, 1e-3), (8, 40_000, 1.0)):
        gs = [bf16_bits_of(rng.standard_t(3, n) * scale * (r + 1)) for r in range(D)]
        exact = math.fsum(float(x) * float(x) for g in gs for x in widen(g).astype(np.float64))
        got = GC.global_sumsq(gs)
        assert abs(got - exact) <= np.spacing(exact), (D, n)
        # fp32 gradients go through the same definition
        gf = [widen(g) * f32(1.0009765625) for g in gs]
        exact = math.fsum(float(x) * float(x) for g in gf for x in g.astype(np.float64))
        assert abs(GC.global_sumsq(gf) - exact) <= np.spacing(exact)


def test_global_coefficient_never_exceeds_a_local_one_and_d1_is_the_local_rule():
    rng = np.random.default_rng(22)
    gs = [bf16_bits_of(rng.normal(0, 1e-3 * (r + 1), 5000)) for r in range(4)]
    cg = GC.global_clip_coef(gs, 0.01)
    for g in gs:
        assert float(cg) <= float(O.clip_coef(O.sumsq(g), 0.01))
    assert GC.global_clip_coef(gs[:1], 0.01) == O.clip_coef(O.sumsq(gs[0]), 0.01)
    # a rank whose gradients are all zero changes nothing
    z = np.zeros(5000, np.uint16)
    assert GC.global_clip_coef(gs + [z], 0.01) == cg
    # rank order does not matter to the value beyond the last rounding of the sum
    a, b = GC.global_sumsq(gs), GC.global_sumsq(gs[::-1])
    assert abs(a - b) <= np.spacing(a)
    # no clip when the global norm is below the threshold
    assert GC.global_clip_coef(gs, 10.0) == f32(1.0)


def test_the_per_rank_local_norm_mistake_is_caught():
    """A group that lets every rank clip by its OWN norm (the plausible wrong implementation) does not
    reproduce the one-shard trajectory — the invariance pin above would fail for it."""
    numels = [3000, 1000]
    layout = [(n, i) for i, n in enumerate(numels)]
    p0, gs = flat_problem(numels, 6)
    one = O.OracleShard(layout, 1, 0, max_grad_norm=0.05)
    one.set_state(cut(p0, one))
    wrong = [O.OracleShard(layout, 2, r, max_grad_norm=0.05) for r in range(2)]
    for s in wrong:
        s.set_state(cut(p0, s))
    one.step(cut(gs[0], one), **HP, step=1)
    differs = False
    for s in wrong:
        s.step(cut(gs[0], s), **HP, step=1)          # local rule
        differs |= not np.array_equal(s.m[:s.n], one.m[s.shard_begin:s.shard_begin + s.n])
    assert differs
