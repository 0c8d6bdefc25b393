"""Pins of the oracle's §8(f2) routine — the paper's own precision (binary32 gradients, no bf16
copy: "BF16 and FP16 disabled") and per-tensor decay groups (reading R5b) —
against things other than itself: the already-pinned bf16 routine as a special case, exact
rationals, a library routine (torch.optim.AdamW with fp32 gradients and two parameter groups),
a float64 shadow, the numpy twin, the wd = 0 equivalence, math.fsum.  CPU only."""
import math
from fractions import Fraction

import numpy as np
import torch

from oracle import oracle as O
from oracle import twin as T

from test_oracle_pins import HP, bf16_bits_of, bits, metric_ii

f32 = np.float32
HPV = (HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], HP["wd"])


def fresh(n):
    return np.zeros(n, f32), np.zeros(n, f32), np.zeros(n, np.uint16)


def test_general_routine_reduces_to_the_pinned_bf16_routine():
    # special case: bf16 gradients, bf16 copy, no mask  ==  phx_oracle_adamw_step, bit for bit
    rng = np.random.default_rng(20)
    n = 30_011
    p0 = rng.normal(0, 0.02, n).astype(f32)
    pa, pb = p0.copy(), p0.copy()
    (ma, va, ha), (mb, vb, hb) = fresh(n), fresh(n)
    for t in range(1, 6):
        g = bf16_bits_of(rng.standard_t(3, n) * 1e-3)
        coef = 0.37 if t == 3 else 1.0
        O.adamw_step(pa, ma, va, g, ha, *HPV, t, coef, 1)
        O.adamw_step_ex(pb, mb, vb, g, hb, None, *HPV, t, coef, 3)
        for x, y in ((pa, pb), (ma, mb), (va, vb), (ha, hb)):
            assert np.array_equal(x.view(np.uint8), y.view(np.uint8)), t
    # an all-zero mask changes nothing either
    O.adamw_step(pa, ma, va, g, ha, *HPV, 6, 1.0, 1)
    O.adamw_step_ex(pb, mb, vb, g, hb, np.zeros(n, np.uint8), *HPV, 6, 1.0, 1)
    assert np.array_equal(bits(pa), bits(pb))


def test_fp32_gradients_equal_bf16_gradients_when_representable():
    # a binary32 gradient that happens to be a bf16 value must give the bf16 routine's bits
    rng = np.random.default_rng(21)
    n = 10_000
    p0 = rng.normal(0, 0.02, n).astype(f32)
    g16 = bf16_bits_of(rng.normal(0, 1e-3, n))
    pa, pb = p0.copy(), p0.copy()
    (ma, va, ha), (mb, vb, _) = fresh(n), fresh(n)
    O.adamw_step(pa, ma, va, g16, ha, *HPV, 1, 1.0, 1)
    O.adamw_step_ex(pb, mb, vb, T.widen(g16).copy(), None, None, *HPV, 1, 1.0, 1)
    assert np.array_equal(bits(pa), bits(pb)) and np.array_equal(bits(ma), bits(mb)) and np.array_equal(bits(va), bits(vb))


def test_fp32_first_step_closed_form_exact_rationals():
    # m1 = (1-b1) g, v1 = (1-b2) g^2, p1 = p0 (1 - lr wd) - lr g/(|g|+eps), exact, g a full 24-bit value
    rng = np.random.default_rng(22)
    n = 2048
    p0 = rng.normal(0, 0.02, n).astype(f32)
    g = (rng.normal(0, 1e-3, n) * rng.uniform(0.5, 2, n)).astype(f32)
    g[g == 0] = f32(1e-3)
    assert np.any(g.view(np.uint32) & 0xFFFF)          # not bf16-representable: the new code path
    p, (m, v, _) = p0.copy(), fresh(n)
    O.adamw_step_ex(p, m, v, g, None, None, *HPV, 1, 1.0, 1)
    for i in range(0, n, 29):
        pe, me, ve = T.adamw_first_step_exact(Fraction(float(p0[i])), Fraction(float(g[i])), **HP)
        assert abs(Fraction(float(m[i])) - me) <= abs(me) * Fraction(3, 2 ** 24)
        assert abs(Fraction(float(v[i])) - ve) <= abs(ve) * Fraction(4, 2 ** 24)   # g*g now rounds too
        tol = Fraction(float(np.spacing(np.abs(p[i])))) * Fraction(3, 2) + Fraction(3e-4) * Fraction(8, 2 ** 24)
        assert abs(Fraction(float(p[i])) - pe) <= tol


def test_fp32_against_torch_adamw_with_two_param_groups():
    # library special case: torch.optim.AdamW, fp32 gradients, a decayed group and a wd = 0 group
    rng = np.random.default_rng(23)
    na, nb = 60_000, 7_001
    n = na + nb
    p0 = rng.normal(0, 0.02, n).astype(f32)
    ta = torch.nn.Parameter(torch.from_numpy(p0[:na].copy()))
    tb = torch.nn.Parameter(torch.from_numpy(p0[na:].copy()))
    opt = torch.optim.AdamW([dict(params=[ta], weight_decay=0.1), dict(params=[tb], weight_decay=0.0)],
                            lr=3e-4, betas=(0.9, 0.95), eps=1e-8, foreach=False, fused=False)
    mask = np.zeros(n, np.uint8)
    mask[na:] = 1
    p, (m, v, _) = p0.copy(), fresh(n)
    for t in range(1, 11):
        g = (rng.normal(0, 1e-3, n) * rng.uniform(0.5, 2)).astype(f32)
        ta.grad = torch.from_numpy(g[:na].copy())
        tb.grad = torch.from_numpy(g[na:].copy())
        opt.step()
        O.adamw_step_ex(p, m, v, g, None, mask, *HPV, t, 1.0, 2)
        ref = np.concatenate([ta.detach().numpy(), tb.detach().numpy()])
        assert metric_ii(p, ref) < 1e-6, t
        assert metric_ii(p[na:], ref[na:]) < 1e-6, t       # the no-decay group on its own scale
        refm = np.concatenate([opt.state[ta]["exp_avg"].numpy(), opt.state[tb]["exp_avg"].numpy()])
        refv = np.concatenate([opt.state[ta]["exp_avg_sq"].numpy(), opt.state[tb]["exp_avg_sq"].numpy()])
        assert metric_ii(m, refm) < 1e-6 and metric_ii(v, refv) < 2e-6, t
    # the groups really differ: decaying the no-decay group would move it by ~10 * lr * wd relative
    wrong = p0.copy()
    (m2, v2, _) = fresh(n)
    rng = np.random.default_rng(23)
    rng.normal(0, 0.02, n)
    for t in range(1, 11):
        g = (rng.normal(0, 1e-3, n) * rng.uniform(0.5, 2)).astype(f32)
        O.adamw_step_ex(wrong, m2, v2, g, None, None, *HPV, t, 1.0, 1)
    big = np.abs(p0[na:]) > 0.02                            # where 10 steps of decay (3e-4 relative) show
    rel = np.abs(wrong[na:][big] - ref[na:][big]) / np.abs(ref[na:][big])
    assert rel.min() > 1e-4


def test_no_decay_elements_follow_the_wd_zero_trajectory_bitwise():
    # p * 1.0f is exact: a flagged element evolves exactly as under wd = 0, an unflagged one as under wd
    rng = np.random.default_rng(24)
    n = 5000
    p0 = rng.normal(0, 0.02, n).astype(f32)
    mask = (rng.random(n) < 0.3).astype(np.uint8)
    pg, (mg, vg, hg) = p0.copy(), fresh(n)
    pz, (mz, vz, hz) = p0.copy(), fresh(n)
    pw, (mw, vw, hw) = p0.copy(), fresh(n)
    for t in range(1, 8):
        g = bf16_bits_of(rng.normal(0, 1e-3, n))
        O.adamw_step_ex(pg, mg, vg, g, hg, mask, *HPV, t, 1.0, 1)
        O.adamw_step(pz, mz, vz, g, hz, HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], 0.0, t, 1.0, 1)
        O.adamw_step(pw, mw, vw, g, hw, *HPV, t, 1.0, 1)
    k = mask.astype(bool)
    assert np.array_equal(bits(pg)[k], bits(pz)[k]) and np.array_equal(hg[k], hz[k])
    assert np.array_equal(bits(pg)[~k], bits(pw)[~k]) and np.array_equal(hg[~k], hw[~k])
    assert not np.array_equal(bits(pg)[k], bits(pw)[k])
    assert np.array_equal(bits(mg), bits(mw)) and np.array_equal(bits(vg), bits(vw))   # moments never see wd


def test_fp32_against_float64_shadow_and_numpy_twin():
    rng = np.random.default_rng(25)
    n = 100_000
    p0 = rng.normal(0, 0.02, n).astype(f32)
    mask = np.zeros(n, np.uint8)
    mask[::7] = 1
    p, (m, v, _) = p0.copy(), fresh(n)
    P, M, V = p0.astype(np.float64), np.zeros(n), np.zeros(n)
    for t in range(1, 11):
        scale = rng.choice([1e-25, 1e-3, 1.0, 1e3], n) if t % 3 == 0 else 1e-3
        g = (rng.standard_t(3, n) * scale).astype(f32)
        g[::101] = 0
        coef = float(f32(0.61)) if t % 2 else 1.0
        pe, me, ve, he = T.adamw_step_numpy_ex(p, m, v, g, **HP, t=t, coef=coef, no_decay=mask, bf16_copy=False)
        assert he is None
        if t % 3:   # float64 shadow on the well-scaled steps (uniform decay for the shadow: compare unmasked lanes)
            Pn, Mn, Vn = T.adamw_step_f64(P, M, V, g.astype(np.float64) * coef, **HP, t=t)
        O.adamw_step_ex(p, m, v, g, None, mask, *HPV, t, coef, 2)
        assert np.array_equal(bits(p), bits(pe)) and np.array_equal(bits(m), bits(me)) and np.array_equal(bits(v), bits(ve)), t
        if t < 3:
            P, M, V = Pn, Mn, Vn
            k = mask == 0
            lim = 1e-6 if t == 1 else 1e-5
            assert metric_ii(p[k], P[k]) < lim and metric_ii(m, M) < lim and metric_ii(v, V) < lim


def test_sumsq_f32_matches_exactly_rounded_sum_and_hand_case():
    rng = np.random.default_rng(26)
    for n, scale in ((1, 1.0), (1000, 1e-3), (300_000, 1e-3), (300_000, 1.0)):
        g = (rng.standard_t(3, n) * scale).astype(f32)
        a, b = O.sumsq(g), T.sumsq_exact_f32(g)
        # 48-bit squares no longer fit the 64-bit running sum exactly: the sequential long-double sum
        # errs by ~sqrt(n) * 2^-64 relative (bound n * 2^-64), i.e. a few ulps of the double result,
        # 8 orders of magnitude below the fp32 clip coefficient's resolution
        assert abs(a - b) <= 4 * np.spacing(b), (n, a, b)
    g = (np.array([3.0, 4.0, 12.0, 0.0]) * 2.0 ** -12).astype(f32)
    assert O.sumsq(g) == 169.0 * 2.0 ** -24                       # norm 13 * 2^-12, exact
    want = f32(float(f32(1e-3)) / (13 * 2.0 ** -12 + 1e-6))
    assert O.clip_coef(O.sumsq(g), 1e-3) == want


def test_oracle_shard_fp32_precision_and_flags():
    # the stateful wrapper: mask from the segment table, no bf16 copy, snapshot/restore/resume unchanged
    layout = [(1000, 0), (77, 1), (3000, 2), (64, 3)]
    flags = [0, O.TENSOR_NO_DECAY, 0, O.TENSOR_NO_DECAY]
    rng = np.random.default_rng(27)
    shards = [O.OracleShard(layout, 2, r, flags=flags, precision="fp32", chunk_bytes=4096) for r in range(2)]
    flat_mask = np.concatenate([np.full(n, f & 1, np.uint8) for (n, _), f in zip(layout, flags)])
    total = flat_mask.size
    for r, o in enumerate(shards):
        lo = o.shard_begin
        want = np.zeros(o.n_padded, np.uint8)
        k = max(0, min(total - lo, o.n_padded))
        want[:k] = flat_mask[lo:lo + k]
        assert np.array_equal(o.no_decay, want)
        p0 = np.zeros(o.n_padded, f32)
        p0[:o.n] = rng.normal(0, 0.02, o.n)
        o.set_state(p0)
        ref = O.OracleShard(layout, 2, r, flags=flags, precision="fp32", chunk_bytes=4096)
        ref.set_state(p0)
        gs = []
        for t in range(1, 7):
            g = np.zeros(o.n_padded, f32)
            g[:o.n] = rng.normal(0, 1e-3, o.n)
            gs.append(g)
            ref.step(g, **HP, step=t)
        for t in range(1, 5):
            o.step(gs[t - 1], **HP, step=t)
            o.snapshot()
        assert not o.p16.any()
        o.step(gs[4], **HP, step=5)        # in flight, lost
        o.drop_live()
        assert o.restore() == 4
        for t in (5, 6):
            o.step(gs[t - 1], **HP, step=t)
        for a, b in ((o.p, ref.p), (o.m, ref.m), (o.v, ref.v)):
            assert np.array_equal(bits(a), bits(b))
        assert not o.p[o.n:].any() and not o.m[o.n:].any() and not o.v[o.n:].any()
    # flags enter the layout hash: a replica of a differently-grouped shard is foreign
    other = O.OracleShard(layout, 2, 0, flags=[0, 0, 0, 0], precision="fp32")
    assert other.layout_hash != shards[0].layout_hash
