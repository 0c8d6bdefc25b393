"""Pins of the oracle's arithmetic (a1, a3) against things OTHER than itself:
closed forms, exact rationals, degenerate cases, symmetries, a bound, a library routine
(torch.optim.AdamW on CPU), a float64 shadow, torch's bf16 cast, hand-computable norms,
and the SURVEY Appendix A fixture.  CPU only.  (SURVEY.md §8(c) "What pins each part".)
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import oracle as O
from oracle import twin as T

HP = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)
f32 = np.float32
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "appendix_a_pins.txt")


def bits(x):
    return np.asarray(x, dtype=np.float32).view(np.uint32)


def bf16_bits_of(x):
    """bf16 bits of float values using torch's cast (library routine, RNE)."""
    t = torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def rand_state(n, seed, gstd=1e-3):
    rng = np.random.default_rng(seed)
    p = rng.normal(0, 0.02, n).astype(np.float32)
    g = bf16_bits_of(rng.normal(0, gstd, n))
    return p, g, rng


def run_steps(p0, grads, hp=HP, coef=1.0, nthreads=1, m0=None, v0=None):
    n = p0.shape[0]
    p = p0.copy()
    m = np.zeros(n, f32) if m0 is None else m0.copy()
    v = np.zeros(n, f32) if v0 is None else v0.copy()
    p16 = np.zeros(n, np.uint16)
    for t, g in enumerate(grads, start=1):
        O.adamw_step(p, m, v, g, p16, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"],
                     t, coef, nthreads)
    return p, m, v, p16


def metric_ii(a, b):
    """max |a-b| / (|b| + rms(b))  (reading R22)."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    return float(np.max(np.abs(a - b) / (np.abs(b) + math.sqrt(np.mean(b * b)))))


def nearest_f32(fr: Fraction) -> np.float32:
    """Correctly rounded binary32 of a rational (brute force around the double rounding)."""
    c = np.float32(float(fr))
    cands = [c, np.nextafter(c, f32(np.inf)), np.nextafter(c, f32(-np.inf))]
    return min(cands, key=lambda x: abs(Fraction(float(x)) - fr))


# ---------------------------------------------------------------------------- scalars


def test_scalars_are_correctly_rounded_exact_rationals():
    F = lambda x: Fraction(float(f32(x)))
    lr, b1, b2, wd = F(HP["lr"]), F(HP["beta1"]), F(HP["beta2"]), F(HP["wd"])
    for t in (1, 2, 3, 10, 100, 1000):
        sc = O.scalars(**HP, step=t)
        assert sc[0] == nearest_f32(1 - lr * wd)
        assert sc[1] == nearest_f32(1 - b1)
        assert sc[2] == nearest_f32(1 - b2)
        # beta^t in double is not exact; allow 1 ulp of fp32 around the exact rational
        ss_exact = lr / (1 - b1 ** t)
        assert abs(Fraction(float(sc[3])) - ss_exact) <= Fraction(float(np.spacing(sc[3])))
        s2 = float(sc[4]) ** 2
        assert abs(s2 - float(1 - b2 ** t)) <= 4e-7 * s2


def test_scalars_twin_and_c_agree_bitwise():
    for t in list(range(1, 40)) + [100, 1000, 12345, 10 ** 6]:
        assert np.array_equal(bits(O.scalars(**HP, step=t)),
                              bits(np.array(T.scalars_f32(**HP, t=t), dtype=np.float32)))


def _golden():
    sc, tr = [], []
    for line in open(GOLDEN):
        w = line.split()
        if not w or w[0].startswith("#"):
            continue
        if w[0] == "scalar":
            sc.append((w[1], int(w[2]), int(w[3], 16)))
        elif w[0] == "traj":
            tr.append((w[1], int(w[2]), int(w[3], 16), int(w[4], 16), int(w[5], 16),
                       int(w[6], 16), float(w[7])))
    return sc, tr


def test_golden_scalars():
    idx = dict(decay=0, omb1=1, omb2=2, ss=3, sbc2=4)
    sc, _ = _golden()
    assert len(sc) == 9
    for name, t, b in sc:
        assert int(bits(O.scalars(**HP, step=t))[idx[name]]) == b, (name, t)


def test_golden_trajectories():
    _, tr = _golden()
    e = lambda k: bf16_bits_of([2.0 ** k])[0]
    neg = lambda h: np.uint16(h | 0x8000)
    cases = {
        "A": (f32(2.0 ** -6), [e(-10)] * 3),
        "B": (f32(2.0 ** -6), [e(-10), neg(e(-10)), e(-10)]),
        "C": (f32(-(2.0 ** -5)), [e(-9), np.uint16(0), np.uint16(0)]),
    }
    assert len(tr) == 8
    for case, t, pb, mb, vb, hb, p64 in tr:
        p0, gs = cases[case]
        p, m, v, p16 = run_steps(np.array([p0], f32), [np.array([g], np.uint16) for g in gs[:t]])
        assert int(bits(p)[0]) == pb, (case, t, hex(int(bits(p)[0])))
        assert int(bits(m)[0]) == mb and int(bits(v)[0]) == vb, (case, t)
        assert int(p16[0]) == hb
        assert abs(float(p[0]) - p64) <= 2e-7 * abs(p64)


def test_hand_check_case_A_step1():
    # p1 = 2^-6 (1 - 3e-5) - 3e-4 * 2^-10/(2^-10 + 1e-8), by hand = 0.015324534322
    p, m, v, _ = run_steps(np.array([2.0 ** -6], f32), [bf16_bits_of([2.0 ** -10])])
    assert abs(float(p[0]) - 0.015324534322) < 2e-9
    # fp32(0.9), fp32(0.95) differ from the decimals by ~2.4e-7 relative
    assert abs(float(m[0]) - 0.1 * 2.0 ** -10) < 1e-6 * 0.1 * 2.0 ** -10
    assert abs(float(v[0]) - 0.05 * 2.0 ** -20) < 1e-6 * 0.05 * 2.0 ** -20


# ---------------------------------------------------------------------------- closed forms


def test_first_step_closed_form_exact_rationals():
    p0, g, _ = rand_state(4096, 1)
    g[g == 0] = bf16_bits_of([1e-3])[0]
    g[(g & 0x7FFF) == 0] = bf16_bits_of([1e-3])[0]
    p, m, v, _ = run_steps(p0, [g])
    gw = T.widen(g)
    for i in range(0, 4096, 37):
        pe, me, ve = T.adamw_first_step_exact(Fraction(float(p0[i])), Fraction(float(gw[i])), **HP)
        # fp32 chain: a handful of roundings, each <= 2^-24 relative
        assert abs(Fraction(float(m[i])) - me) <= abs(me) * Fraction(3, 2 ** 24)
        assert abs(Fraction(float(v[i])) - ve) <= abs(ve) * Fraction(3, 2 ** 24)
        tol = Fraction(float(np.spacing(np.abs(p[i])))) * Fraction(3, 2) + Fraction(3e-4) * Fraction(8, 2 ** 24)
        assert abs(Fraction(float(p[i])) - pe) <= tol
        # ~ p0 (1 - lr wd) - lr sign(g)
        assert abs(float(p[i]) - (float(p0[i]) * (1 - 3e-5) - 3e-4 * np.sign(gw[i]))) < 1e-7


def test_constant_gradient_trajectory_closed_form():
    # m_hat_t = g, v_hat_t = g^2 for all t  =>  every step moves by lr*g/(|g|+eps); wd = 0
    hp = dict(HP, wd=0.0)
    p0, g, _ = rand_state(2048, 2)
    g[(g & 0x7FFF) == 0] = bf16_bits_of([1e-3])[0]
    gw = T.widen(g).astype(np.float64)
    lr, eps = float(f32(hp["lr"])), float(f32(hp["eps"]))
    p = p0.copy()
    m = np.zeros_like(p)
    v = np.zeros_like(p)
    p16 = np.zeros(p.shape[0], np.uint16)
    for t in range(1, 21):
        O.adamw_step(p, m, v, g, p16, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"], t, 1.0, 1)
        expect = p0.astype(np.float64) - t * lr * gw / (np.abs(gw) + eps)
        assert np.max(np.abs(p - expect)) <= t * 4e-9 + 2e-9, t
        # bias-corrected moments equal g and g^2
        b1, b2 = float(f32(hp["beta1"])), float(f32(hp["beta2"]))
        np.testing.assert_allclose(m / (1 - b1 ** t), gw, rtol=2e-6)
        np.testing.assert_allclose(v / (1 - b2 ** t), gw * gw, rtol=2e-6)


def test_zero_grads_from_zero_moments_is_pure_decay():
    p0, _, _ = rand_state(1024, 3)
    z = np.zeros(1024, np.uint16)
    F = lambda x: Fraction(float(f32(x)))
    decay = nearest_f32(1 - F(HP["lr"]) * F(HP["wd"]))
    p = p0.copy()
    m = np.zeros_like(p)
    v = np.zeros_like(p)
    p16 = np.zeros(1024, np.uint16)
    expect = p0.copy()
    for t in range(1, 11):
        O.adamw_step(p, m, v, z, p16, **{k: HP[k] for k in ("lr", "beta1", "beta2", "eps", "wd")},
                     step=t, coef=1.0, nthreads=1)
        expect = expect * decay  # one fp32 rounding per step
        assert np.array_equal(bits(p), bits(expect))
        assert not m.any() and not v.any()


def test_zero_grads_after_warmup_decay_moments_geometrically():
    p0, g, _ = rand_state(512, 4)
    p, m, v, _ = run_steps(p0, [g])
    m1, v1 = m.copy(), v.copy()
    p16 = np.zeros(512, np.uint16)
    z = np.zeros(512, np.uint16)
    for t in range(2, 8):
        O.adamw_step(p, m, v, z, p16, 3e-4, 0.9, 0.95, 1e-8, 0.1, t, 1.0, 1)
        np.testing.assert_allclose(m, m1.astype(np.float64) * float(f32(0.9)) ** (t - 1), rtol=1e-6)
        np.testing.assert_allclose(v, v1.astype(np.float64) * float(f32(0.95)) ** (t - 1), rtol=1e-6)


def test_lr_zero_leaves_params_bitwise_and_moments_advance():
    hp = dict(HP, lr=0.0)
    p0, g, _ = rand_state(512, 5)
    p, m, v, p16 = run_steps(p0, [g, g], hp)
    assert np.array_equal(bits(p), bits(p0))
    assert m.any() and v.any()
    assert np.array_equal(p16, bf16_bits_of(p0))


def test_wd_zero_gives_unit_decay():
    assert O.scalars(3e-4, 0.9, 0.95, 1e-8, 0.0, 1)[0] == f32(1.0)


def test_sign_symmetry_bitwise():
    p0, g, rng = rand_state(4096, 6)
    gs = [bf16_bits_of(rng.normal(0, 1e-3, 4096)) for _ in range(5)]
    p, m, v, p16 = run_steps(p0, gs)
    pn, mn, vn, p16n = run_steps(-p0, [x ^ np.uint16(0x8000) for x in gs])
    assert np.array_equal(bits(pn), bits(-p))
    assert np.array_equal(bits(mn), bits(-m))
    assert np.array_equal(bits(vn), bits(v))
    assert np.array_equal(p16n, p16 ^ np.uint16(0x8000))


def test_update_magnitude_bound():
    # |p' - p*decay| <= 1.165*lr for betas (0.9, 0.95), all t; equals ~lr at t = 1
    p0, _, rng = rand_state(4096, 7)
    decay = O.scalars(**HP, step=1)[0]
    p = p0.copy()
    m = np.zeros_like(p)
    v = np.zeros_like(p)
    p16 = np.zeros(4096, np.uint16)
    for t in range(1, 31):
        g = bf16_bits_of(rng.standard_t(3, 4096) * 1e-3 * rng.choice([1e-3, 1, 30], 4096))
        before = p.copy()
        O.adamw_step(p, m, v, g, p16, 3e-4, 0.9, 0.95, 1e-8, 0.1, t, 1.0, 1)
        upd = np.abs(p.astype(np.float64) - before.astype(np.float64) * float(decay))
        assert upd.max() <= 1.165 * 3e-4 * (1 + 1e-5) + 1.2e-8, (t, upd.max())
        if t == 1:
            ga = np.abs(T.widen(g).astype(np.float64))
            want = float(f32(3e-4)) * ga / (ga + float(f32(1e-8)))  # = lr when |g| >> eps
            assert np.all(np.abs(upd - want) < 3e-4 * 1e-6 + 1.2e-8)  # two fp32 roundings of |p| <= 0.1


# ---------------------------------------------------------------------------- library / shadow


def _c1_like(n=200_000, steps=10, seed=8):
    rng = np.random.default_rng(seed)
    p0 = rng.normal(0, 0.02, n).astype(np.float32)
    gs = [bf16_bits_of(rng.normal(0, 1e-3, n) * rng.uniform(0.5, 2)) for _ in range(steps)]
    return p0, gs


def test_against_torch_adamw_cpu():
    p0, gs = _c1_like()
    tp = torch.nn.Parameter(torch.from_numpy(p0.copy()))
    opt = torch.optim.AdamW([tp], lr=3e-4, betas=(0.9, 0.95), eps=1e-8, weight_decay=0.1,
                            foreach=False, fused=False)
    n = p0.shape[0]
    p, m, v, p16 = p0.copy(), np.zeros(n, f32), np.zeros(n, f32), np.zeros(n, np.uint16)
    for t, g in enumerate(gs, start=1):
        tp.grad = torch.from_numpy(T.widen(g).copy())
        opt.step()
        O.adamw_step(p, m, v, g, p16, 3e-4, 0.9, 0.95, 1e-8, 0.1, t, 1.0, 1)
        st = opt.state[tp]
        assert metric_ii(p, tp.detach().numpy()) < 1e-6, t
        assert metric_ii(m, st["exp_avg"].numpy()) < 1e-6, t
        assert metric_ii(v, st["exp_avg_sq"].numpy()) < 2e-6, t
    assert metric_ii(p, tp.detach().numpy()) < 1e-6  # measured ~2e-7 after 10 steps


def test_against_float64_shadow():
    p0, gs = _c1_like(seed=9)
    n = p0.shape[0]
    p, m, v, p16 = p0.copy(), np.zeros(n, f32), np.zeros(n, f32), np.zeros(n, np.uint16)
    P, M, V = p0.astype(np.float64), np.zeros(n), np.zeros(n)
    for t, g in enumerate(gs, start=1):
        O.adamw_step(p, m, v, g, p16, 3e-4, 0.9, 0.95, 1e-8, 0.1, t, 1.0, 1)
        P, M, V = T.adamw_step_f64(P, M, V, T.widen(g).astype(np.float64), **HP, t=t)
        lim = 1e-6 if t == 1 else 1e-5
        assert metric_ii(p, P) < lim and metric_ii(m, M) < lim and metric_ii(v, V) < lim
    assert metric_ii(p, P) < 2e-6  # measured ~6e-7 after 10 steps


def test_numpy_twin_agrees_bitwise_incl_clip_and_extremes():
    rng = np.random.default_rng(10)
    n = 50_000
    p = rng.normal(0, 0.02, n).astype(np.float32)
    p[:100] = 0
    m = np.zeros(n, f32)
    v = np.zeros(n, f32)
    p16 = np.zeros(n, np.uint16)
    for t in range(1, 13):
        scale = rng.choice([1e-30, 1e-12, 1e-3, 1.0, 1e4], n)  # denormal squares .. huge
        g = bf16_bits_of(rng.standard_t(3, n) * scale)
        g[::97] = 0
        coef = float(f32(rng.uniform(0.01, 1.0))) if t % 2 else 1.0
        pe, me, ve, he = T.adamw_step_numpy(p, m, v, g, **HP, t=t, coef=coef)
        O.adamw_step(p, m, v, g, p16, 3e-4, 0.9, 0.95, 1e-8, 0.1, t, coef, 1)
        assert np.array_equal(bits(p), bits(pe)), t
        assert np.array_equal(bits(m), bits(me)), t
        assert np.array_equal(bits(v), bits(ve)), t
        assert np.array_equal(p16, he), t


def test_thread_count_does_not_change_bits():
    p0, gs = _c1_like(n=100_003, steps=3, seed=11)
    a = run_steps(p0, gs, nthreads=1)
    b = run_steps(p0, gs, nthreads=5)
    for x, y in zip(a, b):
        assert np.array_equal(x.view(np.uint8), y.view(np.uint8))


# ---------------------------------------------------------------------------- bf16 rounding


def test_rne_bf16_matches_torch_and_ties_to_even():
    rng = np.random.default_rng(12)
    x = np.concatenate([
        rng.normal(0, 0.02, 100_000), rng.normal(0, 1e-20, 1000), rng.normal(0, 1e20, 1000),
        [0.0, -0.0, 1.0, -1.0, 3.0e38, 1e-45]]).astype(np.float32)
    assert np.array_equal(O.rne_bf16(x), bf16_bits_of(x))
    assert np.array_equal(T.rne_bf16_numpy(x), bf16_bits_of(x))
    # ties: low 16 bits == 0x8000 with even and odd upper halves, both signs
    hi = np.array([0x3C7A, 0x3C7B, 0xBD01, 0xBD02, 0x0001, 0x0000, 0x7F7E], np.uint32)
    tie = ((hi << 16) | 0x8000).view(np.float32)
    got = O.rne_bf16(tie)
    want = np.where(hi & 1, hi + 1, hi).astype(np.uint16)
    assert np.array_equal(got, want)
    assert np.array_equal(got, bf16_bits_of(tie))
    # just below / above the tie
    below = ((hi << 16) | 0x7FFF).view(np.float32)
    above = ((hi << 16) | 0x8001).view(np.float32)
    assert np.array_equal(O.rne_bf16(below), hi.astype(np.uint16))
    assert np.array_equal(O.rne_bf16(above), (hi + 1).astype(np.uint16))


# ---------------------------------------------------------------------------- clip


def test_clip_hand_computable_norm():
    g = bf16_bits_of(np.array([3.0, 4.0, 0.0, 0.0]) * 2.0 ** -10)
    S = O.sumsq(g)
    assert S == 25.0 * 2.0 ** -20  # exact
    assert O.clip_coef(S, 1.0) == f32(1.0)  # norm 5*2^-10 < 1: clamp to 1
    want = f32(float(f32(1e-3)) / (5 * 2.0 ** -10 + 1e-6))  # max_norm arrives as a C float
    assert O.clip_coef(S, 1e-3) == want
    assert abs(float(want) - 0.20476) < 1e-4


def test_sumsq_matches_exactly_rounded_sum():
    rng = np.random.default_rng(13)
    for n, scale in ((1, 1.0), (1000, 1e-3), (300_000, 1e-3), (300_000, 1.0)):
        g = bf16_bits_of(rng.standard_t(3, n) * scale)
        a, b = O.sumsq(g), T.sumsq_exact(g)
        assert abs(a - b) <= np.spacing(b), (n, a, b)


def test_clip_is_active_at_c3_statistics():
    # norm ~ sqrt(n * 1e-6 * (0.99 + 0.01*3)) ~ 20.7 at n = 421M  =>  coef ~ 0.048
    n = 421_150_976
    coef = O.clip_coef(n * 1e-6 * (0.99 + 0.01 * 3), 1.0)
    assert 0.04 < float(coef) < 0.06


def test_clip_enters_the_step_as_a_gradient_scale():
    # with coef = 2^-k the scaled step equals the unscaled step on g * 2^-k (exact scaling)
    p0, g, _ = rand_state(1000, 14)
    a = run_steps(p0, [g], coef=0.25)
    g4 = bf16_bits_of(T.widen(g) * 0.25)
    b = run_steps(p0, [g4], coef=1.0)
    for x, y in zip(a, b):
        assert np.array_equal(x.view(np.uint8), y.view(np.uint8))
