"""Pins of oracle/grad_finalize.py (second half; reading R34) against
things other than itself: torch's fp32 multiply + bf16 cast (library routine), math.fsum (the exactly
rounded sum), exact-rational double rounding, enumerated ties, a hand-computable case, and the already
pinned a1 oracle on the produced bits.  CPU only."""
import math
from fractions import Fraction

import numpy as np
import torch

from oracle import grad_finalize as GF
from oracle import oracle as O


def widen(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32)


def torch_bits(g32: np.ndarray, scale: float) -> np.ndarray:
    t = torch.from_numpy(g32.copy()) * torch.tensor(scale, dtype=torch.float32)
    return t.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def rne_fraction_to_grid(x: Fraction, mant_bits: int) -> Fraction:
    """Round an exact rational to the nearest number with `mant_bits` significant bits, ties to even
    (normal range; no libm, no floats)."""
    if x == 0:
        return x
    sgn, a = (-1 if x < 0 else 1), abs(x)
    e = 0
    while a >= 2:
        a /= 2
        e += 1
    while a < 1:
        a *= 2
        e -= 1
    q = a * (1 << (mant_bits - 1))            # in [2^(mb-1), 2^mb)
    f = q.numerator // q.denominator
    r = q - f
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and (f & 1)):
        f += 1
    return sgn * Fraction(f, 1 << (mant_bits - 1)) * (Fraction(2) ** e)


def test_bits_equal_torch_multiply_then_cast():
    rng = np.random.default_rng(5)
    for n, scale in ((1, 1.0), (4097, 1.0), (70_001, 0.125), (50_000, 1.0 / 48.0), (33_333, 3.0e-2)):
        g = (rng.standard_t(3, n) * 1e-3).astype(np.float32)
        bits, _ = GF.grads_finalize(g, scale)
        assert np.array_equal(bits, torch_bits(g, np.float32(scale))), (n, scale)


def test_sumsq_is_the_exactly_rounded_sum_of_the_rounded_squares():
    rng = np.random.default_rng(6)
    for n, scale in ((1000, 1.0), (70_001, 1.0 / 3.0), (40_000, 7.0)):
        g = (rng.normal(0, 1e-3, n) * rng.choice([1.0, 50.0], n)).astype(np.float32)
        bits, s = GF.grads_finalize(g, scale)
        exact = math.fsum(float(x) * float(x) for x in widen(bits).astype(np.float64))
        assert abs(s - exact) <= np.spacing(exact)
        # the plausible mistake — squaring the UNROUNDED products — is far outside that window
        wrong = math.fsum(float(x) * float(x) for x in (g * np.float32(scale)).astype(np.float64))
        assert abs(wrong - exact) > 1e3 * np.spacing(exact)


def test_sumsq_equals_a1_on_the_produced_bits():
    rng = np.random.default_rng(7)
    g = (rng.standard_t(3, 100_003) * 2e-3).astype(np.float32)
    bits, s = GF.grads_finalize(g, 0.5)
    assert s == O.sumsq(bits)                      # the optimizer's own pass over g16 sees the same S
    assert O.clip_coef(s, 1.0) == O.clip_coef(O.sumsq(bits), 1.0)


def test_hand_case_and_identity_on_representable_inputs():
    # g = (3, 4) * 2^-10, scale 0.5: products 1.5*2^-10 and 2^-9 are bf16-representable
    g = np.array([3.0 * 2.0 ** -10, 4.0 * 2.0 ** -10], np.float32)
    bits, s = GF.grads_finalize(g, 0.5)
    assert list(bits) == [0x3AC0, 0x3B00]          # 1.5*2^-10 = 0x3AC00000, 2^-9 = 0x3B000000
    assert Fraction(s) == Fraction(9, 4) * Fraction(1, 1 << 20) + Fraction(1, 1 << 18)
    # scale 1 on bf16-representable inputs is the identity
    rng = np.random.default_rng(8)
    rep = widen(rng.integers(0x3000, 0x4000, 10_000).astype(np.uint16))
    bits, s = GF.grads_finalize(rep, 1.0)
    assert np.array_equal(widen(bits), rep)
    assert s == O.sumsq(bits)
    # zeros stay zeros (pad lanes), sum 0
    bits, s = GF.grads_finalize(np.zeros(64, np.float32), 0.25)
    assert not bits.any() and s == 0.0


def test_ties_round_to_even_and_carry_into_the_exponent():
    def f(u):
        return np.array([u], np.uint32).view(np.float32)
    cases = {0x3F808000: 0x3F80,    # tie, even stays
             0x3F818000: 0x3F82,    # tie, odd goes up
             0x3F808001: 0x3F81,    # just above the tie
             0x3F807FFF: 0x3F80,    # just below
             0x3FFF8000: 0x4000,    # tie carries into the exponent
             0xBF818000: 0xBF82}    # sign symmetric
    for u, want in cases.items():
        bits, s = GF.grads_finalize(f(u), 1.0)
        assert int(bits[0]) == want, hex(u)
        w = float(widen(bits)[0])
        assert s == w * w


def test_the_product_is_rounded_to_binary32_before_the_bf16_rounding():
    """Double rounding is part of the definition (h is a binary32 value).  Exact rationals decide; inputs are
    crafted so that rounding the exact product straight to 8 bits differs from 24-then-8."""
    found = 0
    rng = np.random.default_rng(9)
    scale = np.float32(1.0 / 3.0)
    # products just above a bf16 tie whose binary32 rounding lands exactly ON the tie
    base = np.arange(0x3F808000 - 40, 0x3F808000 + 40, dtype=np.uint32).view(np.float32)
    cands = np.concatenate([base * np.float32(3.0), (rng.standard_normal(20000)).astype(np.float32)])
    bits, _ = GF.grads_finalize(cands, scale)
    for x, b in zip(cands, bits):
        exact = Fraction(float(x)) * Fraction(float(scale))
        h = rne_fraction_to_grid(exact, 24)
        two_step = rne_fraction_to_grid(h, 8)
        direct = rne_fraction_to_grid(exact, 8)
        assert Fraction(float(widen(np.array([b], np.uint16))[0])) == two_step
        found += int(two_step != direct)
    assert found > 0        # the crafted set really separates the two definitions
