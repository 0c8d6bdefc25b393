"""twin.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Independent restatements used to cross-check phx_oracle.c (SURVEY.md §8(c) "what
pins each part"):
  * adamw_step_numpy : the canonical sequence (reading R1) as numpy float32 array
    operations — each numpy ufunc rounds once to binary32, sqrt and divide are
    correctly rounded, there is no FMA — so it must agree with the C loop bit for bit;
  * adamw_step_f64   : the same recurrences in float64 with unrounded derived
    scalars (the "float64 shadow" of the pins);
  * adamw_closed_form_exact : exact rational arithmetic (fractions.Fraction) for the
    first step from m = v = 0, the closed form of SURVEY.md §8(c);
  * sumsq_exact      : math.fsum, the exactly rounded sum of the exact squares.
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np

f32 = np.float32


def pow_sqmul(b: float, t: int) -> float:
    r = 1.0
    while t:
        if t & 1:
            r = r * b
        b = b * b
        t >>= 1
    return r


def scalars_f32(lr, beta1, beta2, eps, wd, t):
    """Python floats are IEEE doubles: the hyperparameters arrive as C floats, are
    widened exactly, combined in double and rounded once to fp32 (reading R6)."""
    lr, b1, b2, wd = float(f32(lr)), float(f32(beta1)), float(f32(beta2)), float(f32(wd))
    return (f32(1.0 - lr * wd), f32(1.0 - b1), f32(1.0 - b2),
            f32(lr / (1.0 - pow_sqmul(b1, t))), f32(math.sqrt(1.0 - pow_sqmul(b2, t))))


def widen(g_bits: np.ndarray) -> np.ndarray:
    return (g_bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


def rne_bf16_numpy(x: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))
    return ((u >> np.uint64(16)) & np.uint64(0xFFFF)).astype(np.uint16)


def adamw_step_numpy(p, m, v, g_bits, lr, beta1, beta2, eps, wd, t, coef=1.0):
    """Returns (p', m', v', p16) — inputs untouched."""
    decay, omb1, omb2, ss, sbc2 = scalars_f32(lr, beta1, beta2, eps, wd, t)
    b1, b2, e = f32(beta1), f32(beta2), f32(eps)
    with np.errstate(all="ignore"):
        g = widen(g_bits) * f32(coef)
        p1 = p * decay
        mn = (b1 * m) + (omb1 * g)
        vn = (b2 * v) + (omb2 * (g * g))
        d = (np.sqrt(vn) / sbc2) + e
        pn = p1 - (ss * (mn / d))
    for a in (g, p1, mn, vn, d, pn):
        assert a.dtype == np.float32
    return pn, mn, vn, rne_bf16_numpy(pn)


def adamw_step_numpy_ex(p, m, v, g, lr, beta1, beta2, eps, wd, t, coef=1.0, no_decay=None, bf16_copy=True):
    """The general routine of SURVEY.md §8(f2) as numpy float32 array operations: `g` is uint16
    bf16 bits (widened exactly) or float32 gradients; `no_decay` is an optional
    boolean/uint8 mask (reading R5b: decay 1.0f on flagged elements).  Returns (p', m', v', p16|None)."""
    decay, omb1, omb2, ss, sbc2 = scalars_f32(lr, beta1, beta2, eps, wd, t)
    b1, b2, e = f32(beta1), f32(beta2), f32(eps)
    with np.errstate(all="ignore"):
        gw = widen(g) if g.dtype == np.uint16 else g
        gw = gw * f32(coef)
        dk = decay if no_decay is None else np.where(np.asarray(no_decay) != 0, f32(1.0), decay).astype(np.float32)
        p1 = p * dk
        mn = (b1 * m) + (omb1 * gw)
        vn = (b2 * v) + (omb2 * (gw * gw))
        d = (np.sqrt(vn) / sbc2) + e
        pn = p1 - (ss * (mn / d))
    for a in (gw, p1, mn, vn, d, pn):
        assert a.dtype == np.float32
    return pn, mn, vn, (rne_bf16_numpy(pn) if bf16_copy else None)


def sumsq_exact_f32(g: np.ndarray) -> float:
    """math.fsum of the exact squares of binary32 gradients (each square is exact in double)."""
    x = np.asarray(g, dtype=np.float32).astype(np.float64)
    return math.fsum((x * x).tolist())


def adamw_step_f64(p, m, v, g, lr, beta1, beta2, eps, wd, t):
    """float64 shadow: textbook AdamW (decoupled decay, bias-corrected, eps outside the
    square root after bias-correcting v) on float64 arrays; hyperparameters are the
    exact values of the C floats."""
    lr, b1, b2 = float(f32(lr)), float(f32(beta1)), float(f32(beta2))
    eps, wd = float(f32(eps)), float(f32(wd))
    mn = b1 * m + (1.0 - b1) * g
    vn = b2 * v + (1.0 - b2) * g * g
    mhat = mn / (1.0 - b1 ** t)
    vhat = vn / (1.0 - b2 ** t)
    pn = p * (1.0 - lr * wd) - lr * mhat / (np.sqrt(vhat) + eps)
    return pn, mn, vn


def adamw_first_step_exact(p0: Fraction, g: Fraction, lr, beta1, beta2, eps, wd):
    """Exact rational value of step 1 from m = v = 0 with g != 0:
    m1 = (1-b1) g, v1 = (1-b2) g^2, p1 = p0 (1 - lr wd) - lr g / (|g| + eps)
    (closed form: the bias corrections cancel exactly)."""
    F = lambda x: Fraction(float(f32(x)))
    lr, b1, b2, eps, wd = F(lr), F(beta1), F(beta2), F(eps), F(wd)
    m1 = (1 - b1) * g
    v1 = (1 - b2) * g * g
    p1 = p0 * (1 - lr * wd) - lr * g / (abs(g) + eps)
    return p1, m1, v1


def sumsq_exact(g_bits: np.ndarray) -> float:
    g = widen(g_bits).astype(np.float64)
    return math.fsum((g * g).tolist())
