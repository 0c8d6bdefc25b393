"""global_clip.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle of the DP-global gradient-norm clip ("Two scalar collectives sit beside
it in real training: all-reduce of sum g^2 for the global clip"; BASELINE.json:configs[2]:
"Global grad-norm clip 1.0").  The paper itself never mentions clipping; reading R7b.

Plain definition.  With D data-parallel ranks, rank r holds the gradient shard g_r of the
contiguous range [r*N/D, (r+1)*N/D) of ONE flat parameter space (a0).  The norm that decides the
clip is the norm of the WHOLE gradient,

    S    = sum_r sum_i g_{r,i}^2        (every square exact, one long-double running sum taken over
                                         the concatenation g_0 ‖ g_1 ‖ ... ‖ g_{D-1}, rounded to
                                         double once — the same routine as the shard-local S of R7)
    coef = fp32( min(1, max_norm / (sqrt(S) + 1e-6)) )

and EVERY rank applies the same coef in its AdamW step.  Pad lanes hold g = 0 and add nothing.

There is no blocking, tree or per-rank partial here: the definition does not have one.  (The CUDA
path computes one fp64 partial per rank, exchanges the D scalars and sums them in rank order; that
differs from this by reassociation only, <~1e-16 relative — the caveat already stated for R7.)

Pins (tests/test_oracle_global_clip.py): partition invariance against the already pinned dp_size=1
shard-local clip (bitwise, on the union of the shards); a hand-computable norm whose coefficient is
re-derived with exact rationals; math.fsum over all ranks; monotonicity (coef_global <= every
coef_local); D=1 reduces to R7; a wrong "local norm per rank" implementation is shown to fail.
Nothing here is "parity unpinned".
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np

from . import oracle as O


def global_sumsq(grads_by_rank: Sequence[np.ndarray]) -> float:
    """S over all ranks: the sum of squares of the concatenation in rank order."""
    assert len(grads_by_rank) >= 1
    dt = grads_by_rank[0].dtype
    assert all(g.dtype == dt for g in grads_by_rank)
    cat = np.ascontiguousarray(np.concatenate([np.asarray(g).reshape(-1) for g in grads_by_rank]))
    return O.sumsq(cat)


def global_clip_coef(grads_by_rank: Sequence[np.ndarray], max_norm: float) -> np.float32:
    """The one coefficient all D ranks apply."""
    return O.clip_coef(global_sumsq(grads_by_rank), max_norm)


class OracleDPGroup:
    """D oracle shards of one flat parameter space that step together under the global clip."""

    def __init__(self, layout, dp_size: int, max_grad_norm: float, **shard_kw):
        assert max_grad_norm > 0.0
        self.D = int(dp_size)
        self.max_grad_norm = float(max_grad_norm)
        # the shards never decide the clip themselves: max_grad_norm=0 in each, coef is passed in
        self.shards: List[O.OracleShard] = [O.OracleShard(layout, dp_size, r, max_grad_norm=0.0, **shard_kw)
                                            for r in range(self.D)]
        self.last_sumsq = 0.0
        self.last_coef = np.float32(1.0)

    def step(self, grads_by_rank: Sequence[np.ndarray], lr, beta1, beta2, eps, wd, step):
        assert len(grads_by_rank) == self.D
        self.last_sumsq = global_sumsq(grads_by_rank)
        self.last_coef = O.clip_coef(self.last_sumsq, self.max_grad_norm)
        for s, g in zip(self.shards, grads_by_rank):
            s.step(g, lr, beta1, beta2, eps, wd, step, coef=self.last_coef)
        return self.last_coef
