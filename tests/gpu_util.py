"""Shared helpers of the GPU parity tests: drive the CUDA path (through the C ABI) and the
oracle on the same seeded inputs and compare bit patterns."""
import math

import numpy as np
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

DEV = "cuda:0"


def bits16(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().view(torch.int16).numpy().view(np.uint16)


def grad_record(g: torch.Tensor) -> np.ndarray:
    """The oracle's view of a gradient tensor: bf16 bits, or the float32 values themselves."""
    return g.detach().cpu().numpy().copy() if g.dtype == torch.float32 else bits16(g).copy()


def make_pair(wl, *, steps, grads=None, chunk_bytes=8 << 20, user=b"", init_mv=False, **shard_kw):
    """(Shard, OracleShard, [grad tensors on GPU], [grad bits for the oracle]) with equal initial state."""
    s = Shard(wl, device=DEV, chunk_bytes=chunk_bytes, **shard_kw)
    mgn = shard_kw.get("max_grad_norm", None)
    o = O.OracleShard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank), (wl.pp_size, wl.pp_rank),
                      chunk_bytes=(chunk_bytes + 255) & ~255,  # the library rounds chunks up to 256 B
                      max_grad_norm=wl.hyper.max_grad_norm if mgn is None else mgn, user=user,
                      flags=wl.flags(), precision=wl.precision)
    assert (o.n, o.n_padded) == (s.n, s.n_padded)
    osegs = [(tid, off, ln) for tid, _, off, ln in o.segments]
    assert osegs == s.segments
    p0 = W.init_params(s.n, s.n_padded, wl.seed)
    m0 = v0 = None
    if init_mv:
        g = torch.Generator().manual_seed(99)
        m0 = torch.randn(s.n_padded, generator=g) * 1e-4
        v0 = torch.rand(s.n_padded, generator=g) * 1e-7
        m0[s.n:] = 0
        v0[s.n:] = 0
        s.m.copy_(m0)
        s.v.copy_(v0)
    s.p.copy_(p0)
    s.set_state(0)
    o.set_state(p0.numpy(), None if m0 is None else m0.numpy(), None if v0 is None else v0.numpy())
    if user:
        B.phx_set_user_metadata(s.h, user)
    if grads is None:
        gdt = torch.float32 if wl.precision == "fp32" else torch.bfloat16
        grads = [W.gen_grads(wl, osegs, s.n_padded, t, wl.seed, dtype=gdt) for t in range(1, steps + 1)]
    gdev = [g.to(DEV) for g in grads]
    gbits = [grad_record(g) for g in grads]
    torch.cuda.synchronize()
    return s, o, gdev, gbits


def assert_state_equal(s: Shard, o: O.OracleShard, what=""):
    torch.cuda.synchronize()
    for name, dev, ref in (("p", s.p, o.p), ("m", s.m, o.m), ("v", s.v, o.v)):
        got = dev.detach().cpu().numpy().view(np.uint32)
        exp = ref.view(np.uint32)
        if not np.array_equal(got, exp):
            bad = np.flatnonzero(got != exp)
            raise AssertionError(f"{what}: {name} differs at {bad.size} of {exp.size} lanes, first {bad[:5]}: "
                                 f"{got[bad[:3]]} vs {exp[bad[:3]]}")
    if s.p16 is not None:
        got = bits16(s.p16)
        if not np.array_equal(got, o.p16):
            bad = np.flatnonzero(got != o.p16)
            raise AssertionError(f"{what}: p16 differs at {bad.size} lanes, first {bad[:5]}")
    assert B.phx_last_step(s.h) == o.last_step, what


def metric_ii(a, b):
    """max |a-b| / (|b| + rms(b)) — DESIGN.md reading R22 (the floor-normalised relative error)."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    return float(np.max(np.abs(a - b) / (np.abs(b) + math.sqrt(np.mean(b * b)) + 1e-300)))


def hp_of(wl):
    h = wl.hyper
    return dict(lr=h.lr, beta1=h.beta1, beta2=h.beta2, eps=h.eps, wd=h.wd)
