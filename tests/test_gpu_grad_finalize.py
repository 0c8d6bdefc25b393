"""GPU parity for SURVEY.md §8(f) row f4, second half — the gradient producer's epilogue
(phx_grads_finalize_async, reading R34) against oracle/grad_finalize.py: bf16 bits exact,
sum of squares to the last-bit window of a fixed tree (the SAME tree as a1's: equal bit for bit), and the step that consumes the sum (no a1 pass of
its own) bit-identical to the oracle's and to the library's own a1 path."""
import numpy as np
import pytest
import torch

from oracle import grad_finalize as GF
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

from gpu_util import DEV, assert_state_equal, bits16, hp_of, make_pair

pytestmark = pytest.mark.gpu


def main_grads(n_padded, n, seed, heavy=True):
    g = torch.Generator().manual_seed(seed)
    x = torch.randn(n_padded, generator=g) * 1e-3
    if heavy:
        mask = torch.rand(n_padded, generator=g) < 0.01
        x[mask] *= 300.0
    x[n:] = 0
    return x


@pytest.mark.parametrize("numels,scale", [([64], 1.0), ([2048 * 9 + 64 * 3], 0.125), ([1_000_000, 17], 1.0 / 48.0),
                                          ([592 * 256 * 8 * 5 + 4096], 1.0),     # many one-shot CTAs + a ragged last one
                                          ([1024 * 256 * 64 + 256 * 64 * 3 + 72], 0.5)])  # > 1024 per-CTA partials
def test_finalize_bits_and_sum_match_the_oracle(numels, scale):
    wl = W.tiny_workload(numels, dp_size=1, hyper=W.Hyper(max_grad_norm=0.5))
    s, o, _, _ = make_pair(wl, steps=0)
    g32 = main_grads(s.n_padded, s.n, 3)
    want_bits, want_S = GF.grads_finalize(g32.numpy(), scale)
    d32 = g32.to(DEV)
    out = torch.full((s.n_padded,), 7.0, dtype=torch.bfloat16, device=DEV)
    S = torch.zeros(1, dtype=torch.float64, device=DEV)
    s.grads_finalize(d32, scale, out, S)
    torch.cuda.synchronize()
    assert np.array_equal(bits16(out), want_bits)
    assert torch.equal(d32.cpu(), g32)                                  # the main gradients are read-only
    got_S = float(S.item())
    assert abs(got_S - want_S) <= 4 * np.spacing(want_S)                # fixed fp64 tree vs long-double running sum
    # the step fed with that sum launches no a1 pass and is bit-identical to the oracle's step on the produced bits
    l0 = B.phx_kernel_launches(s.h)
    B.phx_set_clip_partials(s.h, S, 1)
    s.step_and_snapshot(out, 1)
    assert B.phx_kernel_launches(s.h) - l0 == 2                         # coefficient kernel + fused step, no sumsq pass
    coef, S_used = B.phx_last_clip(s.h)
    assert S_used == got_S
    assert np.float32(coef) == O.clip_coef(got_S, wl.hyper.max_grad_norm)
    o.step(want_bits, **hp_of(wl), step=1, coef=coef)
    assert_state_equal(s, o, "step fed by the producer's sum")
    s.close()


def test_producer_sum_gives_the_same_coefficient_as_the_optimizers_own_pass():
    wl = W.tiny_workload([700_000, 333], dp_size=2, dp_rank=1, hyper=W.Hyper(max_grad_norm=0.3))
    a, oa, _, _ = make_pair(wl, steps=0)
    b, ob, _, _ = make_pair(wl, steps=0)
    for t in range(1, 4):
        d32 = main_grads(a.n_padded, a.n, 40 + t).to(DEV)
        g16 = torch.empty(a.n_padded, dtype=torch.bfloat16, device=DEV)
        S = torch.zeros(1, dtype=torch.float64, device=DEV)
        a.grads_finalize(d32, 0.5, g16, S)
        B.phx_set_clip_partials(a.h, S, 1)
        a.step_and_snapshot(g16, t)                 # clip_source = producer
        b.step_and_snapshot(g16, t)                 # clip_source = the shard's own a1 pass over the same bf16 gradients
        ca, Sa = B.phx_last_clip(a.h)
        cb, Sb = B.phx_last_clip(b.h)
        assert Sa == Sb and ca == cb                # one tree shape for both kernels: the same sum, bit for bit
        torch.cuda.synchronize()
        for x, y in ((a.p, b.p), (a.m, b.m), (a.v, b.v), (a.p16, b.p16)):
            assert torch.equal(x, y)
        bits, So = GF.grads_finalize(d32.cpu().numpy(), 0.5)
        assert np.array_equal(bits16(g16), bits)
        oa.step(bits, **hp_of(wl), step=t)          # the oracle's own local clip on the oracle's bits
        assert np.float32(ca) == oa.last_coef
        assert_state_equal(a, oa, f"step {t}")
    a.close(); b.close()


def test_finalize_argument_errors():
    wl = W.tiny_workload([4096], dp_size=1, hyper=W.Hyper(max_grad_norm=1.0))
    s, _, _, _ = make_pair(wl, steps=0)
    L = B.lib()
    g32 = torch.zeros(s.n_padded + 64, device=DEV)
    g16 = torch.zeros(s.n_padded, dtype=torch.bfloat16, device=DEV)
    S = torch.zeros(2, dtype=torch.float64, device=DEV)
    assert L.phx_grads_finalize_async(s.h, g32.data_ptr() + 4, 1.0, g16.data_ptr(), S.data_ptr(), None) == B.PHX_ERR_ALIGNMENT
    assert L.phx_grads_finalize_async(s.h, g32.data_ptr(), 1.0, g16.data_ptr(), S.data_ptr() + 4, None) == B.PHX_ERR_ALIGNMENT
    assert L.phx_grads_finalize_async(s.h, g32.data_ptr(), float("nan"), g16.data_ptr(), S.data_ptr(), None) == B.PHX_ERR_INVALID_ARG
    # overlapping input and output
    assert L.phx_grads_finalize_async(s.h, g32.data_ptr(), 1.0, g32.data_ptr() + 256, S.data_ptr(), None) == B.PHX_ERR_INVALID_ARG
    s.close()
    wl32 = W.tiny_workload([4096], dp_size=1, precision="fp32")
    s32, _, _, _ = make_pair(wl32, steps=0)
    assert L.phx_grads_finalize_async(s32.h, g32.data_ptr(), 1.0, g16.data_ptr(), S.data_ptr(), None) == B.PHX_ERR_INVALID_ARG
    s32.close()
