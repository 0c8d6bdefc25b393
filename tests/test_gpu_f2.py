"""GPU parity for SURVEY.md §8(f2): the paper's own precision (binary32 gradients, no bf16 copy,
PAPER.md:270) and per-tensor decay groups, through the C ABI against the CPU oracle — bit-exact on
p, m, v, the packed snapshot, the committed replica, restore and resume."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, assert_state_equal, bits16, grad_record, hp_of, make_pair

pytestmark = pytest.mark.gpu

SIZES = [[1], [64], [70], [2047, 1], [2048 * 3 + 64], [256 * 8 * 5 + 192, 33, 1000], [300_000, 77, 12_345]]


@pytest.mark.parametrize("numels", SIZES)
@pytest.mark.parametrize("dp", [1, 3])
def test_fp32_precision_sizes_snapshot_restore(numels, dp):
    wl = W.tiny_workload(numels, dp_size=dp, dp_rank=dp - 1, precision="fp32", grad_kind="heavy_tail")
    s, o, gdev, gbits = make_pair(wl, steps=4, chunk_bytes=4096, init_mv=True)
    assert s.p16 is None and gdev[0].dtype == torch.float32
    side = torch.cuda.Stream(device=DEV)
    for t in range(1, 4):
        s.step_and_snapshot(gdev[t - 1], t)
        s.flush_async(side)
        o.step(gbits[t - 1], **hp_of(wl), step=t)
        o.snapshot()
        assert_state_equal(s, o, f"{numels} dp{dp} step {t}")
        assert np.array_equal(s.staging_slot(t).cpu().numpy(), o.packed_snapshot())
        s.wait(t)
        assert np.array_equal(s.replica_slot(t).numpy(), o.replica[t % 2])
    if s.n < s.n_padded:
        for a in (s.p, s.m, s.v):
            assert not a[s.n:].cpu().numpy().view(np.uint32).any()
    s.step_and_snapshot(gdev[3], 4)        # in flight when the fault hits
    s.drop_live()
    assert s.restore() == 3 and o.last_step == 3
    assert_state_equal(s, o, "restore")
    s.step_and_snapshot(gdev[3], 4)        # recompute
    o.step(gbits[3], **hp_of(wl), step=4)
    assert_state_equal(s, o, "recompute")
    s.close()


# tensors chosen so that decay/no-decay boundaries fall inside 2048-element tiles, on tile edges, inside an
# 8-element group, at the very start, and at the very end of a rank's range
GROUP_CASES = [
    ([5000, 7, 4096, 1, 1, 3000], (1, 3), 1),
    ([5000, 7, 4096, 1, 1, 3000], (0, 2, 5), 1),
    ([2048, 2048, 2048, 2048], (1, 2), 1),
    ([2048 * 5 + 3, 10, 2048 * 3 - 13, 100, 5], (1, 3, 4), 3),
    ([100_000, 256, 256, 300_000, 1024, 77], (1, 2, 4), 2),
    ([64], (0,), 1),
]


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("numels,nd,dp", GROUP_CASES)
def test_decay_groups_bit_exact_on_every_rank(numels, nd, dp, precision):
    for rank in range(dp):
        wl = W.tiny_workload(numels, dp_size=dp, dp_rank=rank, precision=precision, no_decay_ids=tuple(nd))
        s, o, gdev, gbits = make_pair(wl, steps=4, chunk_bytes=8192, init_mv=True)
        side = torch.cuda.Stream(device=DEV)
        for t in range(1, 5):
            s.step_and_snapshot(gdev[t - 1], t)
            s.flush_async(side)
            o.step(gbits[t - 1], **hp_of(wl), step=t)
            o.snapshot()
            assert_state_equal(s, o, f"{numels} nd{nd} rank {rank}/{dp} {precision} step {t}")
        s.wait(4)
        assert np.array_equal(s.replica_slot(4).numpy(), o.replica[0])
        s.close()


def test_decay_groups_differ_from_uniform_decay_and_match_wd_zero():
    numels, nd = [4096, 512, 4096], (1,)
    wl_g = W.tiny_workload(numels, dp_size=1, no_decay_ids=nd)
    wl_u = W.tiny_workload(numels, dp_size=1)
    wl_z = dataclasses.replace(wl_u, hyper=W.Hyper(wd=0.0))
    out = {}
    for key, wl in (("g", wl_g), ("u", wl_u), ("z", wl_z)):
        s, o, gdev, gbits = make_pair(wl, steps=5)
        for t in range(1, 6):
            s.step_and_snapshot(gdev[t - 1], t)
        torch.cuda.synchronize()
        out[key] = s.p.cpu().numpy().view(np.uint32).copy()
        s.close()
    a, b = 4096, 4096 + 512
    assert np.array_equal(out["g"][a:b], out["z"][a:b])          # flagged tensor == wd = 0 trajectory
    assert np.array_equal(out["g"][:a], out["u"][:a]) and np.array_equal(out["g"][b:], out["u"][b:])
    assert not np.array_equal(out["g"][a:b], out["u"][a:b])


@pytest.mark.parametrize("rank", [1, 3])
@pytest.mark.parametrize("precision", ["bf16", "fp32"])
def test_c1_with_gpt_parameter_groups_ten_steps(precision, rank):
    # config c1's real tensor list: biases and LayerNorm weights flagged no-decay (34 small tensors, most
    # toggles inside a tile); rank 0 holds only the embedding, so the ranks that hold layers are used
    wl = dataclasses.replace(W.CONFIGS["c1"], decay_groups=True, precision=precision, dp_rank=rank)
    assert sum(wl.flags()) == 4 * 8 + 2
    s, o, gdev, gbits = make_pair(wl, steps=10)
    assert o.no_decay is not None and 0 < int(o.no_decay.sum()) < o.n
    side = torch.cuda.Stream(device=DEV)
    for t in range(1, 11):
        s.step_and_snapshot(gdev[t - 1], t)
        s.flush_async(side)
        o.step(gbits[t - 1], **hp_of(wl), step=t, nthreads=4)
        o.snapshot()
        assert_state_equal(s, o, f"c1 groups {precision} step {t}")
    s.wait(10)
    assert np.array_equal(s.replica_slot(10).numpy(), o.replica[0])
    s.drop_live()
    assert s.restore() == 10
    assert_state_equal(s, o, "restore")
    s.close()


@pytest.mark.parametrize("n,max_norm", [(64, 1e-3), (5000, 0.01), (1_000_000, 0.5), (1_000_000, 1e6)])
def test_fp32_clip_coefficient_and_clipped_step(n, max_norm):
    wl = W.tiny_workload([n], dp_size=1, precision="fp32", grad_kind="heavy_tail",
                         hyper=W.Hyper(max_grad_norm=max_norm))
    s, o, gdev, gbits = make_pair(wl, steps=3)
    for t in range(1, 4):
        s.step_and_snapshot(gdev[t - 1], t)
        o.step(gbits[t - 1], **hp_of(wl), step=t)
        coef, S = B.phx_last_clip(s.h)
        So = O.sumsq(gbits[t - 1])
        assert abs(S - So) <= 1e-13 * So
        assert np.float32(coef) == o.last_coef
        assert_state_equal(s, o, f"clip step {t}")
    s.close()


def test_fp32_hand_computable_clip():
    # g = (3, 4, 12) * 2^-12  =>  S = 169 * 2^-24 exactly, norm 13 * 2^-12
    wl = W.tiny_workload([64], dp_size=1, precision="fp32", hyper=W.Hyper(max_grad_norm=1e-3))
    g = torch.zeros(64, dtype=torch.float32)
    g[:3] = torch.tensor([3.0, 4.0, 12.0]) * 2.0 ** -12
    s, o, gdev, gbits = make_pair(wl, steps=1, grads=[g])
    s.step_and_snapshot(gdev[0], 1)
    coef, S = B.phx_last_clip(s.h)
    assert S == 169.0 * 2.0 ** -24
    assert np.float32(coef) == np.float32(float(np.float32(1e-3)) / (13 * 2.0 ** -12 + 1e-6))
    o.step(gbits[0], **hp_of(wl), step=1)
    assert_state_equal(s, o, "hand clip")
    s.close()


def test_f2_fp32_shard_needs_no_bf16_buffer_but_bf16_precision_does():
    wl = W.tiny_workload([4096], dp_size=1, precision="fp32")
    s = Shard(wl, device=DEV)
    assert s.p16 is None
    s.close()
    # a bf16-precision shard still requires the bf16 buffer
    h = B.phx_shard_create([(4096, 0)], 1, 0)
    p = torch.zeros(4096, device=DEV)
    with pytest.raises(B.PhxError) as e:
        B.phx_shard_bind(h, p, p.clone(), p.clone(), None, torch.zeros(2 * (256 + 12 * 4096), dtype=torch.uint8, device=DEV),
                         torch.zeros(2 * (256 + 12 * 4096), dtype=torch.uint8).pin_memory())
    assert e.value.code == B.PHX_ERR_INVALID_ARG
    B.phx_shard_destroy(h)
