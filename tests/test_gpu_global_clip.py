"""GPU parity for the DP-global gradient-norm clip (BASELINE.json:configs[2]): D logical
ranks on one device step through the C ABI (phx_grad_sumsq_async -> gather -> phx_set_clip_partials ->
phx_step_and_snapshot) and are compared bit for bit with oracle/global_clip.py's OracleDPGroup."""
import numpy as np
import pytest
import torch

from oracle import global_clip as GC
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import clip as PC
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, assert_state_equal, bits16, grad_record, hp_of

pytestmark = pytest.mark.gpu


def make_group(numels, D, max_norm, precision="bf16", steps=4, **shard_kw):
    wls = [W.tiny_workload(numels, dp_size=D, dp_rank=r, precision=precision, grad_kind="heavy_tail",
                           hyper=W.Hyper(max_grad_norm=max_norm)) for r in range(D)]
    shards = [Shard(wl, device=DEV, chunk_bytes=1 << 16, **shard_kw) for wl in wls]
    grp = GC.OracleDPGroup(wls[0].layout(), D, max_norm, precision=precision, chunk_bytes=1 << 16)
    gdt = torch.float32 if precision == "fp32" else torch.bfloat16
    gdev, grec = [], []
    for r, (s, o) in enumerate(zip(shards, grp.shards)):
        assert (s.n, s.n_padded) == (o.n, o.n_padded)
        p0 = W.init_params(s.n, s.n_padded, 10 + r)
        s.p.copy_(p0)
        s.set_state(0)
        o.set_state(p0.numpy())
    for t in range(1, steps + 1):
        row = []
        for r, s in enumerate(shards):
            g = W.gen_grads(wls[r], s.segments, s.n_padded, t, seed=100 + r, dtype=gdt)
            g = (g.float() * (0.25 + r)).to(gdt)          # ranks with very different local norms
            row.append(g)
        gdev.append([g.to(DEV) for g in row])
        grec.append([grad_record(g) for g in row])
    torch.cuda.synchronize()
    return wls, shards, grp, gdev, grec


@pytest.mark.parametrize("precision", ["bf16", "fp32"])
@pytest.mark.parametrize("D,numels", [(1, [5000, 77]), (2, [300_000, 1234, 77]), (3, [2048 * 7 + 5, 64, 1]),
                                      (4, [100, 3]), (8, [70_000, 50_001])])
def test_global_clip_group_matches_the_oracle(D, numels, precision):
    max_norm = 0.002
    wls, shards, grp, gdev, grec = make_group(numels, D, max_norm, precision)
    hp = hp_of(wls[0])
    side = torch.cuda.Stream(device=DEV)
    for t in range(1, 4):
        partials = PC.step_group_in_process(shards, gdev[t - 1], t)
        coef = grp.step(grec[t - 1], **hp, step=t)
        assert float(coef) < 1.0
        torch.cuda.synchronize()
        # per-rank sums: the device tree vs the exactly rounded sum (reassociation only)
        got = partials.cpu().numpy()
        for r in range(D):
            want = O.sumsq(grec[t - 1][r])
            assert abs(got[r] - want) <= 16 * np.spacing(want), (r, got[r], want)
        for r, (s, o) in enumerate(zip(shards, grp.shards)):
            c, S = B.phx_last_clip(s.h)
            assert np.float32(c).view(np.uint32) == coef.view(np.uint32), (t, r, c, float(coef))
            assert abs(S - grp.last_sumsq) <= 16 * np.spacing(grp.last_sumsq)
            assert_state_equal(s, o, f"D{D} {precision} step {t} rank {r}")
            s.flush_async(side)
            o.snapshot()
            s.wait(t)
            assert np.array_equal(s.replica_slot(t).numpy(), o.replica[t % 2])
    # every rank used the SAME coefficient bits
    cs = {np.float32(B.phx_last_clip(s.h)[0]).view(np.uint32).item() for s in shards}
    assert len(cs) == 1
    for s in shards:
        s.close()


def test_restore_clears_the_partials_and_the_recompute_supplies_them_again():
    D, max_norm = 2, 0.02
    wls, shards, grp, gdev, grec = make_group([40_000, 999], D, max_norm, steps=4)
    hp = hp_of(wls[0])
    side = torch.cuda.Stream(device=DEV)
    for t in (1, 2, 3):
        PC.step_group_in_process(shards, gdev[t - 1], t)
        grp.step(grec[t - 1], **hp, step=t)
        for s, o in zip(shards, grp.shards):
            s.flush_async(side)
            o.snapshot()
    for s in shards:
        s.wait(3)
    # step 4 in flight on rank 0 when it is lost; rank 1 finished its step 4
    partials = PC.step_group_in_process(shards, gdev[3], 4)
    keep = partials.clone()
    s0, o0 = shards[0], grp.shards[0]
    # stale one-shot partials must not survive a restore
    B.phx_set_clip_partials(s0.h, torch.full((2,), 1e30, dtype=torch.float64, device=DEV), 2)
    s0.drop_live()
    assert s0.restore() == 3
    assert_state_equal(s0, o0, "restore")
    # recompute: the lost rank recomputes its sum; the survivor's sum of step 4 is still known
    fresh = torch.zeros(2, dtype=torch.float64, device=DEV)
    B.phx_grad_sumsq_async(s0.h, gdev[3][0], fresh.data_ptr(), torch.cuda.current_stream())
    fresh[1] = keep[1]
    B.phx_set_clip_partials(s0.h, fresh, 2)
    s0.step_and_snapshot(gdev[3][0], 4)
    grp.step(grec[3], **hp, step=4)
    assert_state_equal(s0, o0, "recompute rank 0")
    assert_state_equal(shards[1], grp.shards[1], "survivor")
    for s in shards:
        s.close()


def test_count_one_with_the_own_sum_is_bit_identical_to_the_local_clip():
    wl = W.tiny_workload([123_457, 64], dp_size=1, grad_kind="heavy_tail", hyper=W.Hyper(max_grad_norm=0.05))
    a, b = Shard(wl, device=DEV), Shard(wl, device=DEV)
    p0 = W.init_params(a.n, a.n_padded, 3)
    for s in (a, b):
        s.p.copy_(p0)
        s.set_state(0)
    own = torch.zeros(1, dtype=torch.float64, device=DEV)
    for t in (1, 2):
        g = W.gen_grads(wl, a.segments, a.n_padded, t, 7).to(DEV)
        a.step_and_snapshot(g, t)                                   # local a1
        B.phx_grad_sumsq_async(b.h, g, own, torch.cuda.current_stream())
        B.phx_set_clip_partials(b.h, own, 1)
        b.step_and_snapshot(g, t)
        torch.cuda.synchronize()
        assert B.phx_last_clip(a.h) == B.phx_last_clip(b.h)
        for x, y in ((a.p, b.p), (a.m, b.m), (a.v, b.v), (a.p16, b.p16)):
            assert torch.equal(x.view(torch.int32) if x.dtype == torch.float32 else x.view(torch.int16),
                               y.view(torch.int32) if y.dtype == torch.float32 else y.view(torch.int16))
    # one-shot: the next step of b falls back to its own pass
    g = W.gen_grads(wl, a.segments, a.n_padded, 3, 7).to(DEV)
    a.step_and_snapshot(g, 3)
    b.step_and_snapshot(g, 3)
    torch.cuda.synchronize()
    assert B.phx_last_clip(a.h) == B.phx_last_clip(b.h) and torch.equal(a.p, b.p)
    a.close()
    b.close()


def test_argument_errors():
    wl0 = W.tiny_workload([1000], dp_size=1)                         # no clip configured
    s = Shard(wl0, device=DEV)
    d = torch.zeros(4, dtype=torch.float64, device=DEV)
    g = torch.zeros(s.n_padded, dtype=torch.bfloat16, device=DEV)
    L = B.lib()
    assert L.phx_set_clip_partials(s.h, d.data_ptr(), 1) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(s.h, None, 0) == B.PHX_OK
    assert L.phx_grad_sumsq_async(s.h, g.data_ptr(), None, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_grad_sumsq_async(s.h, None, d.data_ptr(), None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_grad_sumsq_async(s.h, g.data_ptr(), d.data_ptr() + 4, None) == B.PHX_ERR_ALIGNMENT
    assert L.phx_grad_sumsq_async(s.h, g.data_ptr() + 2, d.data_ptr(), None) == B.PHX_ERR_ALIGNMENT
    B.phx_grad_sumsq_async(s.h, g, d, None)                           # the sum alone is always available
    s.close()
    wl1 = W.tiny_workload([1000], dp_size=1, hyper=W.Hyper(max_grad_norm=1.0))
    s = Shard(wl1, device=DEV)
    assert L.phx_set_clip_partials(s.h, d.data_ptr(), 0) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(s.h, d.data_ptr(), 1025) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(s.h, d.data_ptr() + 4, 1) == B.PHX_ERR_ALIGNMENT
    assert L.phx_set_clip_partials(s.h, d.data_ptr(), 4) == B.PHX_OK
    s.close()


@pytest.mark.parametrize("n", [64, 4096, 300_032])
def test_sum_of_squares_over_zeros_subnormals_and_extreme_exponents(n):
    """The integer widening of k_sumsq_partial (exponent re-bias, no cvt) against the oracle's double squares on
    bit patterns that exercise both of its paths: zeros of either sign, bf16 subnormals, the smallest and the
    largest normal exponents (whose squares leave the binary32 range but not binary64)."""
    rng = np.random.default_rng(n)
    wl = W.tiny_workload([n], dp_size=1, hyper=W.Hyper(max_grad_norm=1.0))
    s = Shard(wl, device=DEV)
    out = torch.zeros(1, dtype=torch.float64, device=DEV)
    cases = {
        "normal": rng.integers(0x3000, 0x4000, n),                                     # ~1e-10 .. 2
        "signed": rng.integers(0x3000, 0x4000, n) | (rng.integers(0, 2, n) << 15),
        "with zeros": np.where(rng.random(n) < 0.3, 0, rng.integers(0x3000, 0x4000, n)),
        "neg zeros": np.where(rng.random(n) < 0.1, 0x8000, rng.integers(0x3A00, 0x3B00, n)),
        "subnormals": np.where(rng.random(n) < 0.05, rng.integers(1, 0x80, n), rng.integers(0x0080, 0x0200, n)),
        "tiny normals": rng.integers(0x0080, 0x0400, n),                                # squares < 2^-240
        "huge": rng.integers(0x7E00, 0x7F80, n),                                        # squares up to 2^255
        "all zero": np.zeros(n, np.int64),
        "one element": np.where(np.arange(n) == n - 7, 0x3F80, 0),
    }
    for name, bits in cases.items():
        b = np.ascontiguousarray(bits.astype(np.uint16))
        b[s.n:] = 0
        g = torch.from_numpy(b.view(np.int16)).view(torch.bfloat16).to(DEV)
        B.phx_grad_sumsq_async(s.h, g, out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        want = O.sumsq(b)
        got = float(out.item())
        assert np.isfinite(want)
        assert abs(got - want) <= 16 * np.spacing(want), (name, got, want)
    # non-finite gradients keep their IEEE meaning (outside the parity domain, reading R8)
    b = np.full(n, 0x3C00, np.uint16)
    b[3] = 0x7F80
    g = torch.from_numpy(b.view(np.int16)).view(torch.bfloat16).to(DEV)
    B.phx_grad_sumsq_async(s.h, g, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.isinf(out.item())
    b[3] = 0x7FC0
    g = torch.from_numpy(b.view(np.int16)).view(torch.bfloat16).to(DEV)
    B.phx_grad_sumsq_async(s.h, g, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.isnan(out.item())
    s.close()


_NCCL_CHILD = r"""
import os, sys
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, os.path.join(sys.argv[1], "tests"))
import numpy as np, torch, torch.distributed as dist
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B, workloads as W
from paper_2607_01646_b200.clip import GlobalClip
from paper_2607_01646_b200.shard import Shard
from gpu_util import DEV, assert_state_equal, grad_record, hp_of
torch.cuda.set_device(0)
dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device(DEV))
assert dist.get_backend() == "nccl"
wl = W.tiny_workload([300_000, 1234, 77], dp_size=1, grad_kind="heavy_tail", hyper=W.Hyper(max_grad_norm=0.01))
s = Shard(wl, device=DEV, chunk_bytes=1 << 16)
o = O.OracleShard(wl.layout(), 1, 0, chunk_bytes=1 << 16, max_grad_norm=0.01)
p0 = W.init_params(s.n, s.n_padded, 5)
s.p.copy_(p0); s.set_state(0); o.set_state(p0.numpy())
gc = GlobalClip(s)                                   # default group = the NCCL world
st = torch.cuda.Stream(device=DEV)                   # not the default stream: the exchange must follow `st`
for t in range(1, 5):
    g = W.gen_grads(wl, s.segments, s.n_padded, t, 11)
    gd = g.to(DEV)
    torch.cuda.synchronize()
    gc.step_and_snapshot(gd, t, stream=st)           # sumsq -> NCCL all-gather -> coefficient -> fused step, no host sync
    coef = o.step(grad_record(g), **hp_of(wl), step=t)
    torch.cuda.synchronize()
    c, S = B.phx_last_clip(s.h)
    assert np.float32(c).view(np.uint32) == np.float32(o.last_coef).view(np.uint32), (t, c, o.last_coef)
    assert_state_equal(s, o, f"nccl world-1 step {t}")
s.close()
dist.destroy_process_group()
print("NCCL_CLIP_OK")
"""


def test_global_clip_through_a_real_nccl_all_gather():
    """The branch of clip.gather_partials a GPU box takes — a CUDA-tensor all-gather on an NCCL group, enqueued on the
    step's (non-default) stream — run on the one GPU there is (world of ONE rank: D = 1 is the local clip, so the
    oracle is the pinned dp = 1 rule).  In a child process so that the NCCL communicator does not outlive the test."""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r = subprocess.run([sys.executable, "-c", _NCCL_CHILD, root], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0 and "NCCL_CLIP_OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
