"""CPU tier for the DP-global clip plumbing: the one collective of the path — an
all-gather of one double per rank — on world_size-2 and -3 gloo groups, checked against the oracle's
global coefficient; argument errors of the two entry points without a GPU."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import global_clip as GC
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import clip as PC


def _grads(rank, n=4096):
    rng = np.random.default_rng(500 + rank)
    t = torch.as_tensor((rng.standard_t(3, n) * 1e-3 * (rank + 1)).astype(np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo")
    # each rank's local sum (here the oracle's routine stands where phx_grad_sumsq_async runs on a GPU box:
    # this test covers the exchange and its ordering, not the kernel)
    local = torch.tensor([O.sumsq(_grads(rank))], dtype=torch.float64)
    got = PC.gather_partials(local)
    q.put((rank, got.tolist()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_partials_are_gathered_in_rank_order_on_gloo(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29650 + (os.getpid() + 11 * world) % 120
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = [O.sumsq(_grads(r)) for r in range(world)]
    for r in range(world):
        assert res[r] == want                      # every rank holds the same D values, in rank order
    # summing them in rank order reproduces the oracle's global sum up to the last rounding
    S = GC.global_sumsq([_grads(r) for r in range(world)])
    assert abs(sum(want) - S) <= 2 * np.spacing(S)
    assert O.clip_coef(sum(want), 0.01) == GC.global_clip_coef([_grads(r) for r in range(world)], 0.01)


def test_gather_without_a_process_group_is_the_single_rank_case():
    x = torch.tensor([0.375], dtype=torch.float64)
    y = PC.gather_partials(x)
    assert y.tolist() == [0.375] and y.data_ptr() != x.data_ptr()


def test_entry_points_fail_loudly_without_binding_or_gpu():
    L = B.lib()
    h = B.phx_shard_create([(100, 0)], 2, 0, max_grad_norm=1.0)
    assert L.phx_grad_sumsq_async(None, 256, 256, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_grad_sumsq_async(h, 256, 256, None) == B.PHX_ERR_NOT_BOUND       # never a host stand-in
    assert L.phx_grad_sumsq_async(h, None, 256, None) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(None, 256, 1) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(h, 256, 0) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(h, 256, 1025) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_clip_partials(h, 260, 2) == B.PHX_ERR_ALIGNMENT
    assert L.phx_set_clip_partials(h, 256, 2) == B.PHX_OK
    assert L.phx_set_clip_partials(h, None, 0) == B.PHX_OK
    B.phx_shard_destroy(h)
    h = B.phx_shard_create([(100, 0)], 2, 0)                                     # no clip configured
    assert L.phx_set_clip_partials(h, 256, 2) == B.PHX_ERR_INVALID_ARG
    B.phx_shard_destroy(h)
