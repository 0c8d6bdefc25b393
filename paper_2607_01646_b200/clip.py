"""DP-global gradient-norm clip plumbing (BASELINE.json:configs[2] "Global grad-norm
clip 1.0").  Marshalling only: the per-rank sum of squares (phx_grad_sumsq_async) and the coefficient
(inside phx_step_and_snapshot, from the exchanged per-rank sums) are computed by libphx's kernels; the
ONE collective of the path — an all-gather of D doubles, 8*D bytes — is torch.distributed's (NCCL on
the step's stream on a GPU box, gloo in the CPU tests of this plumbing).

An all-GATHER followed by a sum in rank order inside libphx (not an all-reduce) so that the bits of S
do not depend on the collective library's reduction algorithm: every rank sums the same D doubles in
the same fixed tree and gets the same coefficient.

    gc = GlobalClip(shard, group=dp_group)         # one process per GPU
    gc.step_and_snapshot(grads, step)              # sumsq -> all-gather -> step (one stream, no host sync)
Single process (tests, the 1-GPU bench stand-in): step_group_in_process(shards, grads_by_rank, step)
runs D logical ranks living on one device and gathers with a device-side copy instead of NCCL.
"""
from __future__ import annotations

from typing import Optional, Sequence

from . import binding as B


def gather_partials(local, group=None):
    """All-gather of one double per rank, returned in rank order (tensor of D doubles on local's
    device).  Works on CPU tensors with gloo (host-logic tests) and CUDA tensors with NCCL."""
    import torch
    import torch.distributed as dist
    assert local.dtype == torch.float64 and local.numel() == 1
    if not (dist.is_available() and dist.is_initialized()):
        return local.reshape(1).clone()
    world = dist.get_world_size(group)
    if local.is_cuda and dist.get_backend(group) != "nccl":
        # a gloo control plane (CPU tests; bench.py --debug-shared-gpu) cannot all-gather device tensors: stage
        # the 8 bytes through the host.  This synchronises the host with the stream — a functional path only;
        # on a GPU box the group is NCCL and the exchange is enqueued on the step's stream.
        host = torch.empty(world, dtype=torch.float64)
        dist.all_gather_into_tensor(host, local.reshape(1).cpu(), group=group)
        return host.to(local.device)
    out = torch.empty(world, dtype=torch.float64, device=local.device)
    dist.all_gather_into_tensor(out, local.reshape(1), group=group)
    return out


class GlobalClip:
    """One rank's side of the global clip.  `shard` must have been created with max_grad_norm > 0."""

    def __init__(self, shard, group=None):
        import torch
        self.shard, self.group = shard, group
        # two exchange buffers, alternated by step parity: step k+1's sums never overwrite the array
        # step k's coefficient kernel may still be reading
        self.local = [torch.zeros(1, dtype=torch.float64, device=shard.device) for _ in range(2)]
        self.gathered = [None, None]

    def step_and_snapshot(self, grads, step: int, stream=None, hyper=None):
        import torch
        st = stream or torch.cuda.current_stream(self.shard.device)
        k = step & 1
        with torch.cuda.stream(st):
            B.phx_grad_sumsq_async(self.shard.h, grads, self.local[k], st)
            self.gathered[k] = gather_partials(self.local[k], self.group)   # NCCL, enqueued on `st`
            B.phx_set_clip_partials(self.shard.h, self.gathered[k], self.gathered[k].numel())
            self.shard.step_and_snapshot(grads, step, stream=st, hyper=hyper)


def step_group_in_process(shards: Sequence, grads_by_rank: Sequence, step: int, partials=None, stream=None):
    """D logical ranks on ONE device (tests / 1-GPU stand-in): every rank's sum goes straight into slot r
    of one device array (that is the all-gather), then every rank steps with the same D partials."""
    import torch
    dev = shards[0].device
    st = stream or torch.cuda.current_stream(dev)
    D = len(shards)
    if partials is None:
        partials = torch.zeros(D, dtype=torch.float64, device=dev)
    for r, (s, g) in enumerate(zip(shards, grads_by_rank)):
        B.phx_grad_sumsq_async(s.h, g, partials.data_ptr() + 8 * r, st)
    for s, g in zip(shards, grads_by_rank):
        B.phx_set_clip_partials(s.h, partials, D)
        s.step_and_snapshot(g, step, stream=st)
    return partials
