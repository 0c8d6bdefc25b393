"""Device/pinned memory plumbing for one shard: torch allocates, libphx computes.

`Shard` owns the torch tensors the C library is bound to (live p/m/v/bf16 copy, the device
staging ring, the pinned host replica) and forwards the hot-path calls to `binding`.  It holds no
arithmetic and no fallback.
"""
from __future__ import annotations

from typing import Optional

import torch

from . import binding as B
from .workloads import Hyper, Workload


class Shard:
    def __init__(self, wl: Workload, *, device="cuda:0", staging_depth=2, sync_mode=B.PHX_SYNC_STRICT,
                 chunk_bytes=0, snapshot=True, restore_mode=B.PHX_RESTORE_COPY_ENGINE,
                 max_grad_norm: Optional[float] = None, replica: Optional[torch.Tensor] = None,
                 snapshot_source=B.PHX_SNAPSHOT_STAGED, p16: Optional[torch.Tensor] = None,
                 payload=B.PHX_PAYLOAD_OPTIMIZER, W: Optional[torch.Tensor] = None):
        self.wl = wl
        self.device = torch.device(device)
        self.hyper: Hyper = wl.hyper
        mgn = wl.hyper.max_grad_norm if max_grad_norm is None else max_grad_norm
        self.h = B.phx_shard_create(
            wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank), pp=(wl.pp_size, wl.pp_rank),
            staging_depth=staging_depth, sync_mode=sync_mode, chunk_bytes=chunk_bytes,
            snapshot_disabled=not snapshot, restore_mode=restore_mode, max_grad_norm=mgn,
            snapshot_source=snapshot_source, flags=wl.flags(),
            precision=B.PHX_PRECISION_FP32 if wl.precision == "fp32" else B.PHX_PRECISION_BF16_GRADS,
            payload=payload)
        self.full = payload == B.PHX_PAYLOAD_FULL_RANK_STATE
        self.fp32 = wl.precision == "fp32"
        self.info = B.phx_shard_info(self.h)
        self.n, self.n_padded = self.info.n, self.info.n_padded
        self.segments = [(tid, off_s, ln) for tid, _, off_s, ln in B.phx_shard_segments(self.h)]
        N = self.n_padded
        with torch.cuda.device(self.device):
            self.p = torch.zeros(N, dtype=torch.float32, device=self.device)
            self.m = torch.zeros(N, dtype=torch.float32, device=self.device)
            self.v = torch.zeros(N, dtype=torch.float32, device=self.device)
            # no bf16 model-param copy in the all-FP32 precision
            # (p16 may be handed in: the rank's range inside its model-parameter buffer W)
            # §8(f4): W is the rank's model-parameter buffer (dp_size * N model-dtype elements); in the bf16
            # precision the bf16 copy is the rank's own range inside it
            self.W = W
            if self.full and W is None:
                self.W = torch.zeros(wl.dp_size * N, dtype=torch.float32 if self.fp32 else torch.bfloat16,
                                     device=self.device)
            if self.W is not None and not self.fp32 and p16 is None:
                p16 = self.W[wl.dp_rank * N:(wl.dp_rank + 1) * N]
            if p16 is not None:
                assert not self.fp32 and p16.dtype == torch.bfloat16 and p16.numel() == N and p16.is_contiguous()
                self.p16 = p16
            else:
                self.p16 = None if self.fp32 else torch.zeros(N, dtype=torch.bfloat16, device=self.device)
            self.staging = None
            self.replica = None
            if snapshot:
                if self.info.staging_depth > 0:     # PHX_SNAPSHOT_DIRECT needs no staging ring
                    self.staging = torch.zeros(self.info.staging_depth * self.info.slot_stride,
                                               dtype=torch.uint8, device=self.device)
                if replica is None:
                    replica = torch.zeros(2 * self.info.host_slot_stride, dtype=torch.uint8).pin_memory()
                assert replica.is_pinned() and replica.numel() >= 2 * self.info.host_slot_stride
                self.replica = replica
            B.phx_shard_bind(self.h, self.p, self.m, self.v, self.p16, self.staging, self.replica)
            if self.W is not None:
                B.phx_shard_bind_params(self.h, self.W)

    # -- thin forwards -----------------------------------------------------------------
    def set_state(self, step: int = 0, stream=None):
        B.phx_shard_set_state(self.h, step, stream or torch.cuda.current_stream(self.device))

    def step_and_snapshot(self, grads: torch.Tensor, step: int, stream=None, hyper: Optional[Hyper] = None):
        hp = hyper or self.hyper
        assert grads.dtype == (torch.float32 if self.fp32 else torch.bfloat16)
        assert grads.numel() == self.n_padded and grads.is_cuda
        B.phx_step_and_snapshot(self.h, grads, hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, step,
                                stream or torch.cuda.current_stream(self.device))

    def flush_async(self, side_stream):
        B.phx_snapshot_flush_async(self.h, side_stream)

    def wait(self, step: int):
        B.phx_snapshot_wait(self.h, step)

    def restore(self, stream=None) -> int:
        return B.phx_restore(self.h, stream or torch.cuda.current_stream(self.device))

    def restore_async(self, side_stream) -> int:
        """a6 in two phases (include/phx.h): parameters first, moments behind the recomputed forward/backward."""
        return B.phx_restore_async(self.h, side_stream)

    def restore_wait_params(self, stream=None):
        B.phx_restore_wait_params(self.h, stream or torch.cuda.current_stream(self.device))

    def staging_slot(self, step: int) -> torch.Tensor:
        k = step % self.info.staging_depth
        return self.staging[k * self.info.slot_stride: k * self.info.slot_stride + self.info.snapshot_bytes]

    def replica_slot(self, step: int) -> torch.Tensor:
        k = step % 2
        return self.replica[k * self.info.host_slot_stride: k * self.info.host_slot_stride + self.info.host_snapshot_bytes]

    # -- the graph-capturable form (include/phx.h "graph") --------------------------------
    def graph_begin(self, stream=None, hyper: Optional[Hyper] = None):
        hp = hyper or self.hyper
        B.phx_graph_begin(self.h, hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd,
                          stream or torch.cuda.current_stream(self.device))

    def graph_set_hyper(self, hyper: Hyper, stream=None):
        B.phx_graph_set_hyper(self.h, hyper.lr, hyper.beta1, hyper.beta2, hyper.eps, hyper.wd,
                              stream or torch.cuda.current_stream(self.device))

    def graph_step(self, grads: torch.Tensor, stream=None):
        assert grads.numel() == self.n_padded and grads.is_cuda
        B.phx_graph_step_and_snapshot(self.h, grads, stream or torch.cuda.current_stream(self.device))

    def graph_flush(self, side_stream):
        B.phx_graph_flush_async(self.h, side_stream)

    def graph_end(self) -> int:
        return B.phx_graph_end(self.h)

    # -- SURVEY 8(f4) second half: the gradient producer's epilogue -------------------------
    def grads_finalize(self, main_grads_fp32: torch.Tensor, scale: float, grads_bf16_out: torch.Tensor,
                       sumsq_out: torch.Tensor, stream=None):
        assert main_grads_fp32.dtype == torch.float32 and grads_bf16_out.dtype == torch.bfloat16
        assert main_grads_fp32.numel() == self.n_padded == grads_bf16_out.numel()
        assert sumsq_out.dtype == torch.float64 and sumsq_out.is_cuda
        B.phx_grads_finalize_async(self.h, main_grads_fp32, scale, grads_bf16_out, sumsq_out,
                                   stream or torch.cuda.current_stream(self.device))

    def params_ready(self, stream=None):
        B.phx_params_ready(self.h, stream or torch.cuda.current_stream(self.device))

    def params_guard(self, stream=None):
        B.phx_params_guard(self.h, stream or torch.cuda.current_stream(self.device))

    def drop_live(self):
        """'Drop the live shard' (BASELINE.json:configs[3]): zero p, m, v, bf16 copy and scribble
        over the device staging ring — restore must not depend on anything device-resident."""
        for t in (self.p, self.m, self.v, self.p16, self.W):
            if t is not None:
                t.zero_()
        if self.staging is not None:
            self.staging.fill_(0xA5)

    def close(self):
        if self.h:
            B.phx_shard_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
