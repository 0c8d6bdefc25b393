"""Memory-safety by guard regions (compute-sanitizer is closed on this GPU pool): every buffer the
library is bound to — live p, m, v, bf16 copy, gradients, staging ring, pinned host replica, a peer's received
buffer, a published parameter buffer, the producer epilogue's input/output — sits inside a larger allocation with
4 KiB guard bands on both sides; after steps (with clip), flushes, both restore modes, the producer epilogue,
graph-form steps, a peer flush and a fused publication, every guard byte is unchanged."""
import numpy as np
import pytest
import torch

from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

from gpu_util import DEV

pytestmark = pytest.mark.gpu
G = 4096
PAT = 0xC3


class Guarded:
    def __init__(self, nbytes, device, pinned=False):
        self.raw = torch.empty(nbytes + 2 * G, dtype=torch.uint8, device=device)
        if pinned:
            self.raw = self.raw.pin_memory()
        self.raw.fill_(PAT)
        self.body = self.raw[G:G + nbytes]
        self.body.zero_()
        assert self.body.data_ptr() % 256 == 0

    def view(self, dtype):
        return self.body.view(dtype)

    def intact(self):
        return bool((self.raw[:G] == PAT).all()) and bool((self.raw[-G:] == PAT).all())


@pytest.mark.parametrize("numels", [[64], [2048 * 5 + 64 * 3, 77], [300_000, 12_345]])
@pytest.mark.parametrize("rmode", [B.PHX_RESTORE_COPY_ENGINE, B.PHX_RESTORE_BULK_KERNEL])
def test_no_byte_outside_the_bound_buffers_is_touched(numels, rmode):
    D, r = 2, 1
    h = B.phx_shard_create([(n, i) for i, n in enumerate(numels)], D, r, staging_depth=3, max_grad_norm=0.05,
                           chunk_bytes=64 << 10, restore_mode=rmode)
    info = B.phx_shard_info(h)
    N = info.n_padded
    bufs = {k: Guarded(4 * N, DEV) for k in ("p", "m", "v", "g32")}
    bufs["g"] = Guarded(2 * N, DEV)
    bufs["g2"] = Guarded(2 * N, DEV)
    bufs["W"] = Guarded(2 * D * N, DEV)                       # own parameter buffer: the bf16 copy is its range r
    bufs["Wpeer"] = Guarded(2 * D * N, DEV)                   # another rank's parameter buffer (fused publication)
    bufs["staging"] = Guarded(3 * info.slot_stride, DEV)
    bufs["recv"] = Guarded(2 * info.slot_stride, DEV)         # a ring successor's received buffer
    bufs["replica"] = Guarded(2 * info.slot_stride, "cpu", pinned=True)
    bufs["S"] = Guarded(256, DEV)
    p, m, v = (bufs[k].view(torch.float32) for k in ("p", "m", "v"))
    gen = torch.Generator(device=DEV).manual_seed(1)
    p[:info.n].normal_(0, 0.02, generator=gen)
    g32 = bufs["g32"].view(torch.float32)
    g32[:info.n].normal_(0, 1e-3, generator=gen)
    g = bufs["g"].view(torch.bfloat16)
    g.copy_(g32.to(torch.bfloat16))
    p16 = bufs["W"].view(torch.bfloat16)[r * N:(r + 1) * N]
    B.phx_shard_bind(h, p, m, v, p16, bufs["staging"].body, bufs["replica"].body)
    B.phx_shard_bind_peers(h, [bufs["recv"].body])
    B.phx_shard_bind_param_peers(h, [bufs["Wpeer"].body], B.PHX_PUBLISH_FUSED)
    cur, side, peer = torch.cuda.current_stream(), torch.cuda.Stream(device=DEV), torch.cuda.Stream(device=DEV)
    B.phx_shard_set_state(h, 0, cur)
    hp = (3e-4, 0.9, 0.95, 1e-8, 0.1)
    for t in (1, 2, 3, 4):
        B.phx_step_and_snapshot(h, g, *hp, t, cur)            # a1 + a3 (+ fused publication into Wpeer)
        B.phx_snapshot_flush_async(h, side)
        B.phx_snapshot_flush_peers_async(h, peer)
    B.phx_snapshot_wait(h, 4)
    B.phx_snapshot_wait_peers(h, 4)
    # the producer epilogue, then a step fed by its sum
    S = bufs["S"].view(torch.float64)
    B.phx_grads_finalize_async(h, g32, 0.5, bufs["g2"].view(torch.bfloat16), S, cur)
    B.phx_set_clip_partials(h, S, 1)
    B.phx_step_and_snapshot(h, bufs["g2"].view(torch.bfloat16), *hp, 5, cur)
    B.phx_snapshot_flush_async(h, side)
    # drop + restore from the host replica, then from the peer's received buffer
    torch.cuda.synchronize()
    for x in (p, m, v):
        x.zero_()
    assert B.phx_restore(h, cur) == 5
    assert B.phx_restore_async(h, side) == 5                  # two phases on the side stream: {p, bf16 copy} then {m, v}
    B.phx_restore_wait_params(h, cur)
    assert B.phx_restore_from(h, bufs["recv"].body, cur) == 4
    # graph-form steps (prologue writes the envelope into the staging slot) + flushes
    B.phx_graph_begin(h, *hp, cur)
    for t in (5, 6, 7):
        B.phx_graph_step_and_snapshot(h, g, cur)
        B.phx_graph_flush_async(h, side)
    assert B.phx_graph_end(h) == 7
    torch.cuda.synchronize()
    bad = [k for k, b in bufs.items() if not b.intact()]
    assert not bad, f"guard bands overwritten around: {bad}"
    # and the pad lanes inside the buffers stayed zero
    for x in (p, m, v):
        assert not x[info.n:].cpu().numpy().view(np.uint32).any()
    B.phx_shard_bind_param_peers(h, [])
    B.phx_shard_bind_peers(h, [])
    B.phx_shard_destroy(h)


def test_bind_rejects_pointers_that_are_not_device_memory_of_the_current_device():
    """SURVEY §8(b) "Ownership" / VERDICT r2 item 4: phx_shard_bind validates the KIND of every d_* pointer with
    cudaPointerGetAttributes.  A pinned host pointer (which the GPU could even reach) or plain pageable memory passed
    as d_p used to be accepted and fault — or silently train on host memory — at the first step."""
    h = B.phx_shard_create([(4096, 0)], 1, 0, chunk_bytes=64 << 10)
    info = B.phx_shard_info(h)
    N = info.n_padded
    dev = {k: torch.zeros(N, dtype=torch.float32, device=DEV) for k in ("p", "m", "v")}
    p16 = torch.zeros(N, dtype=torch.bfloat16, device=DEV)
    staging = torch.zeros(2 * info.slot_stride, dtype=torch.uint8, device=DEV)
    replica = torch.zeros(2 * info.host_slot_stride, dtype=torch.uint8).pin_memory()
    pinned = torch.zeros(N + 64, dtype=torch.float32).pin_memory()
    pageable = torch.zeros(N + 64, dtype=torch.float32)
    L = B.lib()

    def bind(p=None, m=None, v=None, b16=None, st=None):
        return L.phx_shard_bind(h, (p if p is not None else dev["p"]).data_ptr(), (m if m is not None else dev["m"]).data_ptr(),
                                (v if v is not None else dev["v"]).data_ptr(), (b16 if b16 is not None else p16).data_ptr(),
                                (st if st is not None else staging).data_ptr(), replica.data_ptr())

    def aligned(t):
        off = (-t.data_ptr() % 256) // t.element_size()
        return t[off:]

    assert bind(p=aligned(pinned)) == B.PHX_ERR_INVALID_ARG
    assert bind(m=aligned(pageable)) == B.PHX_ERR_INVALID_ARG
    assert bind(v=aligned(pinned)) == B.PHX_ERR_INVALID_ARG
    assert bind(st=aligned(pinned.view(torch.uint8))) == B.PHX_ERR_INVALID_ARG
    # a device pointer as the host replica is refused as before (not pinned, mapped host memory)
    assert L.phx_shard_bind(h, dev["p"].data_ptr(), dev["m"].data_ptr(), dev["v"].data_ptr(), p16.data_ptr(),
                            staging.data_ptr(), staging.data_ptr()) == B.PHX_ERR_INVALID_ARG
    assert bind() == B.PHX_OK                              # nothing above left the handle half-bound
    assert b"bound on" in L.phx_strerror(B.PHX_ERR_WRONG_DEVICE)
    B.phx_shard_destroy(h)
