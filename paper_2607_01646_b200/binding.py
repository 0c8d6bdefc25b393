"""Thin ctypes binding of libphx.so — same names as include/phx.h, argument marshalling only.

Every step of the hot path runs inside the library's kernels / copy engines; nothing here
computes.  There is no CPU fallback: if libphx.so is missing this module raises on first use
(build it with `python -m paper_2607_01646_b200.build`), and every compute entry point needs a
compute-capability-10.x GPU (PHX_ERR_UNSUPPORTED_DEVICE otherwise).

PyTorch is used by callers for device memory and streams only; pointers cross this boundary as
plain integers (`tensor.data_ptr()`, `stream.cuda_stream`).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence, Tuple

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libphx.so")

PHX_OK = 0
PHX_ERR_INVALID_ARG = -1
PHX_ERR_ALIGNMENT = -2
PHX_ERR_NOT_BOUND = -3
PHX_ERR_STEP_ORDER = -4
PHX_ERR_NO_FLUSH_PENDING = -5
PHX_ERR_NO_COMMITTED_SNAPSHOT = -6
PHX_ERR_LAYOUT_MISMATCH = -7
PHX_ERR_CORRUPT_SLOT = -8
PHX_ERR_CUDA = -9
PHX_ERR_UNSUPPORTED_DEVICE = -10
PHX_ERR_SNAPSHOT_DISABLED = -11
PHX_ERR_NOMEM = -12
PHX_ERR_PARAMS_NOT_READY = -13
PHX_ERR_GRAPH_MODE = -14
PHX_ERR_TOO_LARGE = -15
PHX_ERR_WRONG_DEVICE = -16
PHX_NO_ALLOC_MAX_ELEMS = 1 << 30

PHX_SYNC_STRICT, PHX_SYNC_RELAXED = 0, 1
PHX_RESTORE_COPY_ENGINE, PHX_RESTORE_BULK_KERNEL = 0, 1
PHX_SNAPSHOT_STAGED, PHX_SNAPSHOT_DIRECT = 0, 1
PHX_PRECISION_BF16_GRADS, PHX_PRECISION_FP32 = 0, 1
PHX_PAYLOAD_OPTIMIZER, PHX_PAYLOAD_FULL_RANK_STATE = 0, 1
PHX_TENSOR_NO_DECAY = 1


class phx_tensor_desc_t(C.Structure):
    _fields_ = [("numel", C.c_uint64), ("tensor_id", C.c_uint32), ("flags", C.c_uint32)]


class phx_config_t(C.Structure):
    _fields_ = [("tp_size", C.c_uint32), ("tp_rank", C.c_uint32), ("pp_size", C.c_uint32),
                ("pp_rank", C.c_uint32), ("staging_depth", C.c_uint32), ("sync_mode", C.c_uint32),
                ("chunk_bytes", C.c_uint64), ("snapshot_disabled", C.c_uint32),
                ("restore_mode", C.c_uint32), ("max_grad_norm", C.c_float),
                ("snapshot_source", C.c_uint32), ("precision", C.c_uint32), ("payload", C.c_uint32),
                ("reserved", C.c_uint32 * 2)]


class phx_shard_info_t(C.Structure):
    _fields_ = [("n", C.c_uint64), ("n_padded", C.c_uint64), ("total_numel", C.c_uint64),
                ("shard_begin", C.c_uint64), ("layout_hash", C.c_uint64),
                ("snapshot_bytes", C.c_uint64), ("slot_stride", C.c_uint64),
                ("n_segments", C.c_uint32), ("staging_depth", C.c_uint32),
                ("dp_size", C.c_uint32), ("dp_rank", C.c_uint32),
                ("host_snapshot_bytes", C.c_uint64), ("host_slot_stride", C.c_uint64), ("param_bytes", C.c_uint64)]


class phx_snapshot_header_t(C.Structure):
    _fields_ = [("magic", C.c_uint8 * 8), ("version", C.c_uint32), ("header_bytes", C.c_uint32),
                ("seq_begin", C.c_uint64), ("step", C.c_uint64), ("n", C.c_uint64), ("n_padded", C.c_uint64),
                ("total_numel", C.c_uint64), ("shard_begin", C.c_uint64), ("layout_hash", C.c_uint64),
                ("dp_size", C.c_uint32), ("dp_rank", C.c_uint32), ("tp_size", C.c_uint32), ("tp_rank", C.c_uint32),
                ("pp_size", C.c_uint32), ("pp_rank", C.c_uint32), ("chunk_bytes", C.c_uint64),
                ("user_len", C.c_uint32), ("payload", C.c_uint32), ("user", C.c_uint8 * 128),
                ("header_hash", C.c_uint64), ("seq_end", C.c_uint64)]


PHX_PUBLISH_FUSED, PHX_PUBLISH_COPY_ENGINE = 0, 1
PHX_MAX_PARAM_PEERS = 15
PHX_MAX_PEERS = 4
PHX_IPC_HANDLE_BYTES = 64


class PhxError(RuntimeError):
    def __init__(self, code: int, where: str, cuda: int = 0):
        self.code, self.cuda = code, cuda
        msg = lib().phx_strerror(code).decode()
        super().__init__(f"{where}: {msg} ({code})" + (f", cudaError {cuda}" if cuda else ""))


_lib = None

# name -> (restype, argtypes); the CPU test tier checks that libphx.so exports every one of them
PROTOTYPES = {
    "phx_version": (C.c_uint32, []),
    "phx_strerror": (C.c_char_p, [C.c_int]),
    "phx_last_cuda_error": (C.c_int, [C.c_void_p]),
    "phx_shard_create": (C.c_int, [C.POINTER(phx_tensor_desc_t), C.c_size_t, C.c_uint32, C.c_uint32,
                                   C.POINTER(phx_config_t), C.POINTER(C.c_void_p)]),
    "phx_shard_destroy": (C.c_int, [C.c_void_p]),
    "phx_shard_info": (C.c_int, [C.c_void_p, C.POINTER(phx_shard_info_t)]),
    "phx_shard_segments": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64),
                                     C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.c_uint32]),
    "phx_shard_bind": (C.c_int, [C.c_void_p] * 7),
    "phx_shard_set_state": (C.c_int, [C.c_void_p, C.c_uint64, C.c_void_p]),
    "phx_set_user_metadata": (C.c_int, [C.c_void_p, C.c_char_p, C.c_uint32]),
    "phx_step_and_snapshot": (C.c_int, [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float,
                                        C.c_float, C.c_float, C.c_uint64, C.c_void_p]),
    "phx_snapshot_flush_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_snapshot_wait": (C.c_int, [C.c_void_p, C.c_uint64]),
    "phx_snapshot_query": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_int)]),
    "phx_fault_inject_torn_flush": (C.c_int, [C.c_void_p, C.c_int64]),
    "phx_restore": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_restore_async": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_restore_wait_params": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_restored_user_metadata": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(C.c_uint32)]),
    "phx_last_step": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_last_clip": (C.c_int, [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_double)]),
    "phx_grad_sumsq_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "phx_grad_sumsq_no_alloc": (C.c_int, [C.c_void_p, C.c_int, C.c_uint64, C.c_void_p, C.c_void_p,
                                          C.POINTER(C.c_int)]),
    "phx_set_clip_partials": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint32]),
    "phx_kernel_launches": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_dropped_snapshots": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
    "phx_derived_scalars_host": (C.c_int, [C.c_float, C.c_float, C.c_float, C.c_float, C.c_uint64,
                                           C.POINTER(C.c_float)]),
    "phx_derived_scalars_device": (C.c_int, [C.c_float, C.c_float, C.c_float, C.c_float, C.POINTER(C.c_uint64),
                                             C.c_uint32, C.POINTER(C.c_float)]),
    "phx_grads_finalize_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]),
    "phx_graph_begin": (C.c_int, [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_float, C.c_float, C.c_void_p]),
    "phx_graph_set_hyper": (C.c_int, [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_float, C.c_float, C.c_void_p]),
    "phx_graph_set_user_metadata": (C.c_int, [C.c_void_p, C.c_char_p, C.c_uint32, C.c_void_p]),
    "phx_graph_step_and_snapshot": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "phx_graph_flush_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_graph_flush_peers_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_graph_end": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_ring_peer": (C.c_int, [C.c_uint32, C.c_uint32, C.c_int32, C.POINTER(C.c_uint32)]),
    "phx_ring_peers_topology_aware": (C.c_int, [C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32),
                                                C.POINTER(C.c_uint32)]),
    "phx_peer_buffer_alloc": (C.c_int, [C.c_uint64, C.POINTER(C.c_void_p)]),
    "phx_peer_buffer_free": (C.c_int, [C.c_void_p]),
    "phx_ipc_export": (C.c_int, [C.c_void_p, C.c_char_p]),
    "phx_ipc_open": (C.c_int, [C.c_char_p, C.POINTER(C.c_void_p)]),
    "phx_ipc_close": (C.c_int, [C.c_void_p]),
    "phx_shard_bind_peers": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.c_uint32]),
    "phx_snapshot_flush_peers_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_snapshot_wait_peers": (C.c_int, [C.c_void_p, C.c_uint64]),
    "phx_fault_inject_torn_peer_flush": (C.c_int, [C.c_void_p, C.c_uint32, C.c_int64]),
    "phx_replica_inspect": (C.c_int, [C.c_void_p, C.c_uint64, C.POINTER(phx_snapshot_header_t), C.POINTER(C.c_int)]),
    "phx_restore_from": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]),
    "phx_shard_bind_param_peers": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p), C.c_uint32, C.c_uint32]),
    "phx_publish_params_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_params_restore_from": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "phx_shard_bind_params": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_params_ready": (C.c_int, [C.c_void_p, C.c_void_p]),
    "phx_params_guard": (C.c_int, [C.c_void_p, C.c_void_p]),
}


def lib() -> C.CDLL:
    """Load libphx.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2607_01646_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in PROTOTYPES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _ck(rc: int, where: str, handle=None):
    if rc != PHX_OK:
        cuda = lib().phx_last_cuda_error(handle) if (handle and rc == PHX_ERR_CUDA) else 0
        raise PhxError(rc, where, cuda)


def _ptr(x) -> int:
    """tensor -> data_ptr(), stream -> cuda_stream, int/None pass through."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "cuda_stream"):
        return x.cuda_stream
    raise TypeError(type(x))


# ---- the calls of include/phx.h, same names -------------------------------------------------


def phx_shard_create(layout: Sequence[Tuple[int, int]], dp_size: int, dp_rank: int, *, tp=(1, 0),
                     pp=(1, 0), staging_depth=0, sync_mode=PHX_SYNC_STRICT, chunk_bytes=0,
                     snapshot_disabled=False, restore_mode=PHX_RESTORE_COPY_ENGINE,
                     max_grad_norm=0.0, snapshot_source=PHX_SNAPSHOT_STAGED,
                     flags: Optional[Sequence[int]] = None, precision=PHX_PRECISION_BF16_GRADS,
                     payload=PHX_PAYLOAD_OPTIMIZER) -> int:
    """layout = [(numel, tensor_id)] in flattening order.  Returns the opaque handle."""
    n = len(layout)
    arr = (phx_tensor_desc_t * max(n, 1))()
    for i, (numel, tid) in enumerate(layout):
        arr[i].numel, arr[i].tensor_id = int(numel), int(tid)
        arr[i].flags = int(flags[i]) if flags is not None else 0
    cfg = phx_config_t(tp_size=tp[0], tp_rank=tp[1], pp_size=pp[0], pp_rank=pp[1],
                       staging_depth=staging_depth, sync_mode=sync_mode, chunk_bytes=chunk_bytes,
                       snapshot_disabled=1 if snapshot_disabled else 0, restore_mode=restore_mode,
                       max_grad_norm=max_grad_norm, snapshot_source=snapshot_source, precision=precision,
                       payload=payload)
    h = C.c_void_p()
    _ck(lib().phx_shard_create(arr, n, dp_size, dp_rank, C.byref(cfg), C.byref(h)), "phx_shard_create")
    return h.value


def phx_shard_destroy(h: int) -> None:
    _ck(lib().phx_shard_destroy(h), "phx_shard_destroy")


def phx_shard_info(h: int) -> phx_shard_info_t:
    info = phx_shard_info_t()
    _ck(lib().phx_shard_info(h, C.byref(info)), "phx_shard_info")
    return info


def phx_shard_segments(h: int) -> List[Tuple[int, int, int, int]]:
    """[(tensor_id, off_in_tensor, off_in_shard, len)]"""
    k = phx_shard_info(h).n_segments
    tid = (C.c_uint32 * max(k, 1))()
    a, b, c = ((C.c_uint64 * max(k, 1))() for _ in range(3))
    _ck(lib().phx_shard_segments(h, tid, a, b, c, k), "phx_shard_segments")
    return [(tid[i], a[i], b[i], c[i]) for i in range(k)]


def phx_shard_bind(h: int, d_p, d_m, d_v, d_p_bf16, d_staging, h_replica) -> None:
    _ck(lib().phx_shard_bind(h, _ptr(d_p), _ptr(d_m), _ptr(d_v), _ptr(d_p_bf16), _ptr(d_staging),
                             _ptr(h_replica)), "phx_shard_bind", h)


def phx_shard_set_state(h: int, step: int, stream=None) -> None:
    _ck(lib().phx_shard_set_state(h, step, _ptr(stream)), "phx_shard_set_state", h)


def phx_set_user_metadata(h: int, blob: bytes) -> None:
    _ck(lib().phx_set_user_metadata(h, blob, len(blob)), "phx_set_user_metadata", h)


def phx_step_and_snapshot(h: int, d_grads, lr: float, beta1: float, beta2: float, eps: float,
                          wd: float, step: int, stream=None) -> None:
    _ck(lib().phx_step_and_snapshot(h, _ptr(d_grads), lr, beta1, beta2, eps, wd, step,
                                    _ptr(stream)), "phx_step_and_snapshot", h)


def phx_snapshot_flush_async(h: int, side_stream=None) -> None:
    _ck(lib().phx_snapshot_flush_async(h, _ptr(side_stream)), "phx_snapshot_flush_async", h)


def phx_snapshot_wait(h: int, step: int) -> None:
    _ck(lib().phx_snapshot_wait(h, step), "phx_snapshot_wait", h)


def phx_snapshot_query(h: int) -> Optional[Tuple[int, int]]:
    """(newest committed step, host slot) or None."""
    st, slot = C.c_uint64(), C.c_int()
    rc = lib().phx_snapshot_query(h, C.byref(st), C.byref(slot))
    if rc == PHX_ERR_NO_COMMITTED_SNAPSHOT:
        return None
    _ck(rc, "phx_snapshot_query", h)
    return st.value, slot.value


def phx_fault_inject_torn_flush(h: int, payload_chunks: int) -> None:
    _ck(lib().phx_fault_inject_torn_flush(h, payload_chunks), "phx_fault_inject_torn_flush", h)


def phx_restore(h: int, stream=None) -> int:
    st = C.c_uint64()
    _ck(lib().phx_restore(h, _ptr(stream), C.byref(st)), "phx_restore", h)
    return st.value


def phx_restore_async(h: int, side_stream=None) -> int:
    st = C.c_uint64()
    _ck(lib().phx_restore_async(h, _ptr(side_stream), C.byref(st)), "phx_restore_async", h)
    return st.value


def phx_restore_wait_params(h: int, stream=None) -> None:
    _ck(lib().phx_restore_wait_params(h, _ptr(stream)), "phx_restore_wait_params", h)


def phx_restored_user_metadata(h: int) -> bytes:
    buf = C.create_string_buffer(128)
    n = C.c_uint32()
    _ck(lib().phx_restored_user_metadata(h, buf, 128, C.byref(n)), "phx_restored_user_metadata", h)
    return buf.raw[:n.value]


def phx_last_step(h: int) -> int:
    st = C.c_uint64()
    _ck(lib().phx_last_step(h, C.byref(st)), "phx_last_step", h)
    return st.value


def phx_last_clip(h: int) -> Tuple[float, float]:
    c, q = C.c_float(), C.c_double()
    _ck(lib().phx_last_clip(h, C.byref(c), C.byref(q)), "phx_last_clip", h)
    return c.value, q.value


def phx_grad_sumsq_async(h: int, d_grads, d_out, stream=None) -> None:
    """this rank's sum of squared gradients into a caller-owned device double."""
    _ck(lib().phx_grad_sumsq_async(h, _ptr(d_grads), _ptr(d_out), _ptr(stream)), "phx_grad_sumsq_async", h)


def phx_grad_sumsq_no_alloc(d_grads, grads_fp32: bool, n_elems: int, d_out, stream=None) -> None:
    """Sum of squared gradients into a caller-owned device double, for callers that must not allocate device
    memory (no handle, no cudaMalloc: the reduction scratch is a 512 KiB array built into libphx.so).  Same bits as
    phx_grad_sumsq_async.  n_elems <= PHX_NO_ALLOC_MAX_ELEMS (PHX_ERR_TOO_LARGE beyond).  One scratch per GPU: do not
    let two calls overlap on the device; make the first call on a device before any stream capture (phx.h)."""
    err = C.c_int(0)
    rc = lib().phx_grad_sumsq_no_alloc(_ptr(d_grads), 1 if grads_fp32 else 0, int(n_elems), _ptr(d_out), _ptr(stream),
                                       C.byref(err))
    if rc != PHX_OK:
        raise PhxError(rc, "phx_grad_sumsq_no_alloc", err.value)


def phx_set_clip_partials(h: int, d_partials, count: int) -> None:
    """one-shot per-rank sums (device doubles, rank order) the next step clips by."""
    _ck(lib().phx_set_clip_partials(h, _ptr(d_partials) or None, count), "phx_set_clip_partials", h)


def phx_kernel_launches(h: int) -> int:
    n = C.c_uint64()
    _ck(lib().phx_kernel_launches(h, C.byref(n)), "phx_kernel_launches", h)
    return n.value


def phx_dropped_snapshots(h: int) -> Tuple[int, int]:
    """(snapshots superseded before a host flush, before a peer flush)."""
    a, b = C.c_uint64(), C.c_uint64()
    _ck(lib().phx_dropped_snapshots(h, C.byref(a), C.byref(b)), "phx_dropped_snapshots", h)
    return a.value, b.value


def phx_derived_scalars_host(lr: float, beta1: float, beta2: float, wd: float, step: int) -> List[float]:
    """[decay, omb1, omb2, ss, sbc2] as the library's HOST code derives them (no GPU needed)."""
    out = (C.c_float * 5)()
    _ck(lib().phx_derived_scalars_host(lr, beta1, beta2, wd, step, out), "phx_derived_scalars_host")
    return list(out)


def phx_derived_scalars_device(lr: float, beta1: float, beta2: float, wd: float, steps: Sequence[int]) -> List[List[float]]:
    """Per step index, [decay, omb1, omb2, ss, sbc2] as the graph form's DEVICE prologue derives them."""
    n = len(steps)
    arr = (C.c_uint64 * max(n, 1))(*[int(t) for t in steps])
    out = (C.c_float * (5 * max(n, 1)))()
    _ck(lib().phx_derived_scalars_device(lr, beta1, beta2, wd, arr, n, out), "phx_derived_scalars_device")
    return [list(out[5 * i:5 * i + 5]) for i in range(n)]


def phx_grads_finalize_async(h: int, d_main_grads_fp32, scale: float, d_grads_bf16_out, d_sumsq_out, stream=None) -> None:
    """SURVEY 8(f4) second half: g16 = RNE_bf16(g32 * scale) and the fp64 sum of squares of the rounded values."""
    _ck(lib().phx_grads_finalize_async(h, _ptr(d_main_grads_fp32), scale, _ptr(d_grads_bf16_out), _ptr(d_sumsq_out),
                                       _ptr(stream)), "phx_grads_finalize_async", h)


# ---- the graph-capturable form -------------------------------------------------------------------


def phx_graph_begin(h: int, lr: float, beta1: float, beta2: float, eps: float, wd: float, stream=None) -> None:
    _ck(lib().phx_graph_begin(h, lr, beta1, beta2, eps, wd, _ptr(stream)), "phx_graph_begin", h)


def phx_graph_set_hyper(h: int, lr: float, beta1: float, beta2: float, eps: float, wd: float, stream=None) -> None:
    _ck(lib().phx_graph_set_hyper(h, lr, beta1, beta2, eps, wd, _ptr(stream)), "phx_graph_set_hyper", h)


def phx_graph_set_user_metadata(h: int, blob: bytes, stream=None) -> None:
    _ck(lib().phx_graph_set_user_metadata(h, blob, len(blob), _ptr(stream)), "phx_graph_set_user_metadata", h)


def phx_graph_step_and_snapshot(h: int, d_grads, stream=None) -> None:
    _ck(lib().phx_graph_step_and_snapshot(h, _ptr(d_grads), _ptr(stream)), "phx_graph_step_and_snapshot", h)


def phx_graph_flush_async(h: int, side_stream=None) -> None:
    _ck(lib().phx_graph_flush_async(h, _ptr(side_stream)), "phx_graph_flush_async", h)


def phx_graph_flush_peers_async(h: int, peer_stream=None) -> None:
    _ck(lib().phx_graph_flush_peers_async(h, _ptr(peer_stream)), "phx_graph_flush_peers_async", h)


def phx_graph_end(h: int) -> int:
    """Leaves the graph form; returns the device step counter (raises PHX_ERR_STEP_ORDER on a misaligned replay)."""
    st = C.c_uint64()
    _ck(lib().phx_graph_end(h, C.byref(st)), "phx_graph_end", h)
    return st.value


def phx_version() -> int:
    return lib().phx_version()


# ---- peer replication ------------------------------------------------------


def phx_ring_peers_topology_aware(dp_size: int, dp_rank: int, k: int, domains) -> list:
    dom = (C.c_uint32 * dp_size)(*[int(d) for d in domains])
    out = (C.c_uint32 * max(k, 1))()
    _ck(lib().phx_ring_peers_topology_aware(dp_size, dp_rank, k, dom, out), "phx_ring_peers_topology_aware")
    return [int(out[j]) for j in range(k)]


def phx_ring_peer(dp_size: int, dp_rank: int, j: int) -> int:
    out = C.c_uint32()
    _ck(lib().phx_ring_peer(dp_size, dp_rank, j, C.byref(out)), "phx_ring_peer")
    return out.value


def phx_peer_buffer_alloc(nbytes: int) -> int:
    p = C.c_void_p()
    _ck(lib().phx_peer_buffer_alloc(nbytes, C.byref(p)), "phx_peer_buffer_alloc")
    return p.value


def phx_peer_buffer_free(d_buf: int) -> None:
    _ck(lib().phx_peer_buffer_free(d_buf), "phx_peer_buffer_free")


def phx_ipc_export(d_buf: int) -> bytes:
    buf = C.create_string_buffer(PHX_IPC_HANDLE_BYTES)
    _ck(lib().phx_ipc_export(d_buf, buf), "phx_ipc_export")
    return buf.raw


def phx_ipc_open(handle: bytes) -> int:
    assert len(handle) == PHX_IPC_HANDLE_BYTES
    p = C.c_void_p()
    _ck(lib().phx_ipc_open(handle, C.byref(p)), "phx_ipc_open")
    return p.value


def phx_ipc_close(d_buf: int) -> None:
    _ck(lib().phx_ipc_close(d_buf), "phx_ipc_close")


def phx_shard_bind_peers(h: int, d_peer_replicas: Sequence) -> None:
    k = len(d_peer_replicas)
    arr = (C.c_void_p * max(k, 1))(*[_ptr(x) for x in d_peer_replicas])
    _ck(lib().phx_shard_bind_peers(h, arr, k), "phx_shard_bind_peers", h)


def phx_snapshot_flush_peers_async(h: int, peer_stream=None) -> None:
    _ck(lib().phx_snapshot_flush_peers_async(h, _ptr(peer_stream)), "phx_snapshot_flush_peers_async", h)


def phx_snapshot_wait_peers(h: int, step: int) -> None:
    _ck(lib().phx_snapshot_wait_peers(h, step), "phx_snapshot_wait_peers", h)


def phx_fault_inject_torn_peer_flush(h: int, peer_j: int, payload_chunks: int) -> None:
    _ck(lib().phx_fault_inject_torn_peer_flush(h, peer_j, payload_chunks), "phx_fault_inject_torn_peer_flush", h)


def phx_replica_inspect(replica, slot_stride: int):
    """[(header, valid)] for the two slots of a replica buffer (device, peer-mapped or pinned host)."""
    hdr = (phx_snapshot_header_t * 2)()
    valid = (C.c_int * 2)()
    _ck(lib().phx_replica_inspect(_ptr(replica), slot_stride, hdr, valid), "phx_replica_inspect")
    return [(hdr[i], bool(valid[i])) for i in range(2)]


def phx_restore_from(h: int, replica, stream=None) -> int:
    st = C.c_uint64()
    _ck(lib().phx_restore_from(h, _ptr(replica), _ptr(stream), C.byref(st)), "phx_restore_from", h)
    return st.value


# ---- model-parameter publication and reconstruction ---------------------------


def phx_shard_bind_param_peers(h: int, d_param_bufs: Sequence, mode: int = PHX_PUBLISH_FUSED) -> None:
    k = len(d_param_bufs)
    arr = (C.c_void_p * max(k, 1))(*[_ptr(x) for x in d_param_bufs])
    _ck(lib().phx_shard_bind_param_peers(h, arr, k, mode), "phx_shard_bind_param_peers", h)


def phx_publish_params_async(h: int, stream=None) -> None:
    _ck(lib().phx_publish_params_async(h, _ptr(stream)), "phx_publish_params_async", h)


def phx_params_restore_from(h: int, d_src_param_buf, d_dst_param_buf, stream=None) -> None:
    _ck(lib().phx_params_restore_from(h, _ptr(d_src_param_buf), _ptr(d_dst_param_buf), _ptr(stream)),
        "phx_params_restore_from", h)


# ---- full rank-state local snapshot ---------------------------------------------


def phx_shard_bind_params(h: int, d_W) -> None:
    _ck(lib().phx_shard_bind_params(h, _ptr(d_W)), "phx_shard_bind_params", h)


def phx_params_ready(h: int, stream=None) -> None:
    _ck(lib().phx_params_ready(h, _ptr(stream)), "phx_params_ready", h)


def phx_params_guard(h: int, stream=None) -> None:
    _ck(lib().phx_params_guard(h, _ptr(stream)), "phx_params_guard", h)
