"""phx_grad_sumsq_no_alloc: the gradient sum of squares for callers that must not allocate device memory.

Some users of libphx.so cannot call cudaMalloc where they need a rank's gradient norm: the training framework's
allocator already owns the whole GPU (an allocation beside it fails or starves the framework), the call would sit
on the iteration's critical path (cudaMalloc/cudaFree synchronise the device and would stall the snapshot flush
this library overlaps with compute), or it runs in the fault-handling path where nothing should depend on memory
being obtainable.  The handle-based phx_grad_sumsq_async is closed to them, because phx_shard_bind allocates its
reduction scratch.  The no-alloc entry point keeps that scratch in a 512 KiB array built into the library
(PHX_NO_ALLOC_MAX_ELEMS = 2^30 elements at most) and runs the SAME kernels in the same launch shape, so its result
must have the same bits as the existing call on the same gradients.

What is checked: (1) bit equality with phx_grad_sumsq_async, and agreement with the oracle's exactly rounded sum
within the 16-ulp reassociation bound test_gpu_global_clip.py uses, on TWO calls in a row on the one shared scratch —
the second one smaller and on different gradients, so entries the first call left behind sit right after the range
the second call uses; (2) the largest size it accepts, against a closed form; (3) the documented errors.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure, and a failure of
this add-on must not hide a parity failure of the hot path.  Each test builds everything it needs, so the file
passes alone in a fresh process as well as after the rest of the suite (whatever that left in the scratch).
"""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import build as phx_build
from paper_2607_01646_b200 import workloads as W
from paper_2607_01646_b200.shard import Shard

from gpu_util import DEV, grad_record


@pytest.fixture(scope="module", autouse=True)
def built():
    phx_build.build()


def _both_paths(numels, precision, step, seed):
    """(no-alloc result, handle-based result, oracle sum) for one seeded gradient shard."""
    wl = W.tiny_workload(numels, dp_size=1, dp_rank=0, precision=precision, grad_kind="heavy_tail")
    s = Shard(wl, device=DEV, chunk_bytes=1 << 16)          # the EXISTING path needs a bound shard (it allocates)
    gdt = torch.float32 if precision == "fp32" else torch.bfloat16
    g = W.gen_grads(wl, s.segments, s.n_padded, step, seed=seed, dtype=gdt)
    gd = g.to(DEV)
    out = torch.full((2,), -1.0, dtype=torch.float64, device=DEV)
    st = torch.cuda.current_stream()
    B.phx_grad_sumsq_no_alloc(gd, precision == "fp32", s.n_padded, out[0:1], st)
    B.phx_grad_sumsq_async(s.h, gd, out[1:2], st)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    return got[0], got[1], O.sumsq(grad_record(g))


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["bf16", "fp32"])
def test_two_calls_in_a_row_equal_the_existing_path(precision):
    # call 1: 41 reduction CTAs (16384 elements each) and a ragged tail; call 2: 3 CTAs + a tail of one 64-lane
    # pad unit, other gradients — partials 4..40 of call 1 are still in the scratch and must not leak into it
    for numels, step, seed in (([16384 * 37 + 777, 65536, 5], 1, 7), ([16384 * 3 + 1], 2, 8)):
        new, old, want = _both_paths(numels, precision, step, seed)
        assert np.float64(new).view(np.uint64) == np.float64(old).view(np.uint64), (numels, new, old)
        assert want > 0 and abs(new - want) <= 16 * np.spacing(want), (numels, new, want)


@pytest.mark.gpu
def test_largest_accepted_size_against_a_closed_form():
    # 2^30 gradients of 0.5 (2 GiB of bf16): every square is 2^-2 and every partial sum a power of two or a small
    # multiple of one, so the result is 2^28 exactly whatever the tree; then 1.0 in the last 8 lanes: + 8 * 0.75
    n = B.PHX_NO_ALLOC_MAX_ELEMS
    g = torch.full((n,), 0.5, dtype=torch.bfloat16, device=DEV)
    out = torch.zeros(1, dtype=torch.float64, device=DEV)
    B.phx_grad_sumsq_no_alloc(g, False, n, out, torch.cuda.current_stream())
    assert out.item() == float(1 << 28)
    g[-8:] = 1.0
    B.phx_grad_sumsq_no_alloc(g, False, n, out, torch.cuda.current_stream())
    assert out.item() == float(1 << 28) + 6.0
    # ... and a small call right after the largest one reads none of its 65536 partials
    B.phx_grad_sumsq_no_alloc(g[-128:], False, 128, out, torch.cuda.current_stream())   # 256-byte aligned slice
    assert out.item() == 120 * 0.25 + 8.0
    with pytest.raises(B.PhxError) as e:
        B.phx_grad_sumsq_no_alloc(g, False, n + 8, out, torch.cuda.current_stream())
    assert e.value.code == B.PHX_ERR_TOO_LARGE
    del g
    torch.cuda.empty_cache()


def test_argument_errors_need_no_gpu():
    """Every rejection happens before the first CUDA call, so this runs in the CPU tier too."""
    f = B.lib().phx_grad_sumsq_no_alloc
    err = C.c_int(123)
    ok_ptr, out_ptr = 0x10000, 0x20000                       # never dereferenced: the call must fail first
    assert f(None, 0, 64, out_ptr, None, C.byref(err)) == B.PHX_ERR_INVALID_ARG and err.value == 0
    assert f(ok_ptr, 0, 64, None, None, None) == B.PHX_ERR_INVALID_ARG
    assert f(ok_ptr, 0, 0, out_ptr, None, None) == B.PHX_ERR_INVALID_ARG
    assert f(ok_ptr, 0, 60, out_ptr, None, None) == B.PHX_ERR_INVALID_ARG      # not a multiple of 8
    assert f(ok_ptr, 2, 64, out_ptr, None, None) == B.PHX_ERR_INVALID_ARG      # grads_fp32 is 0 or 1
    assert f(ok_ptr, 0, B.PHX_NO_ALLOC_MAX_ELEMS + 8, out_ptr, None, None) == B.PHX_ERR_TOO_LARGE
    assert f(ok_ptr + 128, 0, 64, out_ptr, None, None) == B.PHX_ERR_ALIGNMENT  # gradients: 256-byte aligned
    assert f(ok_ptr, 1, 64, out_ptr + 4, None, None) == B.PHX_ERR_ALIGNMENT    # result: 8-byte aligned
    assert b"built-in scratch" in B.lib().phx_strerror(B.PHX_ERR_TOO_LARGE)
