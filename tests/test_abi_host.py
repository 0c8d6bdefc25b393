"""CPU tier for the CUDA side: libphx.so builds, loads without a GPU, exports every symbol
include/phx.h declares, and its host logic (a0 shard definition, config defaults, argument and
state checks) agrees with the oracle.  No compute entry point is called here.
"""
import ctypes as C
import os
import re
import struct

import pytest

from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import build as phx_build
from paper_2607_01646_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    phx_build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "phx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return re.findall(r"PHX_API\s+[\w\s\*]+?\b(phx_\w+)\s*\(", src)


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert len(names) >= 20 and len(set(names)) == len(names)
    L = C.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(B.PROTOTYPES), set(names) ^ set(B.PROTOTYPES)
    assert B.phx_version() == 0x00010000
    assert B.lib().phx_strerror(B.PHX_ERR_STEP_ORDER) == b"step is not last_step + 1"


def dynamic_symbols(path):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True, check=True).stdout
    return [ln.split()[-1] for ln in out.splitlines() if ln.strip()]


def test_library_exports_product_symbols_only():
    """nothing but the C ABI of include/phx.h is visible — no tuning knob, no diagnostic,
    no leaked C++ runtime template instantiation (linker version script csrc/phx.map)."""
    syms = dynamic_symbols(B.LIB_PATH)
    assert sorted(syms) == sorted(declared_functions()), set(syms) ^ set(declared_functions())
    assert "phx_set_kernel_variant" not in syms and "phx_hbm_probe_async" not in syms
    # the bench-only diagnostic lives in a library of its own
    from paper_2607_01646_b200 import probe
    assert sorted(dynamic_symbols(probe.LIB_PATH)) == ["phx_hbm_probe_async", "phx_hbm_probe_persistent_async"]


def test_host_derived_scalars_equal_the_oracle_bitwise():
    """the host code of libphx.so must round every binary64 operation like the oracle
    (-ffp-contract=off in build.py); compared for several (lr, wd, beta, t) incl. the Appendix A values."""
    import numpy as np
    cases = [(3e-4, 0.9, 0.95, 0.1), (1e-3, 0.9, 0.999, 0.01), (6e-4, 0.8, 0.98, 0.0), (1.0, 0.5, 0.25, 0.3),
             (2.5e-5, 0.95, 0.9999, 1e-4)]
    steps = [1, 2, 3, 10, 17, 100, 1000, 4097, 65535, 10**6, 2**33 + 5]
    for lr, b1, b2, wd in cases:
        for t in steps:
            got = np.array(B.phx_derived_scalars_host(lr, b1, b2, wd, t), np.float32).view(np.uint32)
            exp = O.scalars(lr, b1, b2, 1e-8, wd, t).view(np.uint32)
            assert np.array_equal(got, exp), (lr, b1, b2, wd, t)
    # SURVEY.md Appendix A bit patterns (lr 3e-4, betas (0.9, 0.95), wd 0.1)
    got = np.array(B.phx_derived_scalars_host(3e-4, 0.9, 0.95, 0.1, 1), np.float32).view(np.uint32)
    assert [hex(x) for x in got] == ["0x3f7ffe09", "0x3dccccd0", "0x3d4cccd0", "0x3b449ba3", "0x3e64f930"]
    assert B.lib().phx_derived_scalars_host(3e-4, 0.9, 0.95, 0.1, 0, (C.c_float * 5)()) == B.PHX_ERR_INVALID_ARG


def test_struct_sizes_match_the_header():
    assert C.sizeof(B.phx_tensor_desc_t) == 16
    assert C.sizeof(B.phx_config_t) == 64
    assert C.sizeof(B.phx_shard_info_t) == 96
    assert C.sizeof(B.phx_snapshot_header_t) == 256


@pytest.mark.parametrize("numels,dp", [([5], 1), ([100, 3, 64, 1], 3), ([63, 1, 64, 129], 2),
                                       ([1000, 24, 7], 4), ([1], 5), ([0, 10, 0], 2)])
def test_shard_definition_matches_oracle(numels, dp):
    layout = [(n, 7 * i + 1) for i, n in enumerate(numels)]
    for r in range(dp):
        for tp, pp in (((1, 0), (1, 0)), ((2, 1), (4, 3))):
            h = B.phx_shard_create(layout, dp, r, tp=tp, pp=pp)
            try:
                info = B.phx_shard_info(h)
                d = O.define_shard(layout, dp, r, tp, pp)
                assert (info.n, info.n_padded, info.total_numel, info.shard_begin) == \
                    (d["n"], d["n_padded"], d["total_numel"], d["shard_begin"])
                assert info.layout_hash == d["layout_hash"]
                assert info.snapshot_bytes == 256 + 12 * d["n_padded"]
                assert info.slot_stride % 256 == 0 and info.slot_stride >= info.snapshot_bytes
                assert B.phx_shard_segments(h) == d["segments"]
            finally:
                B.phx_shard_destroy(h)


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4a", "c4b", "c5"])
def test_config_shards(key):
    wl = W.CONFIGS[key]
    h = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank),
                           pp=(wl.pp_size, wl.pp_rank))
    info = B.phx_shard_info(h)
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank), (wl.pp_size, wl.pp_rank))
    assert info.n == wl.n_expected == info.n_padded and info.layout_hash == d["layout_hash"]
    assert B.phx_shard_segments(h) == d["segments"]
    assert info.staging_depth == 2 and (info.dp_size, info.dp_rank) == (wl.dp_size, wl.dp_rank)
    B.phx_shard_destroy(h)


def test_argument_and_state_errors_without_a_gpu():
    with pytest.raises(B.PhxError) as e:
        B.phx_shard_create([(10, 0)], 0, 0)
    assert e.value.code == B.PHX_ERR_INVALID_ARG
    for kw in (dict(dp_rank=2), dict(staging_depth=5), dict(tp=(2, 2)), dict(pp=(1, 1)), dict(sync_mode=2),
               dict(restore_mode=2), dict(max_grad_norm=float("nan")), dict(snapshot_source=2),
               dict(snapshot_source=B.PHX_SNAPSHOT_DIRECT, sync_mode=B.PHX_SYNC_RELAXED),
               dict(payload=2), dict(payload=B.PHX_PAYLOAD_FULL_RANK_STATE, snapshot_disabled=True)):
        args = dict(dp_size=2, dp_rank=0)
        args.update(kw)
        with pytest.raises(B.PhxError) as e:
            B.phx_shard_create([(10, 0)], **args)
        assert e.value.code == B.PHX_ERR_INVALID_ARG, kw
    h = B.phx_shard_create([(100, 0)], 1, 0)
    L = B.lib()
    # nothing bound yet
    assert L.phx_step_and_snapshot(h, 256, 1e-3, 0.9, 0.95, 1e-8, 0.0, 1, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_snapshot_flush_async(h, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_restore(h, None, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_shard_set_state(h, 0, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_step_and_snapshot(h, None, 1e-3, 0.9, 0.95, 1e-8, 0.0, 1, None) == B.PHX_ERR_INVALID_ARG
    # binding checks that need no device: null and misaligned pointers
    assert L.phx_shard_bind(h, None, 256, 256, 256, 256, 256) == B.PHX_ERR_INVALID_ARG
    assert L.phx_shard_bind(h, 256, 256, 256, 256, None, 256) == B.PHX_ERR_INVALID_ARG
    assert L.phx_shard_bind(h, 256, 256, 264, 256, 256, 256) == B.PHX_ERR_ALIGNMENT
    assert L.phx_set_user_metadata(h, b"x" * 129, 129) == B.PHX_ERR_INVALID_ARG
    assert L.phx_set_user_metadata(h, b"x" * 128, 128) == B.PHX_OK
    # the graph-capturable form and the producer epilogue need bound memory too
    assert L.phx_graph_begin(h, 1e-3, 0.9, 0.95, 1e-8, 0.0, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_graph_step_and_snapshot(h, 256, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_graph_end(h, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_grads_finalize_async(h, 256, 1.0, 512, 1024, None) == B.PHX_ERR_NOT_BOUND
    assert L.phx_grads_finalize_async(h, None, 1.0, 512, 1024, None) == B.PHX_ERR_INVALID_ARG
    assert B.phx_dropped_snapshots(h) == (0, 0)
    assert B.phx_last_step(h) == 0 and B.phx_kernel_launches(h) == 0
    B.phx_shard_destroy(h)
    assert L.phx_shard_destroy(None) == B.PHX_ERR_INVALID_ARG


def test_bind_without_a_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    h = B.phx_shard_create([(100, 0)], 1, 0)
    rc = B.lib().phx_shard_bind(h, 256, 256, 256, 256, 256, 256)
    assert rc in (B.PHX_ERR_CUDA, B.PHX_ERR_UNSUPPORTED_DEVICE)   # never a silent CPU path
    B.phx_shard_destroy(h)


@pytest.mark.parametrize("precision,eb", [(B.PHX_PRECISION_BF16_GRADS, 2), (B.PHX_PRECISION_FP32, 4)])
def test_full_rank_state_slot_sizes(precision, eb):
    # the local slot = optimizer-only snapshot + the model-parameter buffer W (oracle/rank_state.py)
    from oracle import rank_state as RS
    layout, D = [(1000, 0), (333, 1), (77, 2)], 3
    for r in range(D):
        h = B.phx_shard_create(layout, D, r, precision=precision, payload=B.PHX_PAYLOAD_FULL_RANK_STATE)
        h0 = B.phx_shard_create(layout, D, r, precision=precision)
        i, i0 = B.phx_shard_info(h), B.phx_shard_info(h0)
        fr = RS.FullRankState(O.OracleShard(layout, D, r, precision="fp32" if eb == 4 else "bf16"))
        assert i.param_bytes == D * i.n_padded * eb == fr.w_bytes == i0.param_bytes
        assert i.host_snapshot_bytes == fr.snapshot_bytes == i.snapshot_bytes + i.param_bytes
        assert i.host_slot_stride % 256 == 0 and 0 <= i.host_slot_stride - i.host_snapshot_bytes < 256
        assert (i0.host_snapshot_bytes, i0.host_slot_stride) == (i0.snapshot_bytes, i0.slot_stride)
        assert (i.snapshot_bytes, i.slot_stride, i.layout_hash) == (i0.snapshot_bytes, i0.slot_stride, i0.layout_hash)
        L = B.lib()
        assert L.phx_shard_bind_params(h, 256) == B.PHX_ERR_NOT_BOUND
        assert L.phx_params_ready(h, None) == B.PHX_ERR_NOT_BOUND
        assert L.phx_params_guard(h, None) == B.PHX_ERR_NOT_BOUND
        assert L.phx_shard_bind_params(h, None) == B.PHX_ERR_INVALID_ARG
        B.phx_shard_destroy(h)
        B.phx_shard_destroy(h0)
