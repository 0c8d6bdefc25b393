"""The C-ABI boundary used from plain C (tests/c_abi/phx_c_client.c: cudaMalloc/cudaHostAlloc buffers, no Python,
no torch in the process that runs the hot path): step + snapshot + flush, loss of the live shard, restore, recompute,
the gradient producer's epilogue feeding a step, two steps through the graph-capturable form — its output file
compared byte for byte with the CPU oracle.  The header also has to compile as strict C99."""
import os
import struct
import subprocess
import sys

import numpy as np
import pytest
import torch

from oracle import grad_finalize as GF
from oracle import oracle as O
from paper_2607_01646_b200 import binding as B
from paper_2607_01646_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_abi", "phx_c_client.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def test_header_is_strict_c99(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "phx.h"\nint main(void) { return (int)sizeof(phx_config_t) - 64; }\n')
    subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    "-fsyntax-only", str(c)], check=True)


def _build(tmp_path):
    exe = str(tmp_path / "phx_c_client")
    libdir = os.path.dirname(B.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-O1", "-Wall", "-I", os.path.join(ROOT, "include"), "-I", f"{CUDA}/include",
                    SRC, "-o", exe, "-L", libdir, "-lphx", f"-Wl,-rpath,{libdir}", "-L", f"{CUDA}/lib64", "-lcudart",
                    f"-Wl,-rpath,{CUDA}/lib64"], check=True)
    return exe


def test_c_client_builds_against_the_header_and_library(tmp_path):
    B.lib()
    _build(tmp_path)


@pytest.mark.gpu
@pytest.mark.parametrize("numels,dp,rank,max_norm", [([300_000, 1234, 77], 2, 1, 0.0), ([70_001, 64], 3, 0, 0.01)])
def test_c_client_matches_the_oracle(tmp_path, numels, dp, rank, max_norm):
    exe = _build(tmp_path)
    steps, chunk = 3, 1 << 18
    wl = W.tiny_workload(numels, dp_size=dp, dp_rank=rank, grad_kind="heavy_tail", hyper=W.Hyper(max_grad_norm=max_norm))
    blob = b"rng-state-of-the-c-client\0"
    o = O.OracleShard(wl.layout(), dp, rank, chunk_bytes=chunk, max_grad_norm=max_norm, user=blob)
    N = o.n_padded
    p0 = W.init_params(o.n, N, 5).numpy()
    segs = [(tid, off, ln) for tid, _, off, ln in o.segments]
    grads = [W.gen_grads(wl, segs, N, t, 9).view(torch.int16).numpy().view(np.uint16).copy() for t in range(1, steps + 2)]
    inp, outp = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(inp, "wb") as f:
        f.write(struct.pack("<Q", len(numels)))
        f.write(struct.pack(f"<{len(numels)}Q", *numels))
        f.write(struct.pack("<IIIfQ", dp, rank, steps, max_norm, chunk))
        f.write(p0.tobytes())
        for g in grads:
            f.write(g.tobytes())
        rng = np.random.default_rng(4)
        g32 = (rng.standard_t(3, N) * 2e-3).astype(np.float32)
        g32[o.n:] = 0
        scale = np.float32(1.0 / 3.0)
        f.write(struct.pack("<f", scale))
        f.write(g32.tobytes())
    r = subprocess.run([exe, str(inp), str(outp)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "phx_c_client ok" in r.stdout
    # the oracle's run of the same protocol
    hp = dict(lr=3e-4, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)
    o.set_state(p0)
    for t in range(1, steps + 1):
        o.step(grads[t - 1], **hp, step=t)
        o.snapshot()
    o.step(grads[steps], **hp, step=steps + 1)            # in flight, lost
    o.drop_live()
    assert o.restore() == steps
    o.step(grads[steps], **hp, step=steps + 1)            # recompute
    o.snapshot()                                          # ... and its flush
    gbits, _ = GF.grads_finalize(g32, scale)              # producer epilogue -> the next step's gradients
    o.step(gbits, **hp, step=steps + 2)
    for k in (0, 1):                                      # graph form: flush of the pending snapshot, then step
        o.snapshot()
        o.step(grads[k], **hp, step=steps + 3 + k)
    o.snapshot()                                          # second fault: newest snapshot flushed, live shard lost,
    o.drop_live()                                         # two-phase restore, one more step
    assert o.restore_params_first() == steps + 4 and o.restore_finish() == steps + 4
    o.step(grads[0], **hp, step=steps + 5)
    replica = [x.copy() for x in o.replica]               # slots now hold steps+3 and steps+4
    raw = open(outp, "rb").read()
    n_padded, back = struct.unpack_from("<QQ", raw, 0)
    assert (n_padded, back) == (N, steps)
    off = 16
    for name, ref in (("p", o.p), ("m", o.m), ("v", o.v)):
        got = np.frombuffer(raw, np.uint32, N, off)
        assert np.array_equal(got, ref.view(np.uint32)), name
        off += 4 * N
    assert np.array_equal(np.frombuffer(raw, np.uint16, N, off), o.p16)
    off += 2 * N
    stride = (o.snapshot_bytes + 255) // 256 * 256
    for k in range(2):
        got = np.frombuffer(raw, np.uint8, o.snapshot_bytes, off + k * stride)
        assert np.array_equal(got, replica[k]), f"replica slot {k}"
