"""phx_hbm_probe_async (BENCH-ONLY diagnostic of bench.py's roofline context, libphx_probe.so — not part of the
product library): touches exactly the planes it is told to, leaves the read planes and everything behind the
last plane alone, rejects bad arguments."""
import pytest
import torch

from paper_2607_01646_b200 import probe as PB

from gpu_util import DEV

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("r,w", [(1, 0), (0, 1), (1, 1), (3, 6), (8, 8), (4, 0)])
def test_probe_reads_and_writes_only_its_planes(r, w):
    plane = 256 * 37
    buf = torch.full(((r + w + 1) * plane,), 0x5A, dtype=torch.uint8, device=DEV)
    buf[:r * plane].view(torch.float32).fill_(0.25)                   # small values: group index + sum stays exact
    assert PB.phx_hbm_probe_async(buf, plane, r, w, torch.cuda.current_stream()) == 0
    torch.cuda.synchronize()
    assert bool((buf[:r * plane].view(torch.float32) == 0.25).all())  # read planes untouched
    assert bool((buf[(r + w) * plane:] == 0x5A).all())                # nothing behind the last plane
    if w:
        f = buf[r * plane:(r + w) * plane].view(torch.float32).view(w, -1)
        # every written plane holds the same values: group index + the sum of the read planes
        assert bool((f == f[0]).all())
        want = (torch.arange(plane // 32, device=DEV, dtype=torch.float32) + 0.25 * r).repeat_interleave(8)
        assert torch.equal(f[0], want)


def test_probe_argument_errors():
    L = PB.lib()
    buf = torch.zeros(4096, dtype=torch.uint8, device=DEV)
    assert L.phx_hbm_probe_async(None, 256, 1, 1, None) == -1
    assert L.phx_hbm_probe_async(buf.data_ptr(), 0, 1, 1, None) == -1
    assert L.phx_hbm_probe_async(buf.data_ptr(), 100, 1, 1, None) == -1
    assert L.phx_hbm_probe_async(buf.data_ptr(), 256, 9, 0, None) == -1
    assert L.phx_hbm_probe_async(buf.data_ptr(), 256, 0, 0, None) == -1
    assert L.phx_hbm_probe_async(buf.data_ptr() + 16, 256, 1, 1, None) == -2


def test_persistent_structure_writes_the_same_bytes_as_the_one_shot_structure():
    plane = 256 * 1000 + 256 * 3
    a = torch.zeros(9 * plane, dtype=torch.uint8, device=DEV)
    a[:3 * plane].view(torch.float32).fill_(0.5)
    b = a.clone()
    st = torch.cuda.current_stream()
    assert PB.phx_hbm_probe_async(a, plane, 3, 6, st) == 0
    assert PB.phx_hbm_probe_persistent_async(b, plane, 3, 6, 148 * 4, st) == 0
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    assert PB.lib().phx_hbm_probe_persistent_async(b.data_ptr(), plane, 3, 6, 0, None) == -1
