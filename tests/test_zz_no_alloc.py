"""rsos_sums_static against rsos_sums (GPU, run with -m gpu; named test_zz_* so that pytest collects it last).

rsos_sums_static is the one entry point of librsos that allocates nothing.  It is there for users who hold surfaces in
device memory but cannot call cudaMalloc: their process has given all device memory to another pool (here that pool is
torch's allocator, which owns every buffer this test passes in), or they sit in a loop that must not take the
device-wide stall an allocation causes.  Its accumulators live in a fixed array inside the library that every call
shares and that keeps the previous call's contents, so the thing to test is a SEQUENCE of calls: each one has to clear
what it uses.  The calls below go from few realizations to many and back, on lattices of different size, so rows left
over from a larger call would show up in the sums of the next one.

The bar is the one the other GPU tests use for integer work: exact equality, here with the existing context path
(rsos_sums on the same surfaces) and with numpy sums of the heights read back through rsos_get_heights.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rsos():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1605_02620_b200 import build
    build.build()
    import paper_1605_02620_b200 as m
    return m


def static_sums(m, g, torch, out=None):
    """One rsos_sums_static call on the int32 heights of context g; outputs in torch-owned device arrays."""
    R = g.R
    if out is None:
        out = (torch.full((R,), -7, dtype=torch.int64, device="cuda"), torch.full((R,), -7, dtype=torch.int64, device="cuda"),
               torch.full((R,), -7, dtype=torch.int32, device="cuda"))
    s1, s2, mx = out
    d = g.device_heights()                       # int32 h[r][y][x] on the device, current as of this call
    m.sums_static(d, g.L, R, s1.data_ptr(), s2.data_ptr(), mx.data_ptr())      # legacy default stream, like the context
    torch.cuda.synchronize()
    return s1.cpu().numpy(), s2.cpu().numpy().view(np.uint64), mx.cpu().numpy().view(np.uint32)


def check(m, g, torch, what, out=None):
    s1, s2, mx = static_sums(m, g, torch, out)
    e1, e2, _ = g.sums()                         # the existing path: buffers allocated by rsos_init
    assert (s1 == e1).all(), what + ": S1 differs from rsos_sums"
    assert (s2 == e2).all(), what + ": S2 differs from rsos_sums"
    h = g.heights().astype(np.int64)
    assert (s1 == h.sum(axis=(1, 2))).all() and (s2 == (h * h).sum(axis=(1, 2)).astype(np.uint64)).all(), what
    assert (mx == np.abs(h).max(axis=(1, 2))).all(), what + ": max |h|"


def test_static_sums_equal_context_sums_call_after_call(rsos):
    import torch
    m = rsos
    a = m.Rsos(256, 1, 5, 11, tile=64)                       # DT mode, 5 surfaces
    b = m.Rsos(100, 2, 37, 12)                               # L*L = 10^4 (a multiple of 4), serial mode, 37 surfaces
    c = m.Rsos(33, 3, 9, 13)                                 # L*L odd: the one-site-per-load form of the kernel
    a.advance(7)
    b.advance(5)
    c.advance(9)
    check(m, a, torch, "first call (R = 5)")
    check(m, b, torch, "second call (R = 37, rows 5..36 untouched so far)")
    check(m, a, torch, "third call (R = 5 again: rows 0..4 hold the sums of the R = 37 call)")
    check(m, c, torch, "fourth call (R = 9, odd L)")
    a.advance(3)                                             # same rows, new content
    out = (torch.zeros(5, dtype=torch.int64, device="cuda"), torch.zeros(5, dtype=torch.int64, device="cuda"),
           torch.zeros(5, dtype=torch.int32, device="cuda"))
    check(m, a, torch, "fifth call, warm-up of the shape measured below", out)
    a.advance(1)
    free0 = torch.cuda.mem_get_info()[0]
    check(m, a, torch, "sixth call", out)
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed across an rsos_sums_static call"
    for g in (a, b, c):
        g.close()


def test_static_sums_at_the_size_limit_and_beyond(rsos):
    import torch
    m = rsos
    R = m.STATIC_MAX_R
    g = m.Rsos(32, 1, R, 5)                                  # as many surfaces as the fixed array has rows
    g.advance(4)
    check(m, g, torch, "R = RSOS_STATIC_MAX_R")
    small = m.Rsos(64, 1, 3, 6)
    small.advance(6)
    check(m, small, torch, "R = 3 right after the full-size call")
    d = g.device_heights()
    buf = torch.zeros(R + 1, dtype=torch.int64, device="cuda")
    with pytest.raises(m.RsosError) as e:
        m.sums_static(d, 32, R + 1, buf.data_ptr(), buf.data_ptr(), None)
    assert e.value.code == m.binding.RSOS_EINVAL and "RSOS_STATIC_MAX_R" in str(e.value)
    with pytest.raises(m.RsosError):
        m.sums_static(d, 32, 4, None, None, None)            # nowhere to write
    with pytest.raises(m.RsosError):
        m.sums_static(None, 32, 4, buf.data_ptr(), None, None)
    g.close()
    small.close()
