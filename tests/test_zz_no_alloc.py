"""GPU test of the allocation-free entry point fx_exdot_static (include/fx.h): the exact dot product with
the long accumulator's device scratch in a static __device__ array of the library instead of a context's work space.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process (the static path needs no
context: it is called BEFORE the existing path here) and after the other tests."""
import ctypes as C

import numpy as np
import pytest

import fxinputs as fi

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fx():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import paper_1807_01971_b200 as fx
    fx.lib()
    return fx


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def bits(v):
    return np.asarray(v, dtype=np.float64).reshape(-1).view(np.uint64)


def test_static_exdot_equals_existing_path_two_calls_in_a_row(fx, oracle):
    import torch
    n1, n2 = (1 << 22) + 13, 70001                     # several tiles per CTA + ragged tail; then a short one
    x1, y1 = fi.uniform(9101, n1), fi.uniform(9102, n1)
    x2, y2 = fi.uniform(9103, n2) * 1e200, fi.uniform(9104, n2) * 1e-250      # other exponents: stale digits would show
    d = [dev(a) for a in (x1, y1, x2, y2)]
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    fx.exdot_static(d[0][1:9], d[1][1:9], out[2:3]); fx.exdot_static(d[0][:8], d[1][:8], out[2:3])   # (the driver loads a kernel's code at its first launch)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    fx.exdot_static(d[0], d[1], out[0:1])             # two calls in a row on one stream, nothing in between
    fx.exdot_static(d[2], d[3], out[1:2])
    fx.exdot_static(d[0][1:], d[1][1:], out[2:3])      # 8-byte aligned inputs: the scalar-copy variant of the kernel
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                              # the device's free memory did not move
    got = out.cpu().numpy()
    want = [fx.exdot(d[0], d[1]), fx.exdot(d[2], d[3]), fx.exdot(d[0][1:], d[1][1:])]          # the existing path (context scratch)
    assert np.array_equal(bits(got), bits(want)), (got, want)                                  # exact: bit for bit
    assert bits(got[1])[0] == bits(oracle.exdot(x2, y2))[0]
    # again, the other way round, on a stream of the caller's
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    out2 = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    s.wait_stream(torch.cuda.current_stream())
    fx.exdot_static(d[2], d[3], out2[0:1], stream=s)
    fx.exdot_static(d[0], d[1], out2[1:2], stream=s)
    s.synchronize()
    assert np.array_equal(bits(out2.cpu().numpy()), bits([want[1], want[0]]))


def test_static_exdot_special_values_and_empty(fx):
    import torch
    out = torch.full((4,), 7.0, dtype=torch.float64, device="cuda")
    big = dev(np.array([2.0 ** 1000, -2.0 ** 1000, 2.0 ** -1074, 1.0]))
    oth = dev(np.array([2.0 ** 1000, 2.0 ** 1000, 1.0, 3.0]))           # 2^2000 - 2^2000 + 2^-1074 + 3 rounds to 3
    nan = dev(np.array([1.0, float("nan")]))
    inf = dev(np.array([float("inf"), 1.0]))
    fx.exdot_static(big, oth, out[0:1])
    fx.exdot_static(nan, nan, out[1:2])
    fx.exdot_static(inf, inf, out[2:3])                # the flags of the call before (NaN) must not leak into this one
    fx.exdot_static(big[:0], oth[:0], out[3:4])        # n = 0 gives +0.0
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got[0] == 3.0 and np.isnan(got[1]) and got[2] == float("inf") and bits(got[3])[0] == 0


def test_static_exdot_rejects_sizes_beyond_the_maximum(fx):
    import torch
    lib = fx.lib()
    x = torch.ones(8, dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    # the size is checked before anything is touched: no 2 GiB arrays are needed to see the error
    rc = lib.fx_exdot_static(x.data_ptr(), x.data_ptr(), fx.EXDOT_STATIC_MAX_N + 1, out.data_ptr(), None)
    assert rc == fx.EINVAL and b"FX_EXDOT_STATIC_MAX_N" in lib.fx_last_error()
    assert lib.fx_exdot_static(x.data_ptr(), x.data_ptr(), -1, out.data_ptr(), None) == fx.EINVAL
    assert lib.fx_exdot_static(x.data_ptr(), x.data_ptr(), 8, None, None) == fx.EINVAL
    assert lib.fx_exdot_static(x.data_ptr(), x.data_ptr(), 8, out.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert out.item() == 8.0
