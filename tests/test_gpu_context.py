"""GPU tests of the context API of include/fx.h: explicit contexts are independent of each other and of the
default context -- two streams interleaved, two host threads at once -- give the oracle's bits, and leak nothing."""
import ctypes as C
import math
import threading

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


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float64).view(np.uint64)


def test_two_contexts_two_streams_interleaved(fx, oracle):
    """exact dots, an apply and axpbys enqueued alternately on two contexts with their own streams and scratch: every result
    equals the oracle's (one shared digit scratch would mix the two accumulations)"""
    import torch
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    c1, c2 = fx.Context(stream=s1), fx.Context(stream=s2)
    n = (1 << 22) + 13
    xs = [fi.uniform(301 + i, n) for i in range(4)]
    d = [dev(x) for x in xs]
    out1 = [torch.zeros(1, dtype=torch.float64, device="cuda") for _ in range(6)]
    out2 = [torch.zeros(1, dtype=torch.float64, device="cuda") for _ in range(6)]
    g = fx.make_grid(96, 64, 3, 2 * math.pi, 3.0, 0, 1)
    og = oracle.Grid(96, 64, 3, 2 * math.pi, 3.0, 0, 1)
    xa = fi.uniform(311, g.n); chi = 1.0 + 0.5 * fi.uniform(312, g.n)
    dxa, dchi = dev(xa), dev(chi)
    y1 = torch.empty(g.n, dtype=torch.float64, device="cuda"); y2 = torch.empty_like(y1)
    torch.cuda.synchronize()
    for i in range(6):                                   # device-resident results: nothing synchronises in between
        c1.exdot(d[0], d[1], out=out1[i])
        c2.exdot(d[2], d[3], out=out2[i])
        if i == 2:
            c1.dg_elliptic_apply(g, dchi, dxa, y1, sym=True)
            c2.dg_elliptic_apply(g, dchi, dxa, y2, sym=False)
    v_default = fx.exdot(d[0], d[3])                     # the default context works beside them
    torch.cuda.synchronize()
    w1, w2 = oracle.exdot(xs[0], xs[1]), oracle.exdot(xs[2], xs[3])
    for i in range(6):
        assert bits(out1[i].cpu().numpy())[0] == bits(w1)[()] and bits(out2[i].cpu().numpy())[0] == bits(w2)[()], i
    assert bits(v_default)[()] == bits(oracle.exdot(xs[0], xs[3]))[()]
    assert np.array_equal(bits(y1.cpu().numpy()), bits(oracle.dg_apply_canonical(og, chi, xa, normed=False)))
    assert np.array_equal(bits(y2.cpu().numpy()), bits(oracle.dg_apply_canonical(og, chi, xa, normed=True)))
    assert bits(c1.exdot(d[0], d[1]))[()] == bits(w1)[()]          # the synchronising form
    c1.destroy(); c2.destroy()


def test_two_threads_two_contexts_cg(fx, oracle):
    """two host threads solve two different systems at the same time, each on its own context (ctypes releases the GIL)"""
    import torch
    cfgs = [fi.config0(N=24), fi.config2(N=40)]
    wants = []
    for c in cfgs:
        og = oracle.Grid(**c["grid"])
        wants.append(oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], c["tol"], c["maxit"]))
    res = [None, None]

    def work(i):
        torch.cuda.set_device(0)
        c = cfgs[i]
        ctx = fx.Context(stream=torch.cuda.Stream())
        g = fx.make_grid(**c["grid"])
        for rep in range(3):
            phi = dev(c["phi0"])
            info = ctx.cg_solve(g, dev(c["chi"]), dev(c["rho"]), phi, c["tol"], c["maxit"])
            res[i] = (phi.cpu().numpy(), info.iterations)
        ctx.destroy()

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for i in range(2):
        assert res[i] is not None
        assert res[i][1] == wants[i][1].iterations
        assert np.array_equal(bits(res[i][0]), bits(wants[i][0]))


def test_create_destroy_leaks_nothing(fx):
    import torch
    x = dev(fi.uniform(321, 100003))
    g = fx.make_grid(32, 32, 3, 1.0, 1.0, 1, 1)
    chi = dev(1.0 + 0.5 * fi.uniform(322, g.n)); rho = dev(fi.uniform(323, g.n))

    def cycle():
        c = fx.Context()
        c.exdot(x, x)
        phi = torch.zeros(g.n, dtype=torch.float64, device="cuda")
        c.cg_solve(g, chi, rho, phi, 1e-6, 50)
        c.destroy()

    for _ in range(3):
        cycle()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(40):
        cycle()
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < (4 << 20), (free0, free1)      # the caching allocator of torch may move by a block; a leak of 40 work spaces would not fit


def test_context_errors(fx):
    import torch
    lib = fx.lib()
    h = C.c_void_p()
    assert lib.fx_create(C.byref(h), 4096, None) == fx.EINVAL           # no such device
    assert lib.fx_create(None, 0, None) == fx.EINVAL
    x = torch.ones(8, dtype=torch.float64, device="cuda")
    v = C.c_double()
    assert lib.fx_exdot_ex(None, x.data_ptr(), x.data_ptr(), 8, C.byref(v), None) == fx.EINVAL       # null context
    c = fx.Context()
    assert lib.fx_exdot_ex(c._h, x.data_ptr(), x.data_ptr(), 8, None, None) == fx.EINVAL             # nowhere to put the result
    assert c.exdot(x, x) == 8.0
    assert c.exsum(x) == 8.0
    c.destroy()
    lib.fx_destroy(None)                                                 # ignored
    # fx_shutdown releases the default context; the next plain call makes a new one
    assert fx.exdot(x, x) == 8.0
    lib.fx_shutdown()
    assert fx.exdot(x, x) == 8.0
