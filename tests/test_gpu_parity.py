"""GPU parity: libfx.so (through its C ABI) against the CPU oracle, element by element, on the same seeded inputs.

Bars (BASELINE.json north_star / DESIGN.md 7): exact dot and every integer digit bit-exact; axpby, pointwise_dot, dG
weights and the dG apply bit-exact against the oracle's canonical order (so also <= 1e-14), the apply additionally
<= 1e-14 * scale against the 113-bit definition; CG: identical iteration count, relative L2 <= 1e-10 (expected: 0),
bitwise identical across repeats, fused/unfused drivers and launch shapes.
"""
import math

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


def same_bits(a, b):
    return np.array_equal(bits(a), bits(b))


def fbits(v):
    return np.float64(v).view(np.uint64)


@pytest.fixture(autouse=True)
def _default_launch(fx):
    yield
    for k in range(4):
        fx.set_launch(k, 0, 0)
    fx.set_cg_fused(1)
    fx.set_dg_path(0)


# ---- exact dot ----------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [0, 1, 2, 3, 31, 32, 33, 255, 1024, 1025, 4099, 100003, (1 << 20) + 7])
def test_exdot_uniform_sizes(fx, oracle, n):
    x, y = fi.uniform(11, n), fi.uniform(12, n)
    want = oracle.exdot(x, y) if n else 0.0
    got = fx.exdot(dev(x), dev(y)) if n else fx.exdot(dev(np.zeros(0)), dev(np.zeros(0)))
    assert fbits(got) == fbits(want)


@pytest.mark.parametrize("k", [10, 13, 17, 20])
@pytest.mark.parametrize("ci", range(6))
def test_exdot_condition_family(fx, oracle, k, ci):
    x, y, expected = fi.dot_family_a(k, ci)
    want, limbs, flags = oracle.exdot_digits(x, y)
    if expected is not None:
        assert want == expected                      # closed form by construction: 26 * 2^-e
    got, glimbs, gflags = fx.exdot_digits(dev(x), dev(y))
    assert fbits(got) == fbits(want)
    assert np.array_equal(glimbs, limbs)             # the long accumulator itself, digit for digit
    assert np.array_equal(gflags, flags)


def test_exdot_special_cases(fx, oracle):
    for name, x, y in fi.dot_special_cases():
        want, limbs, flags = oracle.exdot_digits(x, y)
        got, glimbs, gflags = fx.exdot_digits(dev(x), dev(y))
        if math.isnan(want):
            assert math.isnan(got), name
        else:
            assert fbits(got) == fbits(want), (name, got, want)
        assert np.array_equal(gflags, flags), name
        if not flags.any():
            assert np.array_equal(glimbs, limbs), name


def test_exdot_paper_example_and_closed_forms(fx):
    import itertools
    for perm in itertools.permutations([-1.0, 1.0, 2.0 ** -53]):
        assert fx.exdot(dev(np.array(perm)), dev(np.ones(3))) == 2.0 ** -53
    n = 300000                                                          # sum i^2 beyond 2^53
    i = np.arange(1, n + 1, dtype=np.float64)
    exact = n * (n + 1) * (2 * n + 1) // 6
    assert fx.exdot(dev(i), dev(i)) == float(exact)
    x = np.ldexp(1.0, -np.arange(1, 55))                                # sum 2^-i, i=1..54 is a tie -> 1.0
    assert fx.exdot(dev(x), dev(np.ones(54))) == 1.0
    assert fx.exdot(dev(x[:53]), dev(np.ones(53))) == 1.0 - 2.0 ** -53


def test_exdot_wide_exponent_spread(fx, oracle):
    """products far below the warp's window take the slow path; all of config 1's range in one vector"""
    g = fi.rng(77)
    n = 20000
    x = np.ldexp(1.0 + g.random(n), g.integers(-500, 500, n)) * np.where(g.random(n) < 0.5, -1, 1)
    y = np.ldexp(1.0 + g.random(n), g.integers(-500, 500, n))
    want, limbs, _ = oracle.exdot_digits(x, y)
    got, glimbs, _ = fx.exdot_digits(dev(x), dev(y))
    assert fbits(got) == fbits(want)
    assert np.array_equal(glimbs, limbs)


def test_exdot_launch_shape_and_alignment_invariance(fx, oracle):
    n = 300007
    x, y = fi.uniform(21, n + 1), fi.uniform(22, n + 1)
    x[:100] *= 1e-30
    y[5000:5100] *= 1e25
    dx, dy = dev(x), dev(y)
    want = oracle.exdot(x[:n], y[:n])
    for grid, block in [(0, 0), (1, 32), (3, 64), (148, 128), (1000, 256), (7, 1024), (296, 512)]:
        fx.set_launch(0, grid, block)
        assert fbits(fx.exdot(dx[:n], dy[:n])) == fbits(want), (grid, block)
    fx.set_launch(0, 0, 0)
    assert fbits(fx.exdot(dx[1:], dy[1:])) == fbits(oracle.exdot(x[1:], y[1:]))        # both 8-byte aligned only
    assert fbits(fx.exdot(dx[1:], dy[:n])) == fbits(oracle.exdot(x[1:], y[:n]))        # mixed alignment
    assert fbits(fx.exdot(dx, dx)) == fbits(oracle.exdot(x, x))                        # aliasing (norm)


def test_exdot_async_and_host(fx, oracle):
    import torch
    n = 70001
    x, y = fi.uniform(31, n), fi.uniform(32, n)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    fx.exdot_async(dev(x), dev(y), out)
    want = oracle.exdot(x, y)
    assert fbits(out.cpu().numpy()[0]) == fbits(want)
    assert fbits(fx.exdot_host(torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory())) == fbits(want)


def test_exdot_multi_launch_and_host_chunks(fx, oracle):
    """n > 2^28 is accumulated over two launches (limbs carried between them); fx_exdot_host streams 2^23-element chunks"""
    import torch
    n = (1 << 28) + 12345
    x, y = fi.uniform(33, n), fi.uniform(34, n)
    x[::1000003] *= 1e30
    want, limbs, flags = oracle.exdot_digits(x, y)
    got, glimbs, gflags = fx.exdot_digits(dev(x), dev(y))
    assert fbits(got) == fbits(want) and np.array_equal(glimbs, limbs) and np.array_equal(gflags, flags)
    m = (1 << 24) + 77                                            # three host chunks, ragged tail
    assert fbits(fx.exdot_host(x[:m], y[:m])) == fbits(oracle.exdot(x[:m], y[:m]))
    # a negative total: the sign fill of the upper limbs after the first launch must survive the second one
    xn = -np.abs(x[: (1 << 28) + 5]); yn = np.abs(y[: (1 << 28) + 5])
    want, limbs, _ = oracle.exdot_digits(xn, yn)
    got, glimbs, _ = fx.exdot_digits(dev(xn), dev(yn))
    assert fbits(got) == fbits(want) and np.array_equal(glimbs, limbs)


@pytest.mark.parametrize("k", [24, 27])
@pytest.mark.parametrize("ci", range(6))
def test_exdot_full_size_config1(fx, oracle, ci, k):
    """config 1, family A at n = 2^24 and 2^27 (the sizes and launch configuration bench.py times), every condition target:
    the value and all 68 limbs of the long accumulator"""
    x, y, expected = fi.dot_family_a(k, ci)
    want, limbs, flags = oracle.exdot_digits(x, y)
    if expected is not None:
        assert want == expected
    got, glimbs, gflags = fx.exdot_digits(dev(x), dev(y))
    assert fbits(got) == fbits(want)
    assert np.array_equal(glimbs, limbs) and np.array_equal(gflags, flags)


@pytest.mark.parametrize("k,ci", [(20, 1), (20, 2), (20, 3), (20, 4), (20, 5), (21, 3), (22, 5)])
def test_exdot_family_b_residue_cancellation(fx, oracle, k, ci):
    """config 1, family B: the second half drives the running sum down through the whole exponent range, the
    result is what the rounding residues leave.  Value, limbs, and the achieved condition number (exact, from the oracle)."""
    x, y = fi.dot_family_b(k, ci, oracle)
    want, limbs, flags = oracle.exdot_digits(x, y)
    cond = 2.0 * oracle.exdot(np.abs(x), np.abs(y)) / abs(want)
    assert cond >= 1e-3 * fi.COND_TARGETS[ci]
    fx.exdot_stats(reset=True)
    got, glimbs, gflags = fx.exdot_digits(dev(x), dev(y))
    assert fbits(got) == fbits(want)
    assert np.array_equal(glimbs, limbs) and np.array_equal(gflags, flags)
    st = fx.exdot_stats()
    assert st["deposit_product"] == 0                                  # all products inside TwoProd's error-free range
    # launch-shape invariance on the ill-conditioned data too
    for grid, block in [(1, 32), (77, 64), (1000, 256)]:
        fx.set_launch(0, grid, block)
        assert fbits(fx.exdot(dev(x), dev(y))) == fbits(want), (grid, block)


def test_exdot_stats_census(fx, oracle):
    """fx_exdot_stats: uniform data never leaves the register window; a +-500 exponent spread does, and 2^1000-class products
    take the integer-product path -- with the oracle's bits either way"""
    n = 1 << 20
    x, y = fi.uniform(41, n), fi.uniform(42, n)
    fx.exdot_stats(reset=True)
    assert fbits(fx.exdot(dev(x), dev(y))) == fbits(oracle.exdot(x, y))
    st = fx.exdot_stats(reset=True)
    assert st["deposit_product"] == 0 and st["deposit_double"] <= n // 1000
    x, y = fi.dot_wide_spread(n)
    assert fbits(fx.exdot(dev(x), dev(y))) == fbits(oracle.exdot(x, y))
    st = fx.exdot_stats(reset=True)
    assert st["deposit_double"] + st["deposit_product"] > 0 and st["window_moves"] > 0
    assert fx.exdot_stats() == dict(deposit_double=0, deposit_product=0, window_moves=0)


# ---- axpby / pointwise_dot / weights ------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 2, 7, 1023, 2048, 2049, 100003, (1 << 21) + 5])
@pytest.mark.parametrize("alpha,beta", [(0.7, -0.3), (1.25, 1.0), (-2.5, 0.0)])
def test_axpby_bit_exact(fx, oracle, n, alpha, beta):
    x, y = fi.uniform(41, n), fi.uniform(42, n)
    want = oracle.axpby(alpha, x, beta, y)
    got = fx.axpby(alpha, dev(x), beta, dev(y)).cpu().numpy()
    assert same_bits(got, want)


@pytest.mark.parametrize("n", [1, 5, 2047, 100003])
@pytest.mark.parametrize("alpha,beta", [(1.0, 0.0), (0.3, 0.9), (-1.0, 1.0)])
def test_pointwise_dot_bit_exact(fx, oracle, n, alpha, beta):
    x1, x2, y = fi.uniform(43, n), fi.uniform(44, n), fi.uniform(45, n)
    want = oracle.pointwise_dot(alpha, x1, x2, beta, y)
    got = fx.pointwise_dot(alpha, dev(x1), dev(x2), beta, dev(y)).cpu().numpy()
    assert same_bits(got, want)


def test_elementwise_unaligned_alias_and_shapes(fx, oracle):
    n = 5001
    x, y = fi.uniform(46, n + 1), fi.uniform(47, n + 1)
    dx, dy = dev(x), dev(y)
    got = fx.axpby(0.5, dx[1:], 2.0, dy[1:]).cpu().numpy()
    assert same_bits(got, oracle.axpby(0.5, x[1:], 2.0, y[1:]))
    dz = dev(x)
    assert same_bits(fx.axpby(3.0, dz, -1.5, dz).cpu().numpy(), oracle.axpby(3.0, x, -1.5, x))      # x is y
    for grid, block in [(1, 32), (5, 1024), (999, 64)]:
        fx.set_launch(1, grid, block)
        assert same_bits(fx.axpby(0.7, dev(x), -0.3, dev(y)).cpu().numpy(), oracle.axpby(0.7, x, -0.3, y))
    beta0 = fx.axpby(2.0, dev(x), 0.0, dev(np.full(n + 1, np.nan))).cpu().numpy()                   # y not read
    assert same_bits(beta0, oracle.axpby(2.0, x, 0.0, y))


GRIDS = [(1, 1), (2, 3), (3, 2), (31, 5), (30, 9), (61, 17), (64, 64)]
BCS = [(0, 0), (0, 1), (1, 0), (1, 1)]


def _grid(fx, oracle, Nx, Ny, P, bcx, bcy, lx=2 * math.pi, ly=3.0):
    return fx.make_grid(Nx, Ny, P, lx, ly, bcx, bcy), oracle.Grid(Nx, Ny, P, lx, ly, bcx, bcy)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_dg_weights_bit_exact(fx, oracle, P):
    import torch
    g, og = _grid(fx, oracle, 7, 5, P, 0, 1)
    w = torch.empty(g.n, dtype=torch.float64, device="cuda"); v = torch.empty_like(w)
    fx.dg_weights(g, w, v)
    W, V = oracle.dg_weights(og)
    assert same_bits(w.cpu().numpy(), W) and same_bits(v.cpu().numpy(), V)


# ---- dG apply -----------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("path", [0, 1])          # 0: CTA-tile kernels where TMA's rules allow (even pitch), 1: warp-strip kernels
@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("bc", BCS)
def test_dg_apply_bit_exact_small_grids(fx, oracle, P, bc, path):
    """raw bit patterns, the sign of zero included (P = 1 grids produce exact zeros)"""
    import torch
    fx.set_dg_path(path)
    for (Nx, Ny) in GRIDS + [(2, 2), (62, 3), (120, 5), (250, 12)]:
        g, og = _grid(fx, oracle, Nx, Ny, P, *bc)
        x = fi.uniform(51 + P, g.n); chi = 1.0 + 0.5 * fi.uniform(61 + P, g.n)
        for sym in (True, False):
            want = oracle.dg_apply_canonical(og, chi, x, normed=not sym)
            y = torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
            fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=sym)
            got = y.cpu().numpy()
            assert np.array_equal(got, want), (Nx, Ny, P, bc, sym, np.abs(got - want).max())
            assert same_bits(got, want), (Nx, Ny, P, bc, sym)


@pytest.mark.parametrize("P", [1, 2, 3])
def test_dg_apply_exact_zeros_keep_their_sign(fx, oracle, P):
    """inputs that make whole regions of the result exactly zero (constant x on a periodic grid, zero x, x = -0.0):
    the sign of every zero must match the oracle's, in both stencil kernels"""
    import torch
    for bc in [(0, 0), (0, 1), (1, 1)]:
        g, og = _grid(fx, oracle, 32, 6, P, *bc)
        chi = 1.0 + 0.5 * fi.uniform(63, g.n)
        for x in (np.ones(g.n), np.zeros(g.n), -np.zeros(g.n), -np.ones(g.n), np.where(np.arange(g.n) % 7 == 0, 1.0, 0.0)):
            want = oracle.dg_apply_canonical(og, chi, x, normed=False)
            for path in (0, 1):
                fx.set_dg_path(path)
                y = torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
                fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=True)
                assert same_bits(y.cpu().numpy(), want), (P, bc, path)


@pytest.mark.parametrize("P", [2, 3, 5])
def test_dg_apply_against_definition(fx, oracle, P):
    """|y - y_def| <= 1e-14 * (|F^T||W chi||F| + |J|)|x|, y_def from explicit block matrices in 113-bit arithmetic"""
    import torch
    g, og = _grid(fx, oracle, 12, 9, P, 0, 1)
    x = fi.uniform(71, g.n); chi = 1.0 + 0.5 * fi.uniform(72, g.n)
    for sym in (True, False):
        ydef, scale = oracle.dg_apply_definition(og, chi, x, normed=not sym)
        y = torch.empty(g.n, dtype=torch.float64, device="cuda")
        fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=sym)
        assert np.all(np.abs(y.cpu().numpy() - ydef) <= 1e-14 * scale)


def test_dg_apply_launch_shape_invariance(fx, oracle):
    import torch
    g, og = _grid(fx, oracle, 95, 40, 3, 0, 1)
    x = fi.uniform(73, g.n); chi = 1.0 + 0.5 * fi.uniform(74, g.n)
    want = oracle.dg_apply_canonical(og, chi, x, normed=False)
    for rows, block in [(0, 0), (1, 32), (3, 64), (7, 256), (40, 128), (1000, 1024)]:
        fx.set_launch(2, rows, block)
        y = torch.empty(g.n, dtype=torch.float64, device="cuda")
        fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=True)
        assert np.array_equal(y.cpu().numpy(), want), (rows, block)


def test_dg_apply_rejects_overlap_and_bad_grid(fx):
    import torch
    g = fx.make_grid(4, 4, 3, 1.0, 1.0, 0, 1)
    x = torch.zeros(g.n, dtype=torch.float64, device="cuda")
    with pytest.raises(fx.FxError):
        fx.dg_elliptic_apply(g, x, x, x)
    bad = fx.make_grid(4, 4, 6, 1.0, 1.0, 0, 1)
    with pytest.raises(fx.FxError):
        fx.dg_elliptic_apply(bad, torch.zeros(bad.n, dtype=torch.float64, device="cuda"), torch.zeros(bad.n, dtype=torch.float64, device="cuda"),
                             torch.zeros(bad.n, dtype=torch.float64, device="cuda"))


def test_dg_apply_full_size_config3(fx, oracle):
    """1024 x 1024 cells, P = 3: every element against the canonical oracle (default launch shape = bench.py's)"""
    import torch
    c = fi.config3()
    g, og = fx.make_grid(**c["grid"]), oracle.Grid(**c["grid"])
    x = fi.uniform(75, g.n)
    want = oracle.dg_apply_canonical(og, c["chi"], x, normed=False)
    y = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.dg_elliptic_apply(g, dev(c["chi"]), dev(x), y, sym=True)
    assert np.array_equal(y.cpu().numpy(), want)


# ---- CG -----------------------------------------------------------------------------------------------------------

def _solve(fx, c, tol=None, maxit=None):
    g = fx.make_grid(**c["grid"])
    phi = dev(c["phi0"])
    info = fx.cg_solve(g, dev(c["chi"]), dev(c["rho"]), phi, c["tol"] if tol is None else tol, c["maxit"] if maxit is None else maxit)
    return phi.cpu().numpy(), info


def test_cg_config0_matches_oracle(fx, oracle):
    c = fi.config0()
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], c["tol"], c["maxit"])
    got, info = _solve(fx, c)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status == 0
    rel = np.linalg.norm(got - want) / np.linalg.norm(want)
    assert rel <= 1e-10
    assert same_bits(got, want), "expected a bit-identical trajectory (rel = %g)" % rel
    assert info.rel_residual == oinfo.rel_residual
    # the manufactured solution: discretisation error of order P (Q7)
    W, _ = oracle.dg_weights(og)
    err = math.sqrt(np.sum(W * (got - c["phi_exact"]) ** 2) / np.sum(W * c["phi_exact"] ** 2))
    assert err < 1e-5


def test_cg_reproducible_across_runs_drivers_and_shapes(fx):
    c = fi.config0(N=32)
    ref, info0 = _solve(fx, c)
    for _ in range(2):
        got, info = _solve(fx, c)
        assert same_bits(got, ref) and info.iterations == info0.iterations
    for mode in (0, 2, 3):          # unfused / two fused kernels per iteration / persistent cooperative kernel
        fx.set_cg_fused(mode)
        got, info = _solve(fx, c)
        assert same_bits(got, ref) and info.iterations == info0.iterations, mode
    for path in (1, 2):             # warp-strip stencil everywhere / CTA-tile stencil everywhere (K1 included)
        fx.set_dg_path(path); fx.set_cg_fused(2)
        got, info = _solve(fx, c)
        assert same_bits(got, ref) and info.iterations == info0.iterations, path
    fx.set_dg_path(0)
    fx.set_cg_fused(2)
    for (rows, ablock, egrid, eblock, dgrid, dblock) in [(1, 32, 1, 32, 1, 32), (5, 128, 37, 512, 300, 64), (100, 1024, 999, 128, 2, 1024)]:
        fx.set_launch(2, rows, ablock); fx.set_launch(3, egrid, eblock); fx.set_launch(0, dgrid, dblock)
        for mode in (2, 3):
            fx.set_cg_fused(mode)
            got, info = _solve(fx, c)
            assert same_bits(got, ref) and info.iterations == info0.iterations, (mode, rows)


@pytest.mark.parametrize("P", [1, 2, 4, 5])
def test_cg_other_orders(fx, oracle, P):
    c = fi.config0(N=12, P=P)
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 1e-9, 3000)
    got, info = _solve(fx, c, tol=1e-9, maxit=3000)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status
    assert same_bits(got, want)


@pytest.mark.parametrize("Nx,Ny,P,bc", [(64, 24, 3, (0, 1)), (62, 9, 5, (1, 1)), (120, 7, 1, (0, 0)), (34, 40, 2, (1, 0)), (30, 6, 4, (2, 1)),
                                        (250, 5, 3, (3, 4))])
def test_cg_tile_k1_matches_oracle(fx, oracle, Nx, Ny, P, bc):
    """the fused kernel K1 on the CTA-tile stencil (fx_set_dg_path(2)): the oracle's iterates bit for bit, launch-shape invariant"""
    import torch
    g, og = _grid(fx, oracle, Nx, Ny, P, *bc)
    chi = 1.0 + 0.5 * fi.uniform(181, g.n); rho = fi.uniform(182, g.n); phi0 = 0.1 * fi.uniform(183, g.n)
    want, oinfo = oracle.cg_solve(og, chi, rho, phi0, 0.0, 25)
    fx.set_dg_path(2); fx.set_cg_fused(2)
    for rows in (0, 1, 3):
        fx.set_launch(2, rows, 0)
        phi = dev(phi0)
        info = fx.cg_solve(g, dev(chi), dev(rho), phi, 0.0, 25)
        assert info.iterations == oinfo.iterations == 25
        assert same_bits(phi.cpu().numpy(), want), (rows,)


@pytest.mark.parametrize("mode", [1, 2])
def test_cg_config2_reduced_and_maxit(fx, oracle, mode):
    fx.set_cg_fused(mode)
    c = fi.config2(N=48)
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], c["tol"], c["maxit"])
    got, info = _solve(fx, c)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status == 0
    assert same_bits(got, want)
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 0.0, 37)        # fixed iteration count (config 3's mode)
    got, info = _solve(fx, c, tol=0.0, maxit=37)
    assert info.iterations == oinfo.iterations == 37 and info.status == oinfo.status == 1
    assert same_bits(got, want)


def test_cg_zero_rhs_and_nonzero_start(fx, oracle):
    c = fi.config0(N=8)
    og = oracle.Grid(**c["grid"])
    z = np.zeros_like(c["rho"])
    got, info = _solve(fx, dict(c, rho=z, phi0=fi.uniform(81, z.size)))
    assert info.iterations == 0 and np.all(got == 0.0)
    phi0 = 0.1 * fi.uniform(82, z.size)
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], phi0, 1e-9, 2000)
    got, info = _solve(fx, dict(c, phi0=phi0), tol=1e-9, maxit=2000)
    assert info.iterations == oinfo.iterations and same_bits(got, want)


@pytest.mark.parametrize("Nx,Ny,P", [(15, 9, 3), (33, 7, 5), (7, 5, 1), (61, 4, 2)])
def test_cg_odd_pitch_and_unaligned_phi(fx, oracle, Nx, Ny, P):
    """rows that are not 16-byte aligned (odd Nx*P), ragged tiles, and a caller phi that is only 8-byte aligned"""
    import torch
    grid = dict(Nx=Nx, Ny=Ny, P=P, lx=2 * math.pi, ly=1.7, bcx=0, bcy=1)
    g, og = fx.make_grid(**grid), oracle.Grid(**grid)
    chi = 1.0 + 0.5 * fi.uniform(91, g.n); rho = fi.uniform(92, g.n); phi0 = 0.01 * fi.uniform(93, g.n)
    want, oinfo = oracle.cg_solve(og, chi, rho, phi0, 1e-9, 400)
    phi = dev(phi0)
    info = fx.cg_solve(g, dev(chi), dev(rho), phi, 1e-9, 400)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status
    assert same_bits(phi.cpu().numpy(), want)
    buf = torch.zeros(g.n + 1, dtype=torch.float64, device="cuda")
    buf[1:] = dev(phi0)
    info = fx.cg_solve(g, dev(chi), dev(rho), buf[1:], 1e-9, 400)
    assert info.iterations == oinfo.iterations and same_bits(buf[1:].cpu().numpy(), want)


def test_cg_full_size_config3_200_iterations(fx, oracle):
    """config 3's fixed-200-iteration state, GPU against oracle, every bit of all 9.4 M unknowns (the oracle
    takes about 0.75 s per iteration on one host core)"""
    c = fi.config3()
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 0.0, 200)
    got, info = _solve(fx, c, tol=0.0, maxit=200)
    assert info.iterations == oinfo.iterations == 200 and info.status == oinfo.status == 1
    assert info.rel_residual == oinfo.rel_residual
    assert same_bits(got, want)


def test_cg_full_size_config3_first_iterations(fx, oracle):
    """config 3 at full size, the launch shape bench.py times; 6 iterations against the oracle, bit for bit"""
    c = fi.config3()
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 0.0, 6)
    got, info = _solve(fx, c, tol=0.0, maxit=6)
    assert info.iterations == oinfo.iterations == 6 and info.status == 1
    assert same_bits(got, want)


@pytest.mark.parametrize("mode", [0, 2, 3])
def test_cg_breakdown_and_maxit0(fx, oracle, mode):
    """an indefinite operator (chi < 0) must stop with FX_EBREAKDOWN at the same iteration as the oracle; maxit = 0"""
    fx.set_cg_fused(mode)
    c = fi.config0(N=8)
    og, g = oracle.Grid(**c["grid"]), fx.make_grid(**c["grid"])
    chi = -c["chi"]
    want, oinfo = oracle.cg_solve(og, chi, c["rho"], c["phi0"], 1e-10, 50)
    assert oinfo.status == oracle.EBREAKDOWN
    phi = dev(c["phi0"])
    with pytest.raises(fx.FxError):
        fx.cg_solve(g, dev(chi), dev(c["rho"]), phi, 1e-10, 50)
    info = fx.CGInfo()
    rc = fx.lib().fx_cg_solve(__import__("ctypes").byref(g), dev(chi).data_ptr(), dev(c["rho"]).data_ptr(), phi.zero_().data_ptr(), 1e-10, 50,
                              __import__("ctypes").byref(info))
    assert rc == fx.EBREAKDOWN and info.status == fx.EBREAKDOWN and info.iterations == oinfo.iterations
    phi = dev(c["phi0"])
    info = fx.cg_solve(g, dev(c["chi"]), dev(c["rho"]), phi, 1e-10, 0)
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 1e-10, 0)
    assert info.iterations == oinfo.iterations == 0 and info.status == oinfo.status == 1 and same_bits(phi.cpu().numpy(), want)


def test_argument_errors(fx):
    import ctypes
    import torch
    L = fx.lib()
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    assert L.fx_axpby(1.0, x.data_ptr(), 1.0, x.data_ptr(), -1) == fx.EINVAL
    assert L.fx_axpby(1.0, None, 1.0, x.data_ptr(), 8) == fx.EINVAL
    assert L.fx_axpby(1.0, None, 1.0, None, 0) == fx.OK                       # n == 0 is valid
    assert L.fx_pointwise_dot(1.0, x.data_ptr(), None, 0.0, x.data_ptr(), 8) == fx.EINVAL
    assert math.isnan(L.fx_exdot(None, x.data_ptr(), 8)) and b"bad arguments" in L.fx_last_error()
    g = fx.make_grid(2, 2, 1, 1.0, -1.0, 0, 1)
    assert L.fx_dg_weights(ctypes.byref(g), x.data_ptr(), None) == fx.EINVAL
    g = fx.make_grid(2, 2, 1, 1.0, 1.0, 0, 7)
    assert L.fx_cg_solve(ctypes.byref(g), x.data_ptr(), x.data_ptr(), x.data_ptr(), 1e-8, 10, None) == fx.EINVAL
    assert L.fx_set_launch(9, 0, 0) == fx.EINVAL and L.fx_set_launch(0, 0, 33) == fx.EINVAL and L.fx_set_cg_fused(7) == fx.EINVAL
    assert fx.exdot(x[:0], x[:0]) == 0.0 and math.copysign(1.0, fx.exdot(x[:0], x[:0])) == 1.0


def test_cg_host_entry(fx, oracle):
    c = fi.config0(N=8)
    og = oracle.Grid(**c["grid"])
    want, oinfo = oracle.cg_solve(og, c["chi"], c["rho"], c["phi0"], 1e-9, 2000)
    phi = c["phi0"].copy()
    info = fx.cg_solve_host(fx.make_grid(**c["grid"]), c["chi"], c["rho"], phi, 1e-9, 2000)
    assert info.iterations == oinfo.iterations and same_bits(phi, want)


# ---- weighted dot and exact sum ----------------------------------------------------

@pytest.mark.parametrize("n", [0, 1, 33, 1025, 100003, (1 << 21) + 3])
def test_weighted_dot_and_sum(fx, oracle, n):
    import torch
    x, y = fi.uniform(101, n), fi.uniform(102, n)
    w = 0.5 + fi.uniform(103, n) ** 2
    if n > 100:
        x[7] = 2.0 ** 600; y[7] = 2.0 ** 500; w[7] = 2.0 ** -300      # products outside the TwoProd range
        x[11] = 5e-324; y[11] = 3.0
    dx = dev(x) if n else dev(np.zeros(0))
    dw = dev(w) if n else dev(np.zeros(0))
    dy = dev(y) if n else dev(np.zeros(0))
    assert fbits(fx.exdot3(dx, dw, dy)) == fbits(oracle.exdot3(x, w, y) if n else 0.0)
    assert fbits(fx.exsum(dx)) == fbits(oracle.exsum(x) if n else 0.0)
    if n:
        ones = torch.ones(n, dtype=torch.float64, device="cuda")
        assert fbits(fx.exdot3(dx, ones, dy)) == fbits(fx.exdot(dx, dy))         # w == 1 reduces to the exact dot
        assert fbits(fx.exdot3(dx[1:], dw[1:], dy[1:])) == fbits(oracle.exdot3(x[1:], w[1:], y[1:]))   # unaligned


def test_weighted_dot_fig2_integral(fx, oracle):
    """Fig. 2: integral of exp(x) exp(y) over [0,2]^2, P = 3, 20 x 20 cells, as dot(f_x, volume, f_y)"""
    import torch
    g = fx.make_grid(20, 20, 3, 2.0, 2.0, 1, 1)
    W = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.dg_weights(g, W, None)
    xs, ys = oracle.dg_nodes(oracle.Grid(20, 20, 3, 2.0, 2.0, 1, 1))
    fxv = np.exp(np.broadcast_to(xs[None, :], (ys.size, xs.size))).ravel()
    fyv = np.exp(np.broadcast_to(ys[:, None], (ys.size, xs.size))).ravel()
    val = fx.exdot3(dev(fxv), W, dev(fyv))
    assert abs(val / (math.exp(2.0) - 1.0) ** 2 - 1.0) < 2e-12
    assert fbits(val) == fbits(oracle.exdot3(fxv, W.cpu().numpy(), fyv))


# ---- stand-alone dG derivatives ("dxdy") ------------------------------------------------

@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("direction", [0, 1])
def test_dg_derivative_bit_exact(fx, oracle, P, direction):
    import torch
    for (Nx, Ny) in [(1, 1), (2, 3), (31, 5), (33, 4), (64, 40), (70, 9)]:
        for bc in (0, 1):
            g, og = _grid(fx, oracle, Nx, Ny, P, bc, bc)
            x, y0 = fi.uniform(401 + P, g.n), fi.uniform(402 + P, g.n)
            for flux in (0, 1, 2, 3):                                  # forward, backward, centred flux; 3: the jump matrix
                for alpha, beta in ((1.0, 0.0), (0.7, -0.3)):
                    want = oracle.dg_derivative_canonical(og, direction, flux, alpha, x, beta, y0)
                    y = dev(y0) if beta != 0.0 else torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
                    fx.dg_derivative(g, direction, flux, alpha, dev(x), beta, y)
                    got = y.cpu().numpy()
                    assert np.array_equal(got, want), (Nx, Ny, P, bc, flux, alpha, np.abs(got - want).max())


@pytest.mark.parametrize("direction", [0, 1])
def test_dg_derivative_definition_shapes_and_full_size(fx, oracle, direction):
    import torch
    g, og = _grid(fx, oracle, 12, 9, 3, 0, 1)
    x, y0 = fi.uniform(411, g.n), fi.uniform(412, g.n)
    for flux in (0, 1, 2):
        ydef, scale = oracle.dg_derivative_definition(og, direction, flux, 0.7, x, -0.3, y0)
        for rows in (0, 1, 5, 1000):                                   # launch-shape invariance
            fx.set_launch(2, rows, 0)
            y = dev(y0)
            fx.dg_derivative(g, direction, flux, 0.7, dev(x), -0.3, y)
            got = y.cpu().numpy()
            assert np.all(np.abs(got - ydef) <= 1e-14 * scale)
            assert np.array_equal(got, oracle.dg_derivative_canonical(og, direction, flux, 0.7, x, -0.3, y0))
    fx.set_launch(2, 0, 0)
    c = fi.config4(3, 1024)                                            # 1024^2 cells, P = 3: the size the sweep times
    g, og = fx.make_grid(**c["grid"]), oracle.Grid(**c["grid"])
    y = dev(c["y"])
    fx.dg_derivative(g, direction, 2, 0.7, dev(c["x"]), -0.3, y)
    assert np.array_equal(y.cpu().numpy(), oracle.dg_derivative_canonical(og, direction, 2, 0.7, c["x"], -0.3, c["y"]))
    with pytest.raises(fx.FxError):
        fx.dg_derivative(g, direction, 0, 1.0, y, 0.0, y)


@pytest.mark.parametrize("n", [0, 1, 5, 1027, 8191, 8192, 8193, 100003, (1 << 22) + 9])
def test_exdot_f32(fx, oracle, n):
    """binary32 inputs, exact accumulation"""
    import torch
    x = fi.uniform(111, n).astype(np.float32); y = (fi.uniform(112, n) * 1e3).astype(np.float32)
    if n > 100:
        x[3] = np.float32(1e-45); y[3] = np.float32(1e-40); x[5] = np.float32(3e38); y[5] = np.float32(3e38)
    dx, dy = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    assert fbits(fx.exdot_f32(dx, dy)) == fbits(oracle.exdot_f32(x, y) if n else 0.0)
    if n > 4:
        assert fbits(fx.exdot_f32(dx[1:], dy[1:])) == fbits(oracle.exdot_f32(x[1:], y[1:]))      # 4-byte aligned only
        assert fbits(fx.exdot_f32(dx[2:], dy[2:])) == fbits(oracle.exdot_f32(x[2:], y[2:]))      # 8-byte aligned only
        for grid, block in [(1, 32), (9, 128)]:
            fx.set_launch(0, grid, block)
            assert fbits(fx.exdot_f32(dx, dy)) == fbits(oracle.exdot_f32(x, y)), (grid, block)
        fx.set_launch(0, 0, 0)


# ---- fused pointwise product and Arakawa bracket --------------------------------------------------------

@pytest.mark.parametrize("n", [1, 1023, 100003])
@pytest.mark.parametrize("gamma", [0.0, -0.4])
def test_pointwise_dot2_bit_exact(fx, oracle, n, gamma):
    a = [fi.uniform(501 + i, n) for i in range(5)]
    want = oracle.pointwise_dot2(0.7, a[0], a[1], -1.3, a[2], a[3], gamma, a[4])
    z = dev(a[4]) if gamma != 0.0 else dev(np.full(n, np.nan))
    got = fx.pointwise_dot2(0.7, dev(a[0]), dev(a[1]), -1.3, dev(a[2]), dev(a[3]), gamma, z).cpu().numpy()
    assert same_bits(got, want)
    zz = dev(a[0])                                                     # everything aliased
    assert same_bits(fx.pointwise_dot2(0.5, zz, zz, 2.0, zz, zz, 1.0, zz).cpu().numpy(), oracle.pointwise_dot2(0.5, a[0], a[0], 2.0, a[0], a[0], 1.0, a[0]))


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_arakawa_bit_exact(fx, oracle, P):
    """the nine-call oracle against the two tile kernels (even pitch; every launch shape) and the seven-launch fallback"""
    import torch
    for (Nx, Ny, bcx, bcy) in [(1, 1, 0, 0), (7, 5, 0, 1), (33, 12, 1, 0), (64, 40, 0, 0), (2, 2, 1, 1), (62, 9, 1, 1), (34, 7, 0, 1),
                               (120, 5, 1, 0), (250, 12, 0, 0)]:
        g, og = _grid(fx, oracle, Nx, Ny, P, bcx, bcy)
        f, gg = fi.uniform(511 + P, g.n), fi.uniform(512 + P, g.n)
        want = oracle.arakawa(og, f, gg)
        for path, rows in ((0, 0), (0, 1), (0, 3), (1, 0)):
            fx.set_dg_path(path); fx.set_launch(2, rows, 0)
            out = torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
            fx.arakawa(g, dev(f), dev(gg), out)
            assert same_bits(out.cpu().numpy(), want), (Nx, Ny, P, path, rows)
    fx.set_dg_path(0); fx.set_launch(2, 0, 0)
    g, og = _grid(fx, oracle, 256, 256, 3, 0, 0, 2 * math.pi, 2 * math.pi)      # conservation on the GPU result
    xs, ys = oracle.dg_nodes(og)
    X, Y = np.meshgrid(xs, ys)
    f, gg = (np.sin(X) * np.cos(Y)).ravel(), (np.cos(X) * np.sin(2 * Y)).ravel()
    out = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.arakawa(g, dev(f), dev(gg), out)
    W = torch.empty_like(out)
    fx.dg_weights(g, W, None)
    scale = float((W * out.abs()).sum())
    assert abs(fx.exdot(W, out)) < 1e-12 * scale and abs(fx.exdot3(dev(f), W, out)) < 1e-12 * scale
    assert np.array_equal(out.cpu().numpy(), oracle.arakawa(og, f, gg))


# ---- Neumann and mixed walls (Q23, 6.9) ------------------------------------------------------

PER, DIR, NEU, DIR_NEU, NEU_DIR = 0, 1, 2, 3, 4
NEUBCS = [(2, 2), (2, 0), (0, 2), (1, 2), (2, 1), (3, 4), (4, 3), (3, 0), (0, 4), (4, 2), (1, 3)]


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("bc", NEUBCS)
@pytest.mark.parametrize("path", [0, 1])
def test_dg_apply_neumann_bit_exact(fx, oracle, P, bc, path):
    import torch
    fx.set_dg_path(path)
    for (Nx, Ny) in [(1, 1), (2, 3), (3, 2), (31, 5), (30, 9), (61, 17), (64, 33), (62, 4)]:
        if (bc[0] == DIR_NEU and Nx < 2) or (bc[1] == DIR_NEU and Ny < 2):
            with pytest.raises(Exception):
                fx.dg_elliptic_apply(fx.make_grid(Nx, Ny, P, 1.0, 1.0, *bc), dev(np.ones(Nx * Ny * P * P)), dev(np.ones(Nx * Ny * P * P)),
                                     torch.empty(Nx * Ny * P * P, dtype=torch.float64, device="cuda"))
            continue
        g, og = _grid(fx, oracle, Nx, Ny, P, *bc)
        x = fi.uniform(151 + P, g.n); chi = 1.0 + 0.5 * fi.uniform(161 + P, g.n)
        for sym in (True, False):
            want = oracle.dg_apply_canonical(og, chi, x, normed=not sym)
            y = torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
            fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=sym)
            got = y.cpu().numpy()
            assert np.array_equal(got, want), (Nx, Ny, P, bc, sym, np.abs(got - want).max())
            assert same_bits(got, want), (Nx, Ny, P, bc, sym)


def test_dg_apply_neumann_definition_shapes_and_null_space(fx, oracle):
    import torch
    g, og = _grid(fx, oracle, 95, 40, 3, NEU, DIR_NEU)
    x = fi.uniform(171, g.n); chi = 1.0 + 0.5 * fi.uniform(172, g.n)
    want = oracle.dg_apply_canonical(og, chi, x, normed=False)
    for rows, block in [(0, 0), (1, 32), (3, 64), (7, 128), (40, 128), (1000, 1024)]:
        fx.set_launch(2, rows, block)
        y = torch.empty(g.n, dtype=torch.float64, device="cuda")
        fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=True)
        assert np.array_equal(y.cpu().numpy(), want), (rows, block)
    fx.set_launch(2, 0, 0)
    g, og = _grid(fx, oracle, 12, 9, 4, NEU_DIR, NEU)
    x = fi.uniform(173, g.n); chi = 1.0 + 0.5 * fi.uniform(174, g.n)
    ydef, scale = oracle.dg_apply_definition(og, chi, x, normed=False)
    y = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.dg_elliptic_apply(g, dev(chi), dev(x), y, sym=True)
    assert np.all(np.abs(y.cpu().numpy() - ydef) <= 1e-14 * scale)
    # pure Neumann: constants are in the null space (to rounding of the in-cell derivative of 1)
    g, og = _grid(fx, oracle, 64, 48, 3, NEU, NEU)
    chi = 1.0 + 0.5 * fi.uniform(175, g.n)
    y = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.dg_elliptic_apply(g, dev(chi), dev(np.ones(g.n)), y, sym=True)
    assert np.abs(y.cpu().numpy()).max() < 1e-12
    # derivatives and the bracket take PER / DIR only
    with pytest.raises(Exception):
        fx.dg_derivative(g, 0, 0, 1.0, dev(np.ones(g.n)), 0.0, y)
    with pytest.raises(Exception):
        fx.arakawa(g, dev(np.ones(g.n)), dev(np.ones(g.n)), y)


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
@pytest.mark.parametrize("Nx,Ny,P,bc", [(16, 16, 3, (NEU, DIR)), (33, 7, 5, (DIR_NEU, NEU_DIR)), (7, 5, 1, (DIR, NEU)),
                                        (61, 4, 2, (NEU_DIR, NEU)), (40, 35, 4, (NEU, DIR_NEU)), (64, 64, 3, (PER, NEU_DIR))])
def test_cg_neumann_matches_oracle(fx, oracle, mode, Nx, Ny, P, bc):
    """every driver (unfused, automatic, two-kernel, persistent requested) gives the oracle's iterates bit for bit"""
    fx.set_cg_fused(mode)
    grid = dict(Nx=Nx, Ny=Ny, P=P, lx=math.pi, ly=1.7, bcx=bc[0], bcy=bc[1])
    g, og = fx.make_grid(**grid), oracle.Grid(**grid)
    chi = 1.0 + 0.5 * fi.uniform(191, g.n); rho = fi.uniform(192, g.n); phi0 = 0.01 * fi.uniform(193, g.n)
    want, oinfo = oracle.cg_solve(og, chi, rho, phi0, 1e-9, 600)
    phi = dev(phi0)
    info = fx.cg_solve(g, dev(chi), dev(rho), phi, 1e-9, 600)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status
    assert same_bits(phi.cpu().numpy(), want)


def test_cg_neumann_manufactured_solution(fx, oracle):
    """phi = cos x sin(y/2) on [0,pi]^2: zero normal derivative at x = 0, pi (NEU) and y = pi, zero value at y = 0 (DIR_NEU)"""
    P, N = 3, 48
    g = fx.make_grid(N, N, P, math.pi, math.pi, NEU, DIR_NEU)
    og = oracle.Grid(N, N, P, math.pi, math.pi, NEU, DIR_NEU)
    xs, ys = oracle.dg_nodes(og)
    X, Y = np.meshgrid(xs, ys)
    chi = 1 + 0.5 * np.cos(X) * np.cos(Y)
    phi_exact = np.cos(X) * np.sin(Y / 2)
    rho = (-0.5 * np.sin(X) * np.cos(Y)) * (-np.sin(X)) * np.sin(Y / 2) + chi * (-np.cos(X)) * np.sin(Y / 2) \
        + (-0.5 * np.cos(X) * np.sin(Y)) * np.cos(X) * np.cos(Y / 2) / 2 + chi * np.cos(X) * (-np.sin(Y / 2) / 4)
    phi = dev(np.zeros(g.n))
    info = fx.cg_solve(g, dev(chi.ravel()), dev(rho.ravel()), phi, 1e-11, 5000)
    assert info.status == 0
    W, _ = oracle.dg_weights(og)
    e = phi.cpu().numpy() - phi_exact.ravel()
    rel = math.sqrt(oracle.exdot(W * e, e) / oracle.exdot(W * phi_exact.ravel(), phi_exact.ravel()))
    assert rel < 2e-6, rel                 # 1.04e-6 with the oracle; order P


@pytest.mark.parametrize("n", [4095, 4096, 4097, 4098, 4099, 70001, (1 << 22) + 1])
def test_exsum_two_half_path(fx, oracle, n):
    """long vectors are summed as two halves through the dot kernel's ring plus a <= 3-element tail"""
    x = fi.uniform(111, n) * np.ldexp(1.0, fi.rng(112).integers(-200, 200, n))
    want = oracle.exsum(x)
    dx = dev(x)
    assert fbits(fx.exsum(dx)) == fbits(want)
    buf = dev(np.concatenate([[0.0], x]))
    assert fbits(fx.exsum(buf[1:])) == fbits(want)                         # only 8-byte aligned
    for grid, block in [(1, 32), (7, 64), (300, 256)]:
        fx.set_launch(0, grid, block)
        assert fbits(fx.exsum(dx)) == fbits(want), (grid, block)
    fx.set_launch(0, 0, 0)
    # cancellation and specials through the same path
    z = np.concatenate([x, -x]); fi.rng(113).shuffle(z)
    assert fx.exsum(dev(z)) == 0.0
    z[5] = np.inf
    assert fx.exsum(dev(z)) == np.inf
    z[n] = -np.inf
    assert math.isnan(fx.exsum(dev(z)))


def test_exsum_multi_launch(fx, oracle):
    n = (1 << 28) + 5                                                       # two ring launches of 2^27 pairs ... and a tail
    import torch
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    x = torch.rand(n, dtype=torch.float64, device="cuda", generator=g) - 0.5
    got = fx.exsum(x)
    # the oracle over the same values, in four host chunks (the exact sum is order-free: compare through the exact dot with ones)
    want = oracle.exsum(x.cpu().numpy())
    assert fbits(got) == fbits(want)


def test_exdot_f32_widening_cases(fx, oracle):
    """every class of binary32 value through the kernel's integer widening: subnormals, both zeros, extremes, inf, nan"""
    import torch
    r = fi.rng(121)
    n = 50001                                                  # long enough for the ring path (float pairs in 8-byte slots)
    bitsx = r.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
    bitsy = r.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
    for b in (bitsx, bitsy):                                   # no inf / nan in the bulk
        e = (b >> 23) & 0xff
        b[e == 0xff] &= np.uint32(0xbfffffff)
    bitsx[:2000] &= np.uint32(0x807fffff)                      # 2000 subnormals and zeros of either sign
    bitsy[1000:3000] &= np.uint32(0x807fffff)
    bitsx[3000] = 0x80000000; bitsy[3001] = 0x00000001; bitsx[3002] = 0x7f7fffff; bitsy[3002] = 0xff7fffff
    x = bitsx.view(np.float32).copy(); y = bitsy.view(np.float32).copy()
    with np.errstate(all="ignore"):
        want = oracle.exdot_f32(x, y)
    got = fx.exdot_f32(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda())
    assert fbits(got) == fbits(want)
    x[7] = np.inf; y[7] = np.float32(-2.0)
    assert fx.exdot_f32(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()) == -np.inf
    y[9] = np.nan
    assert math.isnan(fx.exdot_f32(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()))


# ---- 3-D product grids (Q24) -----------------------------------------------------------------------
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("P,bc,Nx,Ny,Nz", [(1, (0, 1), 8, 6, 3), (2, (1, 0), 31, 5, 4), (3, (0, 1), 64, 24, 5), (3, (1, 1), 62, 9, 2),
                                           (4, (2, 1), 30, 7, 3), (5, (3, 4), 12, 6, 2), (3, (0, 0), 250, 5, 3)])
def test_dg3_apply_and_weights_bit_exact(fx, oracle, P, bc, Nx, Ny, Nz, path):
    import torch
    fx.set_dg_path(path)
    g = fx.make_grid3(Nx, Ny, Nz, P, 2 * math.pi, 3.0, 1.7, *bc)
    og = oracle.Grid3(Nx, Ny, Nz, P, 2 * math.pi, 3.0, 1.7, *bc)
    x = fi.uniform(191 + P, g.n); chi = 1.0 + 0.5 * fi.uniform(192 + P, g.n)
    w = torch.empty(g.n, dtype=torch.float64, device="cuda"); v = torch.empty_like(w)
    fx.dg3_weights(g, w, v)
    W, V = oracle.dg3_weights(og)
    assert same_bits(w.cpu().numpy(), W) and same_bits(v.cpu().numpy(), V)
    for sym in (True, False):
        want = oracle.dg3_apply_canonical(og, chi, x, normed=not sym)
        for rows in (0, 2):
            fx.set_launch(2, rows, 0)
            y = torch.full((g.n,), float("nan"), dtype=torch.float64, device="cuda")
            fx.dg3_elliptic_apply(g, dev(chi), dev(x), y, sym=sym)
            assert same_bits(y.cpu().numpy(), want), (sym, rows)
        fx.set_launch(2, 0, 0)
    ydef, scale = oracle.dg3_apply_definition(og, chi, x, normed=False)
    y = torch.empty(g.n, dtype=torch.float64, device="cuda")
    fx.dg3_elliptic_apply(g, dev(chi), dev(x), y, sym=True)
    assert np.all(np.abs(y.cpu().numpy() - ydef) <= 1e-14 * scale)


@pytest.mark.parametrize("mode,path", [(0, 0), (1, 0), (2, 0), (2, 2), (3, 1)])
@pytest.mark.parametrize("P,bc,Nx,Ny,Nz", [(3, (0, 1), 16, 12, 4), (2, (1, 1), 34, 9, 3), (5, (1, 0), 12, 6, 2)])
def test_cg3_matches_oracle(fx, oracle, P, bc, Nx, Ny, Nz, mode, path):
    """one PCG over all planes: every driver (unfused, persistent, two fused kernels on either stencil) gives the oracle's bits"""
    fx.set_cg_fused(mode); fx.set_dg_path(path)
    g = fx.make_grid3(Nx, Ny, Nz, P, 2 * math.pi, 2.0, 1.1, *bc)
    og = oracle.Grid3(Nx, Ny, Nz, P, 2 * math.pi, 2.0, 1.1, *bc)
    chi = 1.0 + 0.5 * fi.uniform(195, g.n); rho = fi.uniform(196, g.n); phi0 = 0.1 * fi.uniform(197, g.n)
    want, oinfo = oracle.cg3_solve(og, chi, rho, phi0, 1e-9, 4000)
    phi = dev(phi0)
    info = fx.cg3_solve(g, dev(chi), dev(rho), phi, 1e-9, 4000)
    assert info.iterations == oinfo.iterations and info.status == oinfo.status == 0
    assert info.rel_residual == oinfo.rel_residual
    assert same_bits(phi.cpu().numpy(), want)
    want, oinfo = oracle.cg3_solve(og, chi, rho, phi0, 0.0, 17)
    phi = dev(phi0)
    info = fx.cg3_solve(g, dev(chi), dev(rho), phi, 0.0, 17)
    assert info.iterations == 17 and info.status == 1 and same_bits(phi.cpu().numpy(), want)


def test_cg3_larger_grid(fx, oracle):
    """128 x 128 cells x 8 planes, P = 3 (1.2 M unknowns: the two-kernel loop at its default launch shapes), 30 iterations"""
    g = fx.make_grid3(128, 128, 8, 3, 2 * math.pi, 2 * math.pi, 2 * math.pi, 1, 1)
    og = oracle.Grid3(128, 128, 8, 3, 2 * math.pi, 2 * math.pi, 2 * math.pi, 1, 1)
    chi = 1.0 + 0.5 * fi.uniform(198, g.n); rho = fi.uniform(199, g.n)
    want, oinfo = oracle.cg3_solve(og, chi, rho, np.zeros(g.n), 0.0, 30)
    phi = dev(np.zeros(g.n))
    info = fx.cg3_solve(g, dev(chi), dev(rho), phi, 0.0, 30)
    assert info.iterations == oinfo.iterations == 30 and info.rel_residual == oinfo.rel_residual
    assert same_bits(phi.cpu().numpy(), want)
