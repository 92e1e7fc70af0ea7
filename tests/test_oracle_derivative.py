"""Pins for the oracle's stand-alone dG derivatives ("dxdy"; Q21): polynomial exactness,
adjointness / skew-symmetry in the dG weights, the P = 1 finite-difference special cases, convergence on sin, and
agreement of the canonical fp64 order with the 113-bit explicit-matrix definition."""
import math

import numpy as np
import pytest

import fxinputs as fi

FWD, BWD, CTR = 0, 1, 2


def _w1d(oracle, N, P, h):
    t = oracle.dg_tables(P)
    return np.tile(t["w"], N) * h / 2


def _nodes(oracle, N, P, h):
    t = oracle.dg_tables(P)
    return (h * (np.arange(N)[:, None] + (1 + t["xi"][None, :]) / 2)).ravel()


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("flux", [FWD, BWD, CTR])
def test_polynomial_exactness_in_interior_cells(oracle, P, flux):
    """degree < P polynomials are differentiated exactly away from the boundary cells (any flux, any bc)"""
    N, h = 7, 0.3
    x = _nodes(oracle, N, P, h)
    for bc in (0, 1):
        M = oracle.dg_derivative_matrix_1d(N, P, h, bc, flux)
        for deg in range(P):
            u, du = x ** deg, deg * x ** max(deg - 1, 0) if deg else np.zeros_like(x)
            got = M @ u
            inner = slice(P, (N - 1) * P)
            assert np.max(np.abs(got[inner] - du[inner])) < 1e-11 * max(1.0, np.max(np.abs(du))), (bc, deg)
    if P >= 2 and flux != CTR:                   # degree P is NOT exact for one-sided fluxes: the test above can fail
        M = oracle.dg_derivative_matrix_1d(N, P, h, 0, flux)
        assert np.max(np.abs((M @ x ** P)[P:(N - 1) * P] - P * x[P:(N - 1) * P] ** (P - 1))) > 1e-6


@pytest.mark.parametrize("P", [1, 2, 3, 5])
@pytest.mark.parametrize("bc", [0, 1])
def test_adjointness_and_skew_symmetry(oracle, P, bc):
    """backward = -W^-1 forward^T W (the definition, Q21); centred = mean; periodic centred is W-skew"""
    N, h = 5, 0.7
    W = np.diag(_w1d(oracle, N, P, h))
    F, B, C = (oracle.dg_derivative_matrix_1d(N, P, h, bc, f) for f in (FWD, BWD, CTR))
    assert np.allclose(W @ B, -(W @ F).T, rtol=0, atol=1e-13 * np.abs(F).max())
    assert np.allclose(C, (F + B) / 2, rtol=0, atol=1e-15 * np.abs(F).max())
    assert np.allclose(W @ C, -(W @ C).T, rtol=0, atol=1e-13 * np.abs(F).max())      # skew for both bc (C = (F - F^*)/2)
    if bc == 0:
        assert np.allclose(F @ np.ones(N * P), 0, atol=1e-12) and np.allclose(B @ np.ones(N * P), 0, atol=1e-12)


def test_p1_is_finite_differences(oracle):
    N, h = 6, 0.25
    F = oracle.dg_derivative_matrix_1d(N, 1, h, 0, FWD)
    B = oracle.dg_derivative_matrix_1d(N, 1, h, 0, BWD)
    C = oracle.dg_derivative_matrix_1d(N, 1, h, 0, CTR)
    I = np.eye(N)
    assert np.allclose(F, (np.roll(I, 1, axis=1) - I) / h)              # (u_{i+1} - u_i)/h
    assert np.allclose(B, (I - np.roll(I, -1, axis=1)) / h)             # (u_i - u_{i-1})/h
    assert np.allclose(C, (np.roll(I, 1, axis=1) - np.roll(I, -1, axis=1)) / (2 * h))


@pytest.mark.parametrize("P", [2, 3, 4])
def test_convergence_on_sine(oracle, P):
    """L2 error of d/dx sin on a periodic grid falls like h^(P-1): one order below the approximation order P of the
    function itself (the derivative of the degree-(P-1) interpolant)"""
    errs = []
    for N in (8, 16, 32):
        h = 2 * math.pi / N
        x = _nodes(oracle, N, P, h)
        w = _w1d(oracle, N, P, h)
        M = oracle.dg_derivative_matrix_1d(N, P, h, 0, CTR)
        errs.append(math.sqrt(np.sum(w * (M @ np.sin(x) - np.cos(x)) ** 2)))
    order = math.log2(errs[1] / errs[2])
    assert P - 1 - 0.4 < order < P + 0.6 and errs[2] < errs[0]


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("direction", [0, 1])
def test_canonical_matches_definition(oracle, P, direction):
    for flux in (FWD, BWD, CTR):
        for bc in (0, 1):
            g = oracle.Grid(6, 5, P, 1.3, 0.9, bc, bc)
            x, y = fi.uniform(301 + P, g.n), fi.uniform(302 + P, g.n)
            for alpha, beta in ((1.0, 0.0), (0.7, -0.3)):
                want, scale = oracle.dg_derivative_definition(g, direction, flux, alpha, x, beta, y)
                got = oracle.dg_derivative_canonical(g, direction, flux, alpha, x, beta, y)
                assert np.all(np.abs(got - want) <= 1e-14 * scale + 1e-300), (flux, bc, alpha)


def test_matrix_matches_2d_application(oracle):
    """index layout: the 2-D canonical derivative along x / y equals the 1-D matrix applied to rows / columns"""
    P, Nx, Ny = 3, 4, 5
    g = oracle.Grid(Nx, Ny, P, 2.0, 3.0, 0, 1)
    x = fi.uniform(311, g.n)
    X = x.reshape(Ny * P, Nx * P)
    Mx = oracle.dg_derivative_matrix_1d(Nx, P, 2.0 / Nx, 0, FWD)
    My = oracle.dg_derivative_matrix_1d(Ny, P, 3.0 / Ny, 1, BWD)
    gx = oracle.dg_derivative_canonical(g, 0, FWD, 1.0, x, 0.0, np.zeros(g.n)).reshape(X.shape)
    gy = oracle.dg_derivative_canonical(g, 1, BWD, 1.0, x, 0.0, np.zeros(g.n)).reshape(X.shape)
    assert np.allclose(gx, X @ Mx.T, atol=1e-12) and np.allclose(gy, My @ X, atol=1e-12)


# ---- fused pointwise product and the Arakawa bracket (Q22) ----------------------------------

def test_pointwise_dot2_pins(oracle):
    from fractions import Fraction
    rng = fi.rng(777)
    n = 300
    ints = lambda: rng.integers(-50, 50, n).astype(float)           # small integers: no rounding anywhere
    x1, y1, x2, y2, z = ints(), ints(), ints(), ints(), ints()
    got = oracle.pointwise_dot2(2.0, x1, y1, -3.0, x2, y2, 5.0, z)
    assert np.array_equal(got, 2 * x1 * y1 - 3 * x2 * y2 + 5 * z)
    assert np.array_equal(oracle.pointwise_dot2(2.0, x1, y1, -3.0, x2, y2, 0.0, np.full(n, np.nan)), 2 * x1 * y1 - 3 * x2 * y2)
    # reduces to pointwise_dot when beta = 0 (b*y2 = 0 exactly, fma(a, y1, 0 or RN(gamma z)))
    u, v, w = fi.uniform(1, n), fi.uniform(2, n), fi.uniform(3, n)
    assert np.array_equal(oracle.pointwise_dot2(0.7, u, v, 0.0, u, v, -0.3, w), oracle.pointwise_dot(0.7, u, v, -0.3, w))


@pytest.mark.parametrize("P", [2, 3, 4])
def test_arakawa_converges_and_conserves(oracle, P):
    """{f,g} -> analytic Poisson bracket with order ~P-1; Arakawa's conservation: int J = int f J = int g J = 0 (periodic)"""
    errs = []
    for N in (8, 16, 32):
        g = oracle.Grid(N, N, P, 2 * math.pi, 2 * math.pi, 0, 0)
        xs, ys = oracle.dg_nodes(g)
        X, Y = np.meshgrid(xs, ys)
        f, gg = np.sin(X) * np.cos(Y), np.cos(X) * np.sin(2 * Y) + 0.3 * np.sin(X + Y)
        fx_, fy_ = np.cos(X) * np.cos(Y), -np.sin(X) * np.sin(Y)
        gx_, gy_ = -np.sin(X) * np.sin(2 * Y) + 0.3 * np.cos(X + Y), 2 * np.cos(X) * np.cos(2 * Y) + 0.3 * np.cos(X + Y)
        exact = (fx_ * gy_ - fy_ * gx_).ravel()
        J = oracle.arakawa(g, f.ravel(), gg.ravel())
        W, _ = oracle.dg_weights(g)
        errs.append(math.sqrt(np.sum(W * (J - exact) ** 2) / np.sum(W * exact ** 2)))
        scale = np.sum(W * np.abs(J))
        assert abs(oracle.exdot(W, J)) < 1e-12 * scale                                   # int {f,g} = 0
        assert abs(oracle.exdot3(f.ravel(), W, J)) < 1e-12 * scale                       # int f {f,g} = 0
        assert abs(oracle.exdot3(gg.ravel(), W, J)) < 1e-12 * scale                      # int g {f,g} = 0
        Jr = oracle.arakawa(g, gg.ravel(), f.ravel())
        assert np.max(np.abs(J + Jr)) < 1e-12 * np.max(np.abs(J))                        # antisymmetry
    assert errs[2] < errs[1] < errs[0] and math.log2(errs[1] / errs[2]) > P - 1.5


# ---- the stand-alone jump matrix (flux code 3; "y <- alpha M x + beta y" for dx, dy and jump) -----------
JUMP = 3


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("bc", [0, 1])
def test_jump_is_the_sum_of_squared_face_jumps(oracle, P, bc):
    """x^T J x = sum over the faces of (trace from the right - trace from the left)^2, traces evaluated independently with
    numpy from the Lagrange end values; J symmetric, positive semi-definite, J 1 = 0 on a periodic line"""
    N, h = 7, 0.3
    J = oracle.dg_derivative_matrix_1d(N, P, h, bc, JUMP)
    t = oracle.dg_tables(P)
    assert np.allclose(J, J.T, atol=1e-15)
    ev = np.linalg.eigvalsh(J)
    assert ev.min() > -1e-13
    x = fi.uniform(331 + P, N * P)
    X = x.reshape(N, P)
    tl, tr = X @ t["L"], X @ t["R"]                       # left / right end value of every cell
    if bc == 0:
        jumps = tl[np.arange(1, N + 1) % N] - tr          # face between cell n and n+1 (periodic)
    else:
        jumps = np.concatenate([[tl[0] - 0.0], tl[1:] - tr[:-1], [0.0 - tr[-1]]])      # walls: jump against the zero boundary value
    assert abs(x @ J @ x - np.sum(jumps ** 2)) <= 1e-12 * np.sum(jumps ** 2)
    if bc == 0:
        assert np.abs(J @ np.ones(N * P)).max() <= 1e-14
    if P == 1:                                            # piecewise constants: the second-difference matrix
        want = 2 * np.eye(N) - np.eye(N, k=1) - np.eye(N, k=-1)
        if bc == 0:
            want[0, -1] -= 1; want[-1, 0] -= 1
        assert np.allclose(J, want, atol=1e-15)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("direction", [0, 1])
def test_jump_canonical_matches_definition_and_matrix(oracle, P, direction):
    for bc in (0, 1):
        g = oracle.Grid(6, 5, P, 1.3, 0.9, bc, bc)
        x, y = fi.uniform(341 + P, g.n), fi.uniform(342 + P, g.n)
        for alpha, beta in ((1.0, 0.0), (0.7, -0.3)):
            want, scale = oracle.dg_derivative_definition(g, direction, JUMP, alpha, x, beta, y)
            got = oracle.dg_derivative_canonical(g, direction, JUMP, alpha, x, beta, y)
            assert np.all(np.abs(got - want) <= 1e-14 * scale + 1e-300), (bc, alpha)
        N = g.Nx if direction == 0 else g.Ny
        J = oracle.dg_derivative_matrix_1d(N, P, 1.0, bc, JUMP)           # (no h in the un-normed jump)
        X = x.reshape(g.Ny * P, g.Nx * P)
        got = oracle.dg_derivative_canonical(g, direction, JUMP, 1.0, x, 0.0, np.zeros(g.n)).reshape(X.shape)
        assert np.allclose(got, X @ J.T if direction == 0 else J @ X, atol=1e-12)


def test_jump_is_the_elliptic_operators_penalty(oracle):
    """S - (the two flux terms) = diag(Wy) (x) Jx + Jy (x) diag(Wx): with chi = 0 the elliptic operator IS the weighted jumps"""
    P = 3
    g = oracle.Grid(5, 4, P, 1.7, 2.3, 0, 1)
    x = fi.uniform(351, g.n)
    S0 = oracle.dg_apply_canonical(g, np.zeros(g.n), x, normed=False)
    jx = oracle.dg_derivative_canonical(g, 0, JUMP, 1.0, x, 0.0, np.zeros(g.n)).reshape(g.Ny * P, g.Nx * P)
    jy = oracle.dg_derivative_canonical(g, 1, JUMP, 1.0, x, 0.0, np.zeros(g.n)).reshape(g.Ny * P, g.Nx * P)
    w = oracle.dg_tables(P)["w"]
    Wx = np.tile(w, g.Nx) * (1.7 / 5) / 2; Wy = np.tile(w, g.Ny) * (2.3 / 4) / 2
    want = Wy[:, None] * jx + Wx[None, :] * jy
    assert np.allclose(S0.reshape(want.shape), want, atol=1e-13 * np.abs(want).max())
