"""Pins of the oracle's Gauss-Legendre tables, dG elliptic operator and vector primitives (CPU only).

The paper names the discretisation only by reference; the reading is DESIGN.md
section 3.3.  What pins it: textbook closed forms of the GL rule, the algebraic identities of the
reference element, polynomial exactness of the derivative, symmetry / definiteness of S, the P=1
five-point stencil, agreement of two independent evaluations (explicit 113-bit matrices vs the
canonical fp64 order), and a dense numpy assembly from the 1-D matrices.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import fxinputs as fi
from conftest import golden_path

PER, DIR = 0, 1
BCS = [(PER, PER), (PER, DIR), (DIR, PER), (DIR, DIR)]


# ---------------------------------------------------------------- tables
def test_gl_closed_forms(oracle):
    rows = [l.split() for l in open(golden_path("gauss_legendre_closed_forms.txt")) if not l.startswith("#")]
    for P in range(1, 6):
        t = oracle.dg_tables(P)
        mine = [(r[2], r[3]) for r in rows if int(r[0]) == P]
        assert len(mine) == P
        for k, (xs, ws) in enumerate(mine):
            # correctly rounded doubles of the 40-digit closed forms (Fraction -> float is exact RN)
            assert t["xi"][k] == float(Fraction(xs)), (P, k)
            assert t["w"][k] == float(Fraction(ws)), (P, k)


@pytest.mark.parametrize("P", range(1, 6))
def test_reference_element_identities(oracle, P):
    t = oracle.dg_tables(P)
    w, L, R, D = t["w"], t["L"], t["R"], t["D"]
    eps = 4e-15
    assert abs(w.sum() - 2) < eps and abs(L.sum() - 1) < eps and abs(R.sum() - 1) < eps
    assert np.allclose(D.sum(axis=1), 0, atol=eps * 10)
    assert np.allclose(R, L[::-1], atol=0)                      # mirror symmetry, exact after rounding
    assert np.allclose(D, -D[::-1, ::-1], atol=0)
    # summation by parts: w_k D[k][m] + w_m D[m][k] = R_k R_m - L_k L_m
    sbp = w[:, None] * D + (w[:, None] * D).T - (np.outer(R, R) - np.outer(L, L))
    assert np.abs(sbp).max() < 20 * eps
    # quadrature exact for monomials up to degree 2P-1
    for d in range(2 * P):
        exact = 0.0 if d % 2 else 2.0 / (d + 1)
        assert abs(np.dot(w, t["xi"] ** d) - exact) < eps
    # D differentiates, L/R evaluate, polynomials of degree < P exactly at the nodes / ends
    for d in range(P):
        v = t["xi"] ** d
        dv = d * t["xi"] ** max(d - 1, 0) if d else np.zeros(P)
        assert np.abs(D @ v - dv).max() < 50 * eps
        assert abs(L @ v - (-1.0) ** d) < 20 * eps and abs(R @ v - 1.0) < 20 * eps
    # derived tables
    assert np.allclose(t["B"], R / w, rtol=4e-16, atol=0)
    assert np.allclose(t["T0"], D - np.outer(R, R) / w[:, None], rtol=0, atol=20 * eps)
    assert np.allclose(t["T0L"], t["T0"] + np.outer(L, L) / w[:, None], rtol=0, atol=20 * eps)
    assert np.allclose(t["WW"], np.outer(w, w), rtol=4e-16, atol=0)
    if P == 1:
        assert D[0, 0] == 0 and L[0] == 1 and R[0] == 1 and w[0] == 2


# ---------------------------------------------------------------- 1-D derivative and jump
@pytest.mark.parametrize("P", range(1, 6))
def test_derivative_polynomial_exactness(oracle, P):
    N, length = 6, 2.0
    h = length / N
    F, _ = oracle.dg_matrix_1d(N, P, h, PER)
    g = oracle.Grid(N, 1, P, length, 1.0, PER, PER)
    xs, _ = oracle.dg_nodes(g)
    for d in range(P + 1):
        u = xs ** d
        du = d * xs ** max(d - 1, 0) if d else np.zeros_like(xs)
        err = np.abs(F @ u - du)[: (N - 1) * P].max()          # interior cells (the last one sees the periodic wrap)
        if d < P:
            assert err < 1e-11, (P, d, err)                     # exact for degree < P
        elif P > 1:                                             # (P=1: the forward difference of x is exact, skip)
            assert err > 1e-4, (P, d, err)                      # and not for degree P: the scheme really has P coefficients


@pytest.mark.parametrize("P", range(1, 5))
def test_derivative_dirichlet_rows(oracle, P):
    # DIR: ghost traces are zero.  For u == 1 the interior cells give 0, the boundary cells see the jump to 0.
    N, h = 5, 0.3
    F, J = oracle.dg_matrix_1d(N, P, h, DIR)
    one = np.ones(N * P)
    d = F @ one
    assert np.abs(d[P:(N - 1) * P]).max() < 1e-12
    assert np.abs(d[(N - 1) * P:]).max() > 0.1
    t = oracle.dg_tables(P)
    # integrated against the weights the last cell carries exactly -u(right) : sum_k (h/2) w_k d_k = -1
    assert abs(np.dot(h / 2 * t["w"], d[(N - 1) * P:]) + 1.0) < 1e-12
    # first cell: the +LL^T term replaces the interior trace by the boundary value 0 -> jump 0 -> 1 : integral +1
    assert abs(np.dot(h / 2 * t["w"], d[:P]) - 1.0) < 1e-12
    # so that the derivative of a function vanishing at both ends integrates to u(b) - u(a) = 0 overall
    assert abs(np.dot(np.tile(h / 2 * t["w"], N), d)) < 1e-12
    # jump matrix: symmetric, PSD, constants in its null space iff periodic
    assert np.abs(J - J.T).max() == 0
    assert np.linalg.eigvalsh(J).min() > -1e-12
    _, Jp = oracle.dg_matrix_1d(N, P, h, PER)
    assert np.abs(Jp @ one).max() < 1e-13 and np.abs(J @ one).max() > 0.5
    if P == 1:   # bidiagonal (-1,+1)/h with first row (0,+1) and last row (..,0,-1)
        exp = (np.diag(-np.ones(N)) + np.diag(np.ones(N - 1), 1)) / h
        exp[0, 0] = 0.0
        assert np.allclose(F, exp, atol=1e-14)


# ---------------------------------------------------------------- 2-D operator: dense assembly in numpy
def assemble_S(oracle, g, chi):
    """S = Fx^T diag(W chi) Fx + Fy^T diag(W chi) Fy + diag(Wy) (x) Jx + Jy (x) diag(Wx), from the 1-D matrices."""
    P, Nx, Ny = g.P, g.Nx, g.Ny
    hx, hy = g.lx / Nx, g.ly / Ny
    Fx1, Jx1 = oracle.dg_matrix_1d(Nx, P, hx, g.bcx)
    Fy1, Jy1 = oracle.dg_matrix_1d(Ny, P, hy, g.bcy)
    w = oracle.dg_tables(P)["w"]
    Wx = np.tile(hx / 2 * w, Nx); Wy = np.tile(hy / 2 * w, Ny)
    Ix, Iy = np.eye(Nx * P), np.eye(Ny * P)
    Fx = np.kron(Iy, Fx1); Fy = np.kron(Fy1, Ix)               # x fastest
    Wc = np.kron(Wy, Wx) * chi
    S = Fx.T @ (Wc[:, None] * Fx) + Fy.T @ (Wc[:, None] * Fy) + np.kron(np.diag(Wy), Jx1) + np.kron(Jy1, np.diag(Wx))
    return S, np.kron(Wy, Wx)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("bc", BCS)
def test_definition_and_canonical_match_dense_assembly(oracle, P, bc):
    g = oracle.Grid(5, 4, P, 1.7, 2.3, bc[0], bc[1])
    r = fi.rng(7000 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    x = r.uniform(-1, 1, g.n)
    S, W = assemble_S(oracle, g, chi)
    ydense = S @ x
    ydef, scale = oracle.dg_apply_definition(g, chi, x, normed=False)
    ycan = oracle.dg_apply_canonical(g, chi, x, normed=False)
    assert np.all(scale > 0)
    assert np.abs(ydef - ydense).max() <= 2e-14 * scale.max()
    assert np.all(np.abs(ycan - ydef) <= 1e-14 * scale)        # the north star's 1e-14, in the |A||x| scale (Q16)
    # normed variants: A = V o S
    adef, ascale = oracle.dg_apply_definition(g, chi, x, normed=True)
    acan = oracle.dg_apply_canonical(g, chi, x, normed=True)
    assert np.all(np.abs(adef - ydense / W) <= 2e-14 * ascale.max())
    assert np.all(np.abs(acan - adef) <= 1e-14 * ascale)
    Wo, Vo = oracle.dg_weights(g)
    assert np.allclose(Wo, W, rtol=1e-15) and np.allclose(Vo * Wo, 1.0, rtol=1e-15)
    assert np.array_equal(acan, Vo * ycan)                      # A x = RN(V * (S x)) exactly


@pytest.mark.parametrize("P", [1, 2, 3, 5])
@pytest.mark.parametrize("bc", BCS)
def test_symmetry_and_definiteness(oracle, P, bc):
    g = oracle.Grid(6, 5, P, 2.0, 1.5, bc[0], bc[1])
    r = fi.rng(7100 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    x = r.uniform(-1, 1, g.n); y = r.uniform(-1, 1, g.n)
    Sx = oracle.dg_apply_canonical(g, chi, x); Sy = oracle.dg_apply_canonical(g, chi, y)
    a, b = oracle.exdot(x, Sy), oracle.exdot(y, Sx)             # x.Sy = y.Sx
    assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))
    # the same statement "in the dG weights" for the normed operator: <x, A y>_W = <y, A x>_W
    W, _ = oracle.dg_weights(g)
    Ax = oracle.dg_apply_canonical(g, chi, x, True); Ay = oracle.dg_apply_canonical(g, chi, y, True)
    a, b = oracle.exdot(W * x, Ay), oracle.exdot(W * y, Ax)
    assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))
    assert oracle.exdot(x, Sx) > 0
    one = np.ones(g.n)
    S1 = oracle.dg_apply_canonical(g, chi, one)
    S, _ = assemble_S(oracle, g, chi)
    ev = np.linalg.eigvalsh((S + S.T) / 2)
    if bc == (PER, PER):
        assert np.abs(S1).max() < 1e-12                         # constants are the null space
        assert abs(ev[0]) < 1e-11 * ev[-1] and ev[1] > 1e-6 * ev[-1]   # exactly one null vector
    else:
        assert np.abs(S1).max() > 1e-3
        assert ev[0] > 1e-8 * ev[-1]                            # SPD as soon as one side is Dirichlet


def test_jump_term_is_what_makes_it_definite(oracle):
    # without the jump penalty the LDG operator is singular even with Dirichlet sides (Q8):
    # assemble S - J and look at its smallest eigenvalue
    g = oracle.Grid(4, 4, 3, 1.0, 1.0, DIR, DIR)
    chi = np.ones(g.n)
    S, _ = assemble_S(oracle, g, chi)
    P, hx, hy = g.P, g.lx / g.Nx, g.ly / g.Ny
    _, Jx1 = oracle.dg_matrix_1d(g.Nx, P, hx, DIR); _, Jy1 = oracle.dg_matrix_1d(g.Ny, P, hy, DIR)
    w = oracle.dg_tables(P)["w"]
    J = np.kron(np.diag(np.tile(hy / 2 * w, g.Ny)), Jx1) + np.kron(Jy1, np.diag(np.tile(hx / 2 * w, g.Nx)))
    ev_with = np.linalg.eigvalsh(S); ev_without = np.linalg.eigvalsh(S - J)
    assert ev_with[0] > 1e-6 * ev_with[-1]
    assert abs(ev_without[0]) < 1e-10 * ev_without[-1]


def test_p1_five_point_stencil(oracle):
    # P=1, chi=1, PER x PER:  (S u)_ij = hy(1/hx + 1)(2u_ij - u_i+1j - u_i-1j) + hx(1/hy + 1)(2u_ij - u_ij+1 - u_ij-1)
    Nx, Ny, lx, ly = 7, 5, 2.0, 3.0
    g = oracle.Grid(Nx, Ny, 1, lx, ly, PER, PER)
    hx, hy = lx / Nx, ly / Ny
    u = fi.rng(7200).uniform(-1, 1, (Ny, Nx))
    lapx = 2 * u - np.roll(u, 1, 1) - np.roll(u, -1, 1)
    lapy = 2 * u - np.roll(u, 1, 0) - np.roll(u, -1, 0)
    exp = hy * (1 / hx + 1) * lapx + hx * (1 / hy + 1) * lapy
    got = oracle.dg_apply_canonical(g, np.ones(g.n), u.ravel()).reshape(Ny, Nx)
    assert np.abs(got - exp).max() < 1e-14 * np.abs(exp).max() * 10
    # variable chi: the face between cells i and i+1 carries chi_i (forward flux)
    chi = 1.0 + 0.5 * fi.rng(7201).uniform(-1, 1, (Ny, Nx))
    fx = chi * (np.roll(u, -1, 1) - u)          # chi_i (u_{i+1}-u_i)
    fy = chi * (np.roll(u, -1, 0) - u)
    exp = hy / hx * (np.roll(fx, 1, 1) - fx) + hx / hy * (np.roll(fy, 1, 0) - fy) + hy * lapx + hx * lapy
    got = oracle.dg_apply_canonical(g, chi.ravel(), u.ravel()).reshape(Ny, Nx)
    assert np.abs(got - exp).max() < 1e-13 * np.abs(exp).max()


@pytest.mark.parametrize("shape", [(1, 1), (1, 3), (2, 1), (2, 2), (1, 7)])
@pytest.mark.parametrize("P", [1, 3, 4])
def test_edge_grids(oracle, shape, P):
    for bc in BCS:
        g = oracle.Grid(shape[0], shape[1], P, 1.0, 2.0, bc[0], bc[1])
        r = fi.rng(7300)
        chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n); x = r.uniform(-1, 1, g.n)
        ydef, scale = oracle.dg_apply_definition(g, chi, x)
        ycan = oracle.dg_apply_canonical(g, chi, x)
        assert np.all(np.abs(ycan - ydef) <= 1e-14 * scale)


def test_layout_index_encoding(oracle):
    # idx = ((j*P + l)*Nx + i)*P + k : the weights factorise as Wy[j,l] * Wx[i,k] in exactly that layout
    g = oracle.Grid(3, 2, 4, 1.5, 0.5, PER, DIR)
    W, V = oracle.dg_weights(g)
    w = oracle.dg_tables(4)["w"]
    img = W.reshape(g.Ny * g.P, g.Nx * g.P)
    exp = np.outer(np.tile(0.25 / 2 * w, 2), np.tile(0.5 / 2 * w, 3))
    assert np.allclose(img, exp, rtol=1e-15)
    xs, ys = oracle.dg_nodes(g)
    assert np.all(np.diff(xs) > 0) and np.all(np.diff(ys) > 0) and xs.size == 12 and ys.size == 8
    # input nodes (numpy leggauss) agree with the oracle's to rounding: they are data, not tables
    assert np.allclose(fi.node_coords(3, 4, 1.5), xs, rtol=1e-14)
    # an x-only function must produce an x-only operator image under PER in y (no accidental transposition)
    g2 = oracle.Grid(4, 3, 3, 1.0, 1.0, DIR, PER)
    xs, ys = oracle.dg_nodes(g2)
    u = np.broadcast_to(np.sin(3 * xs)[None, :], (ys.size, xs.size)).ravel()
    y = oracle.dg_apply_canonical(g2, np.ones(g2.n), u, normed=True).reshape(ys.size, xs.size)
    assert np.abs(y - y[0:1, :]).max() < 1e-11


# ---------------------------------------------------------------- vector primitives
def test_axpby_pointwise_canonical_order(oracle):
    r = fi.rng(7400)
    n = 1001
    x = r.uniform(-1, 1, n); y = r.uniform(-1, 1, n); x2 = r.uniform(-1, 1, n)
    a, b = 0.7, -0.3
    # exact rational evaluation of the two-rounding definition  fma(a, x, RN(b*y))   ("t=b*y ... y=fma(a,x,t)")
    got = oracle.axpby(a, x, b, y)
    for i in range(0, n, 50):
        t = float(Fraction(b) * Fraction(y[i]))
        assert got[i] == float(Fraction(a) * Fraction(x[i]) + Fraction(t))
    assert np.array_equal(oracle.axpby(a, x, 0.0, np.full(n, np.nan)), a * x)      # beta = 0: y not read
    assert np.array_equal(oracle.axpby(1.0, x, 1.0, y), x + y)                     # no rounding in the products
    got = oracle.pointwise_dot(a, x, x2, b, y)
    for i in range(0, n, 50):
        u = float(Fraction(a) * Fraction(x[i])); t = float(Fraction(b) * Fraction(y[i]))
        assert got[i] == float(Fraction(u) * Fraction(x2[i]) + Fraction(t))
    assert np.array_equal(oracle.pointwise_dot(1.0, x, x2, 0.0, np.full(n, np.nan)), x * x2)
    # small integers: no rounding anywhere, any order gives the same
    xi = r.integers(-100, 100, n).astype(float); yi = r.integers(-100, 100, n).astype(float)
    assert np.array_equal(oracle.axpby(3.0, xi, -5.0, yi), 3 * xi - 5 * yi)
    assert np.array_equal(oracle.pointwise_dot(2.0, xi, yi, 4.0, xi), 2 * xi * yi + 4 * xi)
