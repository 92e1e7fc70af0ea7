"""Pins of the oracle's Neumann and mixed walls (CPU only).  SURVEY.md 8f-4; reading DESIGN.md Q23: a Neumann wall's
ghost cell mirrors the interior trace, so the wall face carries neither a jump nor a flux correction.

What is pinned, none of it by re-typing the oracle's formulas:
  * a finite-difference closed form for P = 1 written out in numpy (brute force on a tiny grid),
  * exactness of the forward derivative on polynomials in the wall cells without any condition on the wall value,
  * the weak form: sum_k W_k (F u)_k over the whole line telescopes to u(b) - u(a) with the walls' prescribed values,
  * symmetry, semi-definiteness and the null space (constants iff no Dirichlet wall anywhere),
  * definition (113-bit) against dense assembly against the canonical fp64 order, all bc kinds,
  * convergence of the CG solution to an analytic solution with zero normal derivative at the Neumann walls,
  * unchanged results for PER and DIR (golden values written before this change stay valid: test_oracle_dg.py).
"""
import math

import numpy as np
import pytest

import fxinputs as fi
from test_oracle_dg import assemble_S

PER, DIR, NEU, DIR_NEU, NEU_DIR = 0, 1, 2, 3, 4
WALLS = {PER: ("per", "per"), DIR: ("dir", "dir"), NEU: ("neu", "neu"), DIR_NEU: ("dir", "neu"), NEU_DIR: ("neu", "dir")}
ALLBC = [(a, b) for a in range(5) for b in range(5) if a >= NEU or b >= NEU]


# ---------------------------------------------------------------- 1-D matrices
@pytest.mark.parametrize("P", range(1, 6))
@pytest.mark.parametrize("bc", [NEU, DIR_NEU, NEU_DIR])
def test_forward_derivative_is_exact_on_polynomials_at_neumann_walls(oracle, P, bc):
    N, length = 5, 1.5
    h = length / N
    F, _ = oracle.dg_matrix_1d(N, P, h, bc)
    g = oracle.Grid(N, 1, P, length, 1.0, PER, PER)
    xs, _ = oracle.dg_nodes(g)
    lo, hi = WALLS[bc]
    for d in range(P):
        u = (xs + 0.3) ** d                                      # does not vanish at either wall
        du = d * (xs + 0.3) ** max(d - 1, 0) if d else np.zeros_like(xs)
        err = np.abs(F @ u - du)
        # forward flux: the lower wall face uses the cell's own value unless the wall is Dirichlet; the upper wall
        # face uses the ghost: mirrored (NEU, no correction) or zero (DIR, correction -u(b))
        first_ok = lo == "neu"
        last_ok = hi == "neu"
        assert err[P:(N - 1) * P].max() < 1e-11
        if first_ok:
            assert err[:P].max() < 1e-11, (P, bc, d)
        else:
            assert err[:P].max() > 1e-3, (P, bc, d)              # DIR at the lower wall: sees the jump from 0
        if last_ok:
            assert err[(N - 1) * P:].max() < 1e-11, (P, bc, d)
        else:
            assert err[(N - 1) * P:].max() > 1e-3, (P, bc, d)


@pytest.mark.parametrize("P", range(1, 6))
@pytest.mark.parametrize("bc", [PER, DIR, NEU, DIR_NEU, NEU_DIR])
def test_weak_form_telescopes_to_the_wall_values(oracle, P, bc):
    # sum over the line of W (F u) = [u-hat at the upper wall] - [u-hat at the lower wall]; the wall's u-hat is 0 for
    # Dirichlet, the interior trace for Neumann; interior faces cancel; periodic: 0.
    N, length = 4, 2.0
    h = length / N
    F, _ = oracle.dg_matrix_1d(N, P, h, bc)
    t = oracle.dg_tables(P)
    W = np.tile(h / 2 * t["w"], N)
    r = fi.rng(7700 + P)
    u = r.uniform(-1, 1, N * P)
    ua = float(np.dot(t["L"], u[:P])); ub = float(np.dot(t["R"], u[(N - 1) * P:]))   # interior traces at the walls
    lo, hi = WALLS[bc]
    exp = 0.0 if bc == PER else (ub if hi == "neu" else 0.0) - (ua if lo == "neu" else 0.0)
    assert abs(np.dot(W, F @ u) - exp) < 1e-12


@pytest.mark.parametrize("P", range(1, 6))
@pytest.mark.parametrize("bc", [NEU, DIR_NEU, NEU_DIR])
def test_jump_matrix_has_no_wall_face_at_a_neumann_wall(oracle, P, bc):
    N, h = 4, 0.25
    _, J = oracle.dg_matrix_1d(N, P, h, bc)
    _, Jd = oracle.dg_matrix_1d(N, P, h, DIR)
    t = oracle.dg_tables(P)
    L, R = t["L"], t["R"]
    assert np.abs(J - J.T).max() == 0 and np.linalg.eigvalsh(J).min() > -1e-12
    lo, hi = WALLS[bc]
    D = Jd - J                                                    # what the Dirichlet walls add: u(a)^2 + u(b)^2
    exp = np.zeros_like(J)
    if lo == "neu": exp[:P, :P] += np.outer(L, L)
    if hi == "neu": exp[(N - 1) * P:, (N - 1) * P:] += np.outer(R, R)
    assert np.abs(D - exp).max() < 1e-14
    one = np.ones(N * P)
    # u J u = sum over the faces that exist of [u]^2: for u = 1 only Dirichlet wall faces are left
    assert abs(one @ J @ one - ((lo == "dir") + (hi == "dir"))) < 1e-13


def test_p1_finite_difference_closed_form(oracle):
    # P = 1, 1-D (Ny = 1, periodic in y: that part vanishes identically).  F u_n = (u_{n+1} - u_n)/hx with the ghost
    # u_N = 0 (DIR) or u_{N-1} (NEU); at a Dirichlet lower wall the first row is (u_1 - 0)/hx (the wall value 0 replaces
    # u_0); one jump [u] per face that exists (interior faces, Dirichlet wall faces):
    #   S = hy * ( hx F^T diag(chi) F + J ),  J = sum_faces [v][u]
    Nx, lx, ly = 6, 1.2, 0.7
    hx, hy = lx / Nx, ly
    r = fi.rng(7710)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, Nx)
    u = r.uniform(-1, 1, Nx)
    for bc in (NEU, DIR_NEU, NEU_DIR, DIR):
        lo, hi = WALLS[bc]
        F = np.zeros((Nx, Nx))
        for n in range(Nx):
            F[n, n] = -1 / hx
            if n + 1 < Nx: F[n, n + 1] = 1 / hx
            elif hi == "neu": F[n, n] += 1 / hx                   # ghost = own value: forward difference 0
        if lo == "dir": F[0, 0] += 1 / hx                        # u-hat = 0 on the lower wall face
        faces = []                                               # rows of the jump operator, one per existing face
        for n in range(Nx - 1):
            e = np.zeros(Nx); e[n] = 1; e[n + 1] = -1; faces.append(e)
        if lo == "dir": e = np.zeros(Nx); e[0] = 1; faces.append(e)
        if hi == "dir": e = np.zeros(Nx); e[Nx - 1] = 1; faces.append(e)
        Jm = sum(np.outer(e, e) for e in faces)
        S = hy * (hx * F.T @ np.diag(chi) @ F + Jm)
        g = oracle.Grid(Nx, 1, 1, lx, ly, bc, PER)
        got = oracle.dg_apply_canonical(g, chi, u)
        assert np.abs(got - S @ u).max() < 1e-13 * np.abs(S @ u).max(), bc
        gd, _ = oracle.dg_apply_definition(g, chi, u)
        assert np.abs(gd - S @ u).max() < 1e-13 * np.abs(S @ u).max(), bc
        # the same line along y
        g2 = oracle.Grid(1, Nx, 1, ly, lx, PER, bc)
        got2 = oracle.dg_apply_canonical(g2, chi, u)
        assert np.abs(got2 - S @ u).max() < 1e-13 * np.abs(S @ u).max(), bc


# ---------------------------------------------------------------- 2-D operator
@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("bc", ALLBC)
def test_definition_dense_and_canonical_agree(oracle, P, bc):
    g = oracle.Grid(4, 3, P, 1.7, 2.3, bc[0], bc[1])
    r = fi.rng(7720 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    x = r.uniform(-1, 1, g.n)
    S, W = assemble_S(oracle, g, chi)
    ydense = S @ x
    ydef, scale = oracle.dg_apply_definition(g, chi, x, normed=False)
    ycan = oracle.dg_apply_canonical(g, chi, x, normed=False)
    assert np.abs(ydef - ydense).max() <= 2e-14 * scale.max()
    assert np.all(np.abs(ycan - ydef) <= 1e-14 * scale)
    acan = oracle.dg_apply_canonical(g, chi, x, normed=True)
    _, Vo = oracle.dg_weights(g)
    assert np.array_equal(acan, Vo * ycan)


@pytest.mark.parametrize("P", [1, 2, 3, 5])
@pytest.mark.parametrize("bc", ALLBC)
def test_symmetry_definiteness_and_null_space(oracle, P, bc):
    g = oracle.Grid(5, 4, P, 2.0, 1.5, bc[0], bc[1])
    r = fi.rng(7730 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    x = r.uniform(-1, 1, g.n); y = r.uniform(-1, 1, g.n)
    Sx = oracle.dg_apply_canonical(g, chi, x); Sy = oracle.dg_apply_canonical(g, chi, y)
    a, b = oracle.exdot(x, Sy), oracle.exdot(y, Sx)
    assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))
    S, _ = assemble_S(oracle, g, chi)
    ev = np.linalg.eigvalsh((S + S.T) / 2)
    S1 = oracle.dg_apply_canonical(g, chi, np.ones(g.n))
    has_dir = any("dir" in WALLS[c] for c in bc)
    if has_dir:
        assert np.abs(S1).max() > 1e-3 and ev[0] > 1e-8 * ev[-1]             # SPD as soon as one wall is Dirichlet
    else:
        assert np.abs(S1).max() < 1e-12                                      # pure Neumann / periodic: S 1 = 0 ...
        assert abs(ev[0]) < 1e-11 * ev[-1] and ev[1] > 1e-6 * ev[-1]         # ... and nothing else is in the null space


@pytest.mark.parametrize("shape,bc", [((1, 1), (NEU, NEU)), ((1, 3), (NEU, DIR_NEU)), ((2, 1), (DIR_NEU, NEU_DIR)),
                                      ((1, 1), (NEU_DIR, NEU)), ((3, 2), (NEU_DIR, DIR_NEU))])
def test_edge_grids(oracle, shape, bc):
    g = oracle.Grid(shape[0], shape[1], 3, 1.0, 2.0, bc[0], bc[1])
    r = fi.rng(7740)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n); x = r.uniform(-1, 1, g.n)
    ydef, scale = oracle.dg_apply_definition(g, chi, x)
    ycan = oracle.dg_apply_canonical(g, chi, x)
    assert np.all(np.abs(ycan - ydef) <= 1e-14 * scale)


def test_rejected_grids(oracle):
    with pytest.raises(Exception):
        oracle.dg_apply_canonical(oracle.Grid(1, 4, 2, 1.0, 1.0, DIR_NEU, PER), np.ones(16), np.ones(16))   # one cell, two wall kinds
    with pytest.raises(Exception):
        oracle.dg_apply_canonical(oracle.Grid(4, 4, 2, 1.0, 1.0, 5, PER), np.ones(64), np.ones(64))
    g = oracle.Grid(4, 4, 2, 1.0, 1.0, NEU, PER)
    with pytest.raises(Exception):                                # derivatives and the bracket: PER and DIR only
        oracle.dg_derivative_canonical(g, 0, 0, 1.0, np.ones(g.n), 0.0, np.zeros(g.n))


# ---------------------------------------------------------------- CG with Neumann walls
def _manufactured(oracle, N, P, bcx, bcy):
    """phi = X(x) Y(y) on [0,pi]^2 with X, Y chosen per wall kind; chi = 1 + 0.5 cos x cos y (zero normal derivative
    everywhere, positive); rho = div(chi grad phi) evaluated analytically at the nodes."""
    g = oracle.Grid(N, N, P, math.pi, math.pi, bcx, bcy)
    xs, ys = oracle.dg_nodes(g)
    X, Y = np.meshgrid(xs, ys)

    def prof(bc, s):                       # value, first and second derivative
        if bc == DIR: return np.sin(s), np.cos(s), -np.sin(s)
        if bc == NEU: return np.cos(s), -np.sin(s), -np.cos(s)
        if bc == DIR_NEU: return np.sin(s / 2), np.cos(s / 2) / 2, -np.sin(s / 2) / 4
        if bc == NEU_DIR: return np.cos(s / 2), -np.sin(s / 2) / 2, -np.cos(s / 2) / 4
        raise ValueError
    fx, dfx, ddfx = prof(bcx, X); fy, dfy, ddfy = prof(bcy, Y)
    chi = 1 + 0.5 * np.cos(X) * np.cos(Y)
    chix = -0.5 * np.sin(X) * np.cos(Y); chiy = -0.5 * np.cos(X) * np.sin(Y)
    phi = fx * fy
    rho = chix * dfx * fy + chi * ddfx * fy + chiy * fx * dfy + chi * fx * ddfy
    return g, chi.ravel(), rho.ravel(), phi.ravel()


@pytest.mark.parametrize("bc", [(NEU, DIR), (DIR_NEU, NEU_DIR), (DIR, NEU), (NEU_DIR, NEU)])
def test_cg_converges_to_the_analytic_solution(oracle, bc):
    P = 3
    errs = []
    for N in (6, 12, 24):
        g, chi, rho, phi_exact = _manufactured(oracle, N, P, bc[0], bc[1])
        phi, info = oracle.cg_solve(g, chi, rho, np.zeros(g.n), 1e-12, 5000)
        assert info.status == oracle.OK
        W, _ = oracle.dg_weights(g)
        errs.append(math.sqrt(oracle.exdot(W * (phi - phi_exact), phi - phi_exact) / oracle.exdot(W * phi_exact, phi_exact)))
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[-1] < 2e-4 and orders[-1] > 2.6, (bc, errs, orders)


@pytest.mark.parametrize("P,bc", [(2, (NEU, DIR)), (3, (DIR_NEU, PER)), (4, (NEU_DIR, DIR_NEU))])
def test_cg_against_dense_direct_solve(oracle, P, bc):
    g = oracle.Grid(4, 4, P, 1.3, 0.9, bc[0], bc[1])
    r = fi.rng(7750 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    rho = r.uniform(-1, 1, g.n)
    S, W = assemble_S(oracle, g, chi)
    phi_direct = np.linalg.solve(S, -W * rho)
    phi, info = oracle.cg_solve(g, chi, rho, np.zeros(g.n), 1e-13, 3000)
    assert info.status == oracle.OK
    assert np.abs(phi - phi_direct).max() <= 1e-10 * np.abs(phi_direct).max()
