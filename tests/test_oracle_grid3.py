"""Pins of the oracle's 3-D product-grid functions (CPU only, reading DESIGN.md Q24).

The paper's applications are "2D/3D drift-/gyro-fluid simulations" with derivatives "on product spaces"
(P:240); its elliptic equation is the perpendicular one, div(chi grad_perp phi) = rho (Eq. 1c).  Reading: Nz
planes of the 2-D grid, one node per plane in z, weights W3 = hz*W2, the operator acts plane by plane and the planes meet
in the dot products of CG.  Pins: the volume of the box and an integral in closed form, dense block-diagonal assembly from
the 1-D matrices (numpy), symmetry / definiteness / null space with exact dots, definition vs canonical order, CG against
dense direct solves and against a manufactured solution that depends on z."""
import math

import numpy as np
import pytest

import fxinputs as fi
from test_oracle_dg import assemble_S

PER, DIR, NEU = 0, 1, 2


def test_weights_are_the_volume_form(oracle):
    g = oracle.Grid3(5, 4, 3, 3, 1.7, 2.3, 0.9, PER, DIR)
    W, V = oracle.dg3_weights(g)
    assert abs(oracle.exsum(W) - 1.7 * 2.3 * 0.9) <= 1e-13 * 1.7 * 2.3 * 0.9           # sum of the weights = volume of the box
    assert np.array_equal(V, 1.0 / W)
    # integral of exp(x) exp(y) (1 + 0.3 z): Gauss-Legendre in x, y (Fig. 2), midpoint rule in z (exact for linear z)
    g = oracle.Grid3(20, 20, 4, 3, 2.0, 2.0, 1.5, PER, PER)
    W, _ = oracle.dg3_weights(g)
    xs, ys = oracle.dg_nodes(g.plane)
    X, Y = np.meshgrid(xs, ys)
    hz = 1.5 / 4
    f = np.concatenate([(np.exp(X) * np.exp(Y) * (1.0 + 0.3 * hz * (p + 0.5))).ravel() for p in range(4)])
    exact = (math.e ** 2 - 1.0) ** 2 * (1.5 + 0.15 * 1.5 ** 2)
    assert abs(oracle.exdot(W, f) - exact) <= 5e-12 * exact


@pytest.mark.parametrize("P,bc", [(1, (DIR, PER)), (2, (PER, DIR)), (3, (DIR, DIR)), (4, (NEU, DIR)), (5, (PER, PER))])
def test_apply_against_dense_block_assembly_and_definition(oracle, P, bc):
    g = oracle.Grid3(4, 3, 3, P, 1.3, 0.8, 2.1, bc[0], bc[1])
    r = fi.rng(7700 + P)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n); x = r.uniform(-1, 1, g.n)
    hz = 2.1 / 3
    n2 = g.n // g.Nz
    ycan = oracle.dg3_apply_canonical(g, chi, x, normed=False)
    yn = oracle.dg3_apply_canonical(g, chi, x, normed=True)
    ydef, scale = oracle.dg3_apply_definition(g, chi, x, normed=False)
    yndef, nscale = oracle.dg3_apply_definition(g, chi, x, normed=True)
    for z in range(g.Nz):
        sl = slice(z * n2, (z + 1) * n2)
        S2, W2 = assemble_S(oracle, g.plane, chi[sl])                 # numpy, from the 1-D matrices: independent of both oracle paths
        dense = hz * (S2 @ x[sl])
        assert np.abs(ycan[sl] - dense).max() <= 1e-12 * np.abs(dense).max()
        assert np.abs(yn[sl] - (S2 @ x[sl]) / W2).max() <= 1e-12 * np.abs((S2 @ x[sl]) / W2).max()
    assert np.all(np.abs(ycan - ydef) <= 1e-14 * scale)               # canonical fp64 order vs 113-bit definition
    assert np.all(np.abs(yn - yndef) <= 1e-14 * nscale)
    # another plane's data never enters: changing plane 0 leaves planes 1, 2 bit for bit
    x2 = x.copy(); x2[:n2] = r.uniform(-1, 1, n2)
    y2 = oracle.dg3_apply_canonical(g, chi, x2, normed=False)
    assert np.array_equal(y2[n2:], ycan[n2:]) and not np.array_equal(y2[:n2], ycan[:n2])


@pytest.mark.parametrize("bc", [(PER, DIR), (DIR, NEU), (PER, PER)])
def test_symmetry_definiteness_null_space(oracle, bc):
    g = oracle.Grid3(6, 5, 4, 3, 2.0, 1.0, 3.0, bc[0], bc[1])
    r = fi.rng(7800)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n)
    x, y = r.uniform(-1, 1, g.n), r.uniform(-1, 1, g.n)
    Sx, Sy = oracle.dg3_apply_canonical(g, chi, x), oracle.dg3_apply_canonical(g, chi, y)
    a, b = oracle.exdot(y, Sx), oracle.exdot(x, Sy)
    assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))                  # S3 symmetric
    W, V = oracle.dg3_weights(g)
    Ax, Ay = oracle.dg3_apply_canonical(g, chi, x, normed=True), oracle.dg3_apply_canonical(g, chi, y, normed=True)
    a, b = oracle.exdot(W * y, Ax), oracle.exdot(W * x, Ay)
    assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))                  # A3 self-adjoint in the volume form
    assert np.abs(W * Ax - Sx).max() <= 1e-13 * np.abs(Sx).max()      # W3 o A3 = S3 (hz enters through the weights only)
    if bc == (PER, PER):
        ones = oracle.dg3_apply_canonical(g, chi, np.ones(g.n))
        assert np.abs(ones).max() <= 1e-12                             # constants: the null space (per plane)
        assert oracle.exdot(x, Sx) >= 0.0
    else:
        assert oracle.exdot(x, Sx) > 0.0


def test_cg3_against_dense_direct_solves(oracle):
    g = oracle.Grid3(4, 4, 3, 2, 1.3, 0.9, 1.1, DIR, PER)
    r = fi.rng(7900)
    chi = 1.0 + 0.5 * r.uniform(-1, 1, g.n); rho = r.uniform(-1, 1, g.n)
    phi, info = oracle.cg3_solve(g, chi, rho, np.zeros(g.n), 1e-13, 3000)
    assert info.status == oracle.OK and info.iterations > 0
    n2 = g.n // g.Nz
    for z in range(g.Nz):
        sl = slice(z * n2, (z + 1) * n2)
        S2, W2 = assemble_S(oracle, g.plane, chi[sl])
        direct = np.linalg.solve(S2, -W2 * rho[sl])                  # hz cancels: hz S2 phi = hz W2 (-rho)
        assert np.abs(phi[sl] - direct).max() <= 1e-9 * np.abs(direct).max()
    # one system over all planes: the iteration count is one number, and a plane with zero right-hand side stays zero
    rho0 = rho.copy(); rho0[n2:2 * n2] = 0.0
    phi0, info0 = oracle.cg3_solve(g, chi, rho0, np.zeros(g.n), 1e-12, 3000)
    assert not phi0[n2:2 * n2].any() and phi0[:n2].any()
    # degenerate: zero right-hand side, maxit
    z0, i0 = oracle.cg3_solve(g, chi, np.zeros(g.n), np.ones(g.n), 1e-8, 10)
    assert i0.iterations == 0 and not z0.any()
    _, i5 = oracle.cg3_solve(g, chi, rho, np.zeros(g.n), 0.0, 5)
    assert i5.iterations == 5 and i5.status == oracle.MAXIT


def test_cg3_manufactured_solution_depends_on_z(oracle):
    """phi = sin x sin y (1 + 0.5 cos z), chi = 1 + 0.5 sin x sin y cos z on [0,2pi]^3, PER x DIR: the W3-weighted relative
    error falls with order P under refinement in x, y (no derivative in z: the perpendicular operator, reading Q24)"""
    P, Nz = 3, 4
    errs = []
    for N in (8, 16):
        g = oracle.Grid3(N, N, Nz, P, fi.TWO_PI, fi.TWO_PI, fi.TWO_PI, PER, DIR)
        X, Y = fi.mesh(N, N, P, fi.TWO_PI, fi.TWO_PI)
        sx, sy, cx, cy = np.sin(X), np.sin(Y), np.cos(X), np.cos(Y)
        chis, rhos, sols = [], [], []
        for p in range(Nz):
            cz = math.cos(fi.TWO_PI / Nz * (p + 0.5))
            a = 1.0 + 0.5 * cz
            chi = 1.0 + 0.5 * sx * sy * cz
            # div_perp(chi grad_perp phi) with phi = a sin x sin y
            rho = a * (-2.0 * sx * sy * chi + 0.5 * cz * (cx * cx * sy * sy + sx * sx * cy * cy))
            chis.append(chi.ravel()); rhos.append(rho.ravel()); sols.append((a * sx * sy).ravel())
        chi, rho, sol = np.concatenate(chis), np.concatenate(rhos), np.concatenate(sols)
        phi, info = oracle.cg3_solve(g, chi, rho, np.zeros(g.n), 1e-11, 20000)
        assert info.status == oracle.OK
        W, _ = oracle.dg3_weights(g)
        errs.append(math.sqrt(oracle.exdot(W * (phi - sol), phi - sol) / oracle.exdot(W * sol, sol)))
    order = math.log2(errs[0] / errs[1])
    assert errs[1] < 5e-4 and 2.6 < order < 3.6, (errs, order)
