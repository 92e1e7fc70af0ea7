"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no dot, no dG operator, no CG, no GL tables used
by either implementation): it only produces input arrays -- random vectors, coefficient fields chi,
right-hand sides rho -- with the shapes, sizes and value ranges of the paper's workloads (2-D
tensor-product dG vectors, P = 1..5, 0.1-1000 MB; Tables 2-4) and of BASELINE.json's
five configs.  They stand in for the paper's datasets [58],[59], which are not
available.  Both sides receive the same arrays (transcendental functions differ by
libm, so they are evaluated once, here).  Recipe: DESIGN.md section 5.

Node coordinates used to sample chi/rho come from numpy's leggauss: they are input data, not the
tables of the method (which each implementation derives independently at >= 100 bit).
"""
import math

import numpy as np

SEED_BASE = 180701971
PER, DIR = 0, 1


def uniform(seed_offset, n):
    """n doubles in [-1,1): Philox raw 64-bit r -> (r >> 11) * 2^-52 - 1."""
    bg = np.random.Philox(key=SEED_BASE + int(seed_offset))
    r = bg.random_raw(int(n))
    return (r >> np.uint64(11)).astype(np.float64) * 2.0 ** -52 - 1.0


def rng(seed_offset):
    return np.random.Generator(np.random.Philox(key=SEED_BASE + int(seed_offset)))


def node_coords(N, P, length):
    """x(i,k) = h*(i + (1+xi_k)/2), Gauss-Legendre abscissas xi_k on [-1,1] (Fig. 2)."""
    xi, _ = np.polynomial.legendre.leggauss(P)
    h = length / N
    return (h * (np.arange(N)[:, None] + (1.0 + xi[None, :]) / 2.0)).ravel()


def mesh(Nx, Ny, P, lx, ly):
    """-> X, Y of shape (Ny*P, Nx*P): the row-major, x-fastest image layout of DESIGN.md section 4."""
    x = node_coords(Nx, P, lx)
    y = node_coords(Ny, P, ly)
    return np.broadcast_to(x[None, :], (y.size, x.size)), np.broadcast_to(y[:, None], (y.size, x.size))


TWO_PI = 2.0 * math.pi


def config0(N=64, P=3):
    """BASELINE.json configs[0]: manufactured solution phi = sin x sin y, chi = 1 + 0.5 sin x sin y,
    periodic in x, Dirichlet in y, phi0 = 0, tol 1e-10."""
    X, Y = mesh(N, N, P, TWO_PI, TWO_PI)
    sx, sy, cx, cy = np.sin(X), np.sin(Y), np.cos(X), np.cos(Y)
    chi = 1.0 + 0.5 * sx * sy
    phi = sx * sy
    # rho = div(chi grad phi) = chi*lap(phi) + grad(chi).grad(phi)
    rho = -2.0 * sx * sy * chi + 0.5 * (cx * cx * sy * sy + sx * sx * cy * cy)
    grid = dict(Nx=N, Ny=N, P=P, lx=TWO_PI, ly=TWO_PI, bcx=PER, bcy=DIR)
    return dict(grid=grid, chi=chi.ravel().copy(), rho=rho.ravel().copy(), phi_exact=phi.ravel().copy(),
                phi0=np.zeros(chi.size), tol=1e-10, maxit=10000)


def _polarisation(N, P, seed_offset):
    X, Y = mesh(N, N, P, TWO_PI, TWO_PI)
    Ngc = 1.0 + 0.5 * np.exp(-((X - math.pi) ** 2 + (Y - math.pi) ** 2) / 0.5)
    u = uniform(seed_offset, Ngc.size).reshape(Ngc.shape)
    n_e = Ngc + 1e-3 * u                  # n = N + 1e-3 * noise
    rho = n_e - Ngc                       # right-hand side n - N of Eq. (1c)
    grid = dict(Nx=N, Ny=N, P=P, lx=TWO_PI, ly=TWO_PI, bcx=DIR, bcy=DIR)
    return dict(grid=grid, chi=Ngc.ravel().copy(), rho=rho.ravel().copy(), phi0=np.zeros(Ngc.size))


def config2(N=256, P=3):
    """BASELINE.json configs[2]: gyro-fluid polarisation equation div(N grad phi) = n - N, DIR x DIR."""
    d = _polarisation(N, P, 2)
    d.update(tol=1e-8, maxit=20000)
    return d


def config3(N=1024, P=3):
    """BASELINE.json configs[3]: as config 2 on 1024^2 cells, fixed 200 iterations (tol = 0)."""
    d = _polarisation(N, P, 3)
    d.update(tol=0.0, maxit=200)
    return d


def config4(P, N, bcx=PER, bcy=DIR):
    """BASELINE.json configs[4]: latency-bandwidth sweep inputs, uniform[-1,1) vectors."""
    n = P * P * N * N
    off = 4000 + 10 * P + int(round(math.log2(N)))
    x = uniform(off * 10 + 0, n)
    y = uniform(off * 10 + 1, n)
    chi = 1.0 + 0.5 * uniform(off * 10 + 2, n)
    grid = dict(Nx=N, Ny=N, P=P, lx=TWO_PI, ly=TWO_PI, bcx=bcx, bcy=bcy)
    return dict(grid=grid, x=x, y=y, chi=chi)


COND_TARGETS = [1e0, 1e8, 1e16, 1e24, 1e32, 1e40]


def dot_family_a(k, cond_index):
    """BASELINE.json configs[1], family A: n = 2^k elements, target condition COND_TARGETS[cond_index].

    Half the products have random 53-bit mantissas and exponents spread over about [-e, e]; the other half
    are their exact negatives, so everything cancels except a payload of four products 3,5,7,11 (times
    2^-e).  Returns (x, y, expected) where expected = 26 * 2^-e is exact by construction, or None for
    cond_index 0 (no cancelling half: all products positive, the oracle gives the value)."""
    n = 1 << k
    c = COND_TARGETS[cond_index]
    g = rng(1000 * cond_index + k)
    if cond_index == 0:
        x = 1.0 + g.integers(0, 1 << 52, n).astype(np.float64) * 2.0 ** -52
        y = 1.0 + g.integers(0, 1 << 52, n).astype(np.float64) * 2.0 ** -52
        return x, y, None
    e = max(0, int(round((math.log2(c) - math.log2(n)) / 2.0)))
    he = (e + 1) // 2
    h = n // 2
    f = 1.0 + g.integers(0, 1 << 52, h).astype(np.float64) * 2.0 ** -52
    gg = 1.0 + g.integers(0, 1 << 52, h).astype(np.float64) * 2.0 ** -52
    a = g.integers(-he, he + 1, h)
    b = g.integers(-he, he + 1, h)
    sgn = np.where(g.integers(0, 2, h) == 0, 1.0, -1.0)
    xh = sgn * np.ldexp(f, a)
    yh = np.ldexp(gg, b)
    x = np.concatenate([xh, -xh])
    y = np.concatenate([yh, yh])
    for q, cq in enumerate((3.0, 5.0, 7.0, 11.0)):       # payload: exact sum 26 * 2^-e
        x[q] = math.ldexp(cq, -e); y[q] = 1.0
        x[q + h] = 0.0
    perm = g.permutation(n)
    return x[perm].copy(), y[perm].copy(), math.ldexp(26.0, -e)


def dot_family_b(k, cond_index, oracle):
    """BASELINE.json configs[1], family B (rounding-residue cancellation): n = 2^k elements (k <= 22).

    First half as family A's first half (random 53-bit mantissas, product exponents spread over about [-e, e]).
    Second half: x_j random as above and y_j = RN((t_j - sigma_j)/x_j), sigma_j the correctly rounded running sum and
    t_j = u_j * 2^(e_j) with e_j descending linearly from e to -e, so that the partial sums are driven down through the
    whole exponent range and the final sum is what the rounding residues leave.  The running sums need the method's
    arithmetic, so they come from the oracle passed in (`oracle.exdot_cancel_fill`); this module computes none of it.
    No permutation is applied (the construction is order dependent).  Returns (x, y)."""
    assert 1 <= cond_index < len(COND_TARGETS) and k <= 22
    n = 1 << k
    c = COND_TARGETS[cond_index]
    g = rng(2000 * cond_index + k)
    e = max(1, int(round((math.log2(c) - math.log2(n)) / 2.0)))
    he = (e + 1) // 2
    h = n // 2

    def rand_half(m):
        f = 1.0 + g.integers(0, 1 << 52, m).astype(np.float64) * 2.0 ** -52
        a = g.integers(-he, he + 1, m)
        sgn = np.where(g.integers(0, 2, m) == 0, 1.0, -1.0)
        return sgn * np.ldexp(f, a)

    x = np.concatenate([rand_half(h), rand_half(n - h)])
    y = np.concatenate([np.abs(rand_half(h)), np.zeros(n - h)])
    u = uniform(2500 + 40 * cond_index + k, n)
    ej = np.round(np.linspace(e, -e, n - h)).astype(np.int64)
    t = np.zeros(n)
    t[h:] = np.ldexp(u[h:], ej)
    y = oracle.exdot_cancel_fill(x, y, h, t)
    return x, y


def dot_wide_spread(n, seed_offset=1700, spread=500):
    """products with exponents uniform over about [-2*spread, 2*spread] (no cancellation): every element far from its
    neighbours' binades -- the exact dot's worst case for a windowed expansion"""
    g = rng(seed_offset)
    f = 1.0 + g.integers(0, 1 << 52, n).astype(np.float64) * 2.0 ** -52
    gg = 1.0 + g.integers(0, 1 << 52, n).astype(np.float64) * 2.0 ** -52
    sgn = np.where(g.integers(0, 2, n) == 0, 1.0, -1.0)
    return sgn * np.ldexp(f, g.integers(-spread, spread + 1, n)), np.ldexp(gg, g.integers(-spread, spread + 1, n))


def dot_special_cases():
    """BASELINE.json configs[1] special set: zeros, denormals, +-2^1000, each mixed into a uniform
    background.  Returns a list of (name, x, y).  Expected values come from the oracle."""
    out = []
    n = 4099                                   # ragged
    bgx, bgy = uniform(1500, n), uniform(1501, n)

    def mixed(name, xs, ys, off):
        x, y = bgx.copy(), bgy.copy()
        pos = rng(1600 + off).permutation(n)[:len(xs)]
        x[pos] = xs; y[pos] = ys
        out.append((name, x, y))

    tiny = 5e-324
    mixed("signed_zeros", [0.0, -0.0, 0.0, -0.0], [1.0, 1.0, -0.0, -3.0], 0)
    mixed("subnormal_times_large", [tiny * 3, -tiny * 7, 2.0 ** -1060], [2.0 ** 1000, 2.0 ** 900, 2.0 ** 1023], 1)
    mixed("subnormal_times_subnormal", [tiny * 3, tiny * 5, -tiny], [tiny * 9, -tiny * 11, tiny], 2)
    mixed("pm_2p1000_safe", [2.0 ** 1000, -2.0 ** 1000, 2.0 ** 1000], [2.0 ** 23, 2.0 ** 23, -1.5], 3)
    mixed("overflow_products_cancel", [2.0 ** 1000, -2.0 ** 1000, 1.5], [2.0 ** 1000, 2.0 ** 1000, 1.0], 4)
    mixed("near_overflow_same_sign", [2.0 ** 1000] * 8, [2.0 ** 20] * 8, 5)
    mixed("underflow_products", [2.0 ** -600, 2.0 ** -600, -2.0 ** -700], [2.0 ** -600, -2.0 ** -500, 2.0 ** -370], 6)
    # without background: results that live entirely outside the double range of single products
    out.append(("pure_overflow_cancel", np.array([2.0 ** 1000, -2.0 ** 1000, 1.5]), np.array([2.0 ** 1000, 2.0 ** 1000, 1.0])))
    out.append(("pure_sub_sub", np.array([tiny] * 4), np.array([tiny] * 4)))
    out.append(("pure_quarter_ulp_sub", np.array([2.0 ** -538] * 4), np.array([2.0 ** -537] * 4)))
    out.append(("true_overflow", np.array([2.0 ** 1000, 2.0 ** 1000]), np.array([2.0 ** 23, 2.0 ** 23])))
    out.append(("inf_input", np.array([np.inf, 1.0]), np.array([2.0, 1.0])))
    out.append(("inf_minus_inf", np.array([np.inf, -np.inf]), np.array([2.0, 1.0])))
    out.append(("zero_times_inf", np.array([0.0, 1.0]), np.array([np.inf, 1.0])))
    out.append(("nan_input", np.array([np.nan, 1.0]), np.array([2.0, 1.0])))
    out.append(("neg_inf", np.array([-np.inf, 1.0, 3.0]), np.array([2.0, 1.0, np.inf * 0 + 1.0])))
    return out
