"""Pins of the oracle's exact dot product (CPU only).

The oracle computes RN(sum_i x_i*y_i) ("correctly rounded (rounding-to-nearest)").
None of these pins retypes the oracle's limb arithmetic: they compare against Python's exact
rationals, closed forms, the paper's printed example, math.fsum, and algebraic invariants.
"""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

import fxinputs as fi
from conftest import golden_path


def frac_round(fr):
    """correctly rounded double of an exact rational: CPython's Fraction->float is round-half-even
    (int/int true division), incl. subnormals; overflow -> +-inf"""
    try:
        return float(fr)
    except OverflowError:
        return math.inf if fr > 0 else -math.inf


def frac_dot(x, y):
    return sum((Fraction(float(a)) * Fraction(float(b)) for a, b in zip(x, y)), Fraction(0))


def bits(v):
    return np.float64(v).view(np.uint64)


def same(a, b):
    return bits(a) == bits(b)


# ---------------------------------------------------------------- the paper's example
def test_paper_associativity_example(oracle):
    xs = exp = None
    for line in open(golden_path("paper_assoc_example.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "x":
            xs = [float.fromhex(v) for v in t[1:]]
        if t[0] == "expected":
            exp = float.fromhex(t[1])
    assert xs == [-1.0, 1.0, 2.0 ** -53] and exp == 2.0 ** -53
    # binary64 itself gives two different answers (the paper's point) ...
    assert (xs[0] + xs[1]) + xs[2] == 2.0 ** -53 and xs[0] + (xs[1] + xs[2]) == 0.0
    # ... the exact dot gives one, for every ordering
    for perm in itertools.permutations(xs):
        assert same(oracle.exdot(list(perm), [1.0, 1.0, 1.0]), exp)


def test_accumulator_width_covers_kulisch(oracle):
    kul = int([l.split()[1] for l in open(golden_path("kulisch_accumulator.txt")) if l.startswith("kulisch_bits")][0])
    _, limbs, _ = oracle.exdot_digits([1.0], [1.0])
    assert limbs.size * 64 >= kul == 4288
    # 1.0*1.0 = 2^0 sits at bit 2176: limb 34, bit 0
    assert limbs[34] == 1 and limbs.sum() == 1
    # extremes of the product range are representable: (2^-1074)^2 and ~(2^1024)^2
    tiny = 5e-324
    _, l1, _ = oracle.exdot_digits([tiny], [tiny])
    assert l1[(2176 - 2148) // 64] == np.uint64(1) << np.uint64((2176 - 2148) % 64) and np.count_nonzero(l1) == 1
    big = float.fromhex("0x1.fffffffffffffp+1023")
    _, l2, _ = oracle.exdot_digits([big], [big])
    top = max(k for k in range(68) if l2[k])
    assert 64 * top + int(l2[top]).bit_length() - 1 == 2176 + 2047


# ---------------------------------------------------------------- rational brute force
@pytest.mark.parametrize("seed", range(6))
def test_brute_force_random(oracle, seed):
    g = fi.rng(9000 + seed)
    n = [1, 2, 7, 64, 333, 2000][seed]
    spread = [0, 5, 40, 200, 600, 1000][seed]
    x = np.ldexp(g.uniform(-1, 1, n), g.integers(-spread, spread + 1, n))
    y = np.ldexp(g.uniform(-1, 1, n), g.integers(-spread // 2, spread // 2 + 1, n))
    assert same(oracle.exdot(x, y), frac_round(frac_dot(x, y)))


def test_brute_force_cancellation(oracle):
    # adversarial: huge terms cancel exactly, the result lives 600 binades below
    g = fi.rng(9100)
    for trial in range(20):
        n = 50
        x = np.ldexp(g.uniform(1, 2, n), g.integers(-300, 300, n))
        y = np.ldexp(g.uniform(1, 2, n), g.integers(-300, 300, n))
        xx = np.concatenate([x, -x, np.ldexp(g.uniform(-1, 1, 3), -600)])
        yy = np.concatenate([y, y, np.ones(3)])
        p = g.permutation(xx.size)
        assert same(oracle.exdot(xx[p], yy[p]), frac_round(frac_dot(xx[p], yy[p])))


def test_brute_force_subnormal_and_overflow_range(oracle):
    g = fi.rng(9200)
    tiny = 5e-324
    for trial in range(30):
        n = 12
        # subnormal results and subnormal inputs
        x = np.ldexp(g.uniform(-1, 1, n), g.integers(-1074, -1000, n))
        y = np.ldexp(g.uniform(-1, 1, n), g.integers(-30, 30, n))
        assert same(oracle.exdot(x, y), frac_round(frac_dot(x, y)))
        xs = g.integers(-5000, 5000, n).astype(np.float64) * tiny
        ys = g.integers(-5000, 5000, n).astype(np.float64) * tiny
        assert same(oracle.exdot(xs, ys), frac_round(frac_dot(xs, ys)))      # all below 2^-1075 -> rounding of tiny sums
        ys2 = np.ldexp(g.uniform(-1, 1, n), g.integers(1000, 1024, n))
        assert same(oracle.exdot(xs, ys2), frac_round(frac_dot(xs, ys2)))
        # near and beyond the overflow threshold
        xb = np.ldexp(g.uniform(-1, 1, n), g.integers(990, 1024, n))
        yb = np.ldexp(g.uniform(-1, 1, n), g.integers(-2, 40, n))
        assert same(oracle.exdot(xb, yb), frac_round(frac_dot(xb, yb)))


def test_special_set_against_rationals(oracle):
    for name, x, y in fi.dot_special_cases():
        if not (np.all(np.isfinite(x)) and np.all(np.isfinite(y))):
            continue
        got = oracle.exdot(x, y)
        assert same(got, frac_round(frac_dot(x, y))), name


# ---------------------------------------------------------------- closed forms
def test_closed_forms(oracle):
    # sum i^2 beyond 2^53: n(n+1)(2n+1)/6 for n = 400000 is ~2.1e16 > 2^53
    n = 400000
    i = np.arange(1, n + 1, dtype=np.float64)
    assert same(oracle.exdot(i, i), frac_round(Fraction(n * (n + 1) * (2 * n + 1), 6)))
    # geometric: sum_{i=1..n} 2^-i = 1 - 2^-n : n=53 exact, n=54 is a tie -> even -> 1.0
    for n, exp in ((53, 1.0 - 2.0 ** -53), (54, 1.0), (55, 1.0), (60, 1.0)):
        x = np.ldexp(1.0, -np.arange(1, n + 1))
        assert same(oracle.exdot(x, np.ones(n)), exp)
    # tie to even the other way: 1 + 2^-52 + 2^-53 -> 1 + 2^-51
    assert same(oracle.exdot([1.0, 2.0 ** -52, 2.0 ** -53], [1, 1, 1]), 1.0 + 2.0 ** -51)
    # tie broken by a far-away sticky bit
    assert same(oracle.exdot([1.0, 2.0 ** -53, 2.0 ** -1000], [1, 1, 1]), 1.0 + 2.0 ** -52)
    assert same(oracle.exdot([1.0, 2.0 ** -53, -2.0 ** -1000], [1, 1, 1]), 1.0)
    # n copies of the double 0.1: exact value n * Fraction(0.1)
    for n in (10, 1000, 12345):
        assert same(oracle.exdot(np.full(n, 0.1), np.ones(n)), frac_round(n * Fraction(0.1)))
    # subnormal tie: 3 * 2^-1075 -> 2^-1073 (tie between 2^-1074 and 2^-1073, even = 2^-1073)
    a = 2.0 ** -537
    b = 2.0 ** -538                      # a*b = 2^-1075
    assert same(oracle.exdot([a, a, a], [b, b, b]), 2.0 ** -1073)
    assert same(oracle.exdot([a], [b]), 0.0)                       # 2^-1075: tie -> even -> 0
    assert same(oracle.exdot([a, a, a, a], [b, b, b, b]), 2.0 ** -1073)
    # overflow threshold: 2^1024 - 2^970 rounds to +inf, one bit less is the largest double
    big = float.fromhex("0x1.fffffffffffffp+1023")
    assert oracle.exdot([big, 2.0 ** 970], [1, 1]) == math.inf
    assert same(oracle.exdot([big, 2.0 ** 970, -2.0 ** 900], [1, 1, 1]), big)
    assert oracle.exdot([-big, -2.0 ** 970], [1, 1]) == -math.inf
    # products beyond the double range that cancel
    assert same(oracle.exdot([2.0 ** 1000, -2.0 ** 1000, 1.5], [2.0 ** 1000, 2.0 ** 1000, 1.0]), 1.5)


def test_zero_and_empty(oracle):
    assert same(oracle.exdot([], []), 0.0)
    assert same(oracle.exdot([0.0, -0.0], [-1.0, 5.0]), 0.0)          # +0.0, never -0.0 (Q3)
    assert same(oracle.exdot([3.0, -3.0], [7.0, 7.0]), 0.0)
    g = fi.rng(9300)
    x = g.uniform(-1, 1, 500); y = g.uniform(-1, 1, 500)
    xx = np.concatenate([x, -x]); yy = np.concatenate([y, y]); p = g.permutation(1000)
    assert same(oracle.exdot(xx[p], yy[p]), 0.0)


def test_nonfinite_semantics(oracle):
    inf, nan = math.inf, math.nan
    assert oracle.exdot([inf, 1.0], [2.0, 1.0]) == inf
    assert oracle.exdot([inf, 1.0], [-2.0, 1.0]) == -inf
    assert oracle.exdot([1.0, -inf, 3.0], [1.0, 2.0, 1.0]) == -inf
    assert math.isnan(oracle.exdot([inf, -inf], [2.0, 1.0]))
    assert math.isnan(oracle.exdot([0.0, 1.0], [inf, 1.0]))
    assert math.isnan(oracle.exdot([nan, 1.0], [2.0, 1.0]))
    # order independence of the flags
    for perm in itertools.permutations(range(3)):
        x = np.array([inf, 5.0, -inf])[list(perm)]; y = np.array([1.0, 2.0, 1.0])[list(perm)]
        assert bits(oracle.exdot(x, y)) == np.uint64(0x7FF8000000000000)


# ---------------------------------------------------------------- library special case
def test_exact_products_match_fsum(oracle):
    # 26-bit mantissas: every product is exact in binary64, so RN(sum) == math.fsum(products)
    g = fi.rng(9400)
    for n in (5, 100, 5000):
        x = np.ldexp(g.integers(-(1 << 26), 1 << 26, n).astype(np.float64), g.integers(-60, 60, n))
        y = np.ldexp(g.integers(-(1 << 26), 1 << 26, n).astype(np.float64), g.integers(-60, 60, n))
        assert same(oracle.exdot(x, y), math.fsum((x * y).tolist()))


# ---------------------------------------------------------------- invariances
def test_invariances(oracle):
    g = fi.rng(9500)
    n = 3000
    x = np.ldexp(g.uniform(-1, 1, n), g.integers(-80, 80, n))
    y = np.ldexp(g.uniform(-1, 1, n), g.integers(-80, 80, n))
    r = oracle.exdot(x, y)
    assert r != 0.0
    for _ in range(3):
        p = g.permutation(n)
        assert same(oracle.exdot(x[p], y[p]), r)                   # permutation
    assert same(oracle.exdot(y, x), r)                             # commutativity
    assert same(oracle.exdot(-x, y), -r)                           # odd symmetry
    for k in (-300, -17, 1, 250):
        assert same(oracle.exdot(np.ldexp(x, k), y), math.ldexp(r, k))   # exact power-of-two scaling
    # concatenation = integer sum of the two accumulators
    _, la, _ = oracle.exdot_digits(x[:1000], y[:1000])
    _, lb, _ = oracle.exdot_digits(x[1000:], y[1000:])
    _, lall, _ = oracle.exdot_digits(x, y)
    ia = int.from_bytes(la.tobytes(), "little"); ib = int.from_bytes(lb.tobytes(), "little")
    iall = int.from_bytes(lall.tobytes(), "little")
    assert (ia + ib) % (1 << 4352) == iall
    summed = np.frombuffer(((ia + ib) % (1 << 4352)).to_bytes(544, "little"), dtype=np.uint64)
    assert same(oracle.round_digits(summed), r)


def test_digits_are_the_exact_integer(oracle):
    # the accumulator, read as a two's complement integer scaled by 2^-2176, IS the rational sum
    g = fi.rng(9600)
    x = np.ldexp(g.uniform(-1, 1, 200), g.integers(-500, 500, 200))
    y = np.ldexp(g.uniform(-1, 1, 200), g.integers(-500, 500, 200))
    _, limbs, flags = oracle.exdot_digits(x, y)
    v = int.from_bytes(limbs.tobytes(), "little")
    if v >> 4351:
        v -= 1 << 4352
    assert Fraction(v, 1 << 2176) == frac_dot(x, y)
    assert list(flags) == [0, 0, 0]


# ---------------------------------------------------------------- config 1 families
@pytest.mark.parametrize("ci", range(1, 6))
def test_family_a_closed_form(oracle, ci):
    for k in (10, 13):
        x, y, expected = fi.dot_family_a(k, ci)
        assert same(oracle.exdot(x, y), expected)
        # and a naive floating-point dot generally fails on the ill-conditioned ones (the paper's motivation)
    x, y, expected = fi.dot_family_a(12, 5)
    assert float(np.dot(x, y)) != expected


def test_family_a_cond0_matches_rationals(oracle):
    x, y, expected = fi.dot_family_a(10, 0)
    assert expected is None
    assert same(oracle.exdot(x, y), frac_round(frac_dot(x, y)))


# ---------------------------------------------------------------- Fig. 2 of the paper
def test_fig2_integral(oracle):
    kv = {}
    for line in open(golden_path("paper_fig2_integral.txt")):
        t = line.split()
        if t and not t[0].startswith("#"):
            kv.update(dict(zip(t[0::2], t[1::2])))
    g = oracle.Grid(int(kv["Nx"]), int(kv["Ny"]), int(kv["P"]), float(kv["x1"]), float(kv["y1"]), 1, 1)
    W, _ = oracle.dg_weights(g)
    xs, ys = oracle.dg_nodes(g)
    f = (np.exp(ys)[:, None] * np.exp(xs)[None, :]).ravel()
    val = oracle.exdot(W, f)
    exact = float(kv["exact"])
    assert abs(exact - (math.e ** 2 - 1) ** 2) < 1e-13
    assert abs(val - exact) / exact < float(kv["rel_bound"])
    assert abs(val - exact) / exact > 1e-14          # P=3 quadrature is not exact for exp: a real approximation


# ---- weighted dot and exact sum (Q14) -------------------------------------------------

def test_weighted_dot_pins(oracle):
    import math
    from fractions import Fraction
    import fxinputs as fi
    rng = fi.rng(4242)
    n = 500
    # (1) small integers: every product exact, so the result is the correctly rounded exact triple sum
    x = rng.integers(-1000, 1000, n).astype(float); w = rng.integers(1, 1000, n).astype(float); y = rng.integers(-1000, 1000, n).astype(float)
    exact = sum(Fraction(a) * Fraction(b) * Fraction(c) for a, b, c in zip(x, w, y))
    assert oracle.exdot3(x, w, y) == float(exact)
    # (2) w == 1 reduces to the exact dot; (3) general case: rational brute force of sum RN(x w) y
    x, y, w = fi.uniform(1, n), fi.uniform(2, n), 0.5 + fi.uniform(3, n) ** 2
    assert oracle.exdot3(x, np.ones(n), y) == oracle.exdot(x, y)
    exact = sum(Fraction(float(a * b)) * Fraction(float(c)) for a, b, c in zip(x, w, y))
    assert oracle.exdot3(x, w, y) == float(exact)
    # (4) Fig. 2: integral of exp(x)exp(y) on [0,2]^2 as the weighted dot of f_x, volume, f_y
    g = oracle.Grid(20, 20, 3, 2.0, 2.0, 1, 1)
    W, _ = oracle.dg_weights(g)
    xs, ys = oracle.dg_nodes(g)
    fx_, fy_ = np.exp(np.broadcast_to(xs[None, :], (ys.size, xs.size))).ravel(), np.exp(np.broadcast_to(ys[:, None], (ys.size, xs.size))).ravel()
    val = oracle.exdot3(fx_, W, fy_)
    assert abs(val / (math.exp(2.0) - 1.0) ** 2 - 1.0) < 2e-12
    # (5) exact sum: brute force, permutation invariance, cancellation
    v = np.ldexp(fi.uniform(5, n), rng.integers(-60, 60, n))
    assert oracle.exsum(v) == float(sum(Fraction(float(t)) for t in v))
    assert oracle.exsum(v[::-1].copy()) == oracle.exsum(v)
    assert oracle.exsum(np.concatenate([v, -v])) == 0.0 and oracle.exsum(np.array([1e308, 1e308, -1e308])) == 1e308


def test_exdot_f32_pins(oracle):
    """binary32 inputs: rational brute force, agreement with the fp64 dot of the converted inputs, subnormals, overflow"""
    from fractions import Fraction
    import fxinputs as fi
    n = 700
    x = fi.uniform(51, n).astype(np.float32); y = (fi.uniform(52, n) * 1e3).astype(np.float32)
    x[3] = np.float32(1e-45); y[3] = np.float32(1e-40); x[5] = np.float32(3e38); y[5] = np.float32(3e38)     # subnormal*subnormal, beyond float range
    exact = sum(Fraction(float(a)) * Fraction(float(b)) for a, b in zip(x, y))
    assert oracle.exdot_f32(x, y) == float(exact)
    assert oracle.exdot_f32(x, y) == oracle.exdot(x.astype(np.float64), y.astype(np.float64))
    assert oracle.exdot_f32(x[:0], y[:0]) == 0.0
    # naive float32 accumulation loses the small terms that the exact accumulation keeps
    big = np.array([1e8, 1.0, -1e8, 1.0], dtype=np.float32)
    assert oracle.exdot_f32(big, np.ones(4, dtype=np.float32)) == 2.0


# ---------------------------------------------------------------- config 1, family B (rounding-residue cancellation)
def test_cancel_fill_against_rationals(oracle):
    """fxo_exdot_cancel_fill: every y_j = RN(RN(t_j - sigma_j)/x_j) with sigma_j recomputed from exact rationals"""
    g = fi.rng(9101)
    n, h = 160, 64
    x = np.ldexp(1.0 + g.random(n), g.integers(-30, 31, n)) * np.where(g.integers(0, 2, n) == 0, 1.0, -1.0)
    y0 = np.concatenate([np.ldexp(1.0 + g.random(h), g.integers(-30, 31, h)), np.zeros(n - h)])
    t = np.concatenate([np.zeros(h), np.ldexp(fi.uniform(9102, n - h), np.round(np.linspace(40, -40, n - h)).astype(np.int64))])
    y = oracle.exdot_cancel_fill(x, y0, h, t)
    assert np.array_equal(y[:h], y0[:h])
    run = frac_dot(x[:h], y[:h])
    for j in range(h, n):
        sigma = frac_round(run)
        want = (float(t[j]) - sigma) / float(x[j])                  # two IEEE operations, as the definition writes them
        assert same(y[j], want), j
        run += Fraction(float(x[j])) * Fraction(float(y[j]))
    # the construction does what it is for: partial sums follow t_j, the total is tiny against the terms
    assert abs(frac_round(run)) <= 2.0 * abs(t[-1]) + 1e-300
    assert same(oracle.exdot(x, y), frac_round(run))


@pytest.mark.parametrize("ci", [1, 3, 5])
def test_family_b_is_ill_conditioned_and_exact(oracle, ci):
    x, y = fi.dot_family_b(10, ci, oracle)
    val = oracle.exdot(x, y)
    assert same(val, frac_round(frac_dot(x, y)))
    cond = 2.0 * oracle.exdot(np.abs(x), np.abs(y)) / abs(val)
    assert cond >= 1e-3 * fi.COND_TARGETS[ci]                      # achieved condition number: the target's order of magnitude or more
