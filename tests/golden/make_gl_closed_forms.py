"""Writes gauss_legendre_closed_forms.txt from the textbook radicals with Python's decimal (50 digits).

Independent of oracle/ and of the CUDA path.  Run: python tests/golden/make_gl_closed_forms.py
"""
import os
from decimal import Decimal as D, getcontext

getcontext().prec = 60


def rows():
    s = lambda v: D(v).sqrt()
    yield 1, [D(0)], [D(2)]
    a = 1 / s(3)
    yield 2, [-a, a], [D(1), D(1)]
    a = s(D(3) / 5)
    yield 3, [-a, D(0), a], [D(5) / 9, D(8) / 9, D(5) / 9]
    r = D(2) / 7 * s(D(6) / 5)
    a, b = (D(3) / 7 - r).sqrt(), (D(3) / 7 + r).sqrt()
    wa, wb = (18 + s(30)) / 36, (18 - s(30)) / 36
    yield 4, [-b, -a, a, b], [wb, wa, wa, wb]
    r = 2 * s(D(10) / 7)
    a, b = (5 - r).sqrt() / 3, (5 + r).sqrt() / 3
    wa, wb = (322 + 13 * s(70)) / 900, (322 - 13 * s(70)) / 900
    yield 5, [-b, -a, D(0), a, b], [wb, wa, D(128) / 225, wa, wb]


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "gauss_legendre_closed_forms.txt")
    with open(out, "w") as f:
        f.write("# Gauss-Legendre nodes xi_k (ascending) and weights w_k on [-1,1], closed forms, 40 digits.\n")
        f.write("# written by tests/golden/make_gl_closed_forms.py (decimal arithmetic on the textbook radicals)\n")
        f.write("# P k xi w\n")
        for P, xs, ws in rows():
            for k, (x, w) in enumerate(zip(xs, ws)):
                f.write("%d %d %s %s\n" % (P, k, format(x, ".40f"), format(w, ".40f")))
