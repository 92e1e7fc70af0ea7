// fx_tables.cpp -- host-side reference-element tables of the dG kernels (compiled with g++, libquadmath).
//
// Gauss-Legendre nodes/weights for P = 1..5 from their closed-form radicals, Lagrange-basis derivative and
// boundary-trace tables from the barycentric formula, all in 113-bit arithmetic, each entry rounded ONCE to
// fp64 (DESIGN.md 3.4 "Tables").  Fig. 2 of the paper fixes Gauss-Legendre nodes; P is the
// number of polynomial coefficients per cell and direction.
//
// This file is part of the product (libfx.so) and shares nothing with oracle/: the oracle finds the nodes by
// Newton iteration on the Legendre recurrence and differentiates the Lagrange basis by products of node
// differences; tests/test_abi.py asserts that the two independently derived tables agree bit for bit.

#include <quadmath.h>
#include <stdint.h>

#include <mutex>

#include "fx_tables.h"

typedef __float128 q;

namespace {

void gauss_legendre(int P, q* xi, q* w) {
    switch (P) {
    case 1: xi[0] = 0; w[0] = 2; break;
    case 2: { q a = 1 / sqrtq((q)3); xi[0] = -a; xi[1] = a; w[0] = w[1] = 1; } break;
    case 3: { q a = sqrtq((q)3 / 5); xi[0] = -a; xi[1] = 0; xi[2] = a; w[0] = w[2] = (q)5 / 9; w[1] = (q)8 / 9; } break;
    case 4: {
        q s = (q)2 / 7 * sqrtq((q)6 / 5), r30 = sqrtq((q)30);
        q a = sqrtq((q)3 / 7 - s), b = sqrtq((q)3 / 7 + s);
        xi[0] = -b; xi[1] = -a; xi[2] = a; xi[3] = b;
        w[0] = w[3] = (18 - r30) / 36; w[1] = w[2] = (18 + r30) / 36;
    } break;
    case 5: {
        q s = 2 * sqrtq((q)10 / 7), r70 = sqrtq((q)70);
        q a = sqrtq(5 - s) / 3, b = sqrtq(5 + s) / 3;
        xi[0] = -b; xi[1] = -a; xi[2] = 0; xi[3] = a; xi[4] = b;
        w[0] = w[4] = (322 - 13 * r70) / 900; w[1] = w[3] = (322 + 13 * r70) / 900; w[2] = (q)128 / 225;
    } break;
    }
}

// entries of these tables are either exactly zero in exact arithmetic or of order 0.01..10
double rnd(q v) { q a = v < 0 ? -v : v; return a < 1e-25Q ? 0.0 : (double)v; }

}  // namespace

struct Ref { q xi[FX_PMAX], w[FX_PMAX], L[FX_PMAX], R[FX_PMAX], D[FX_PMAX][FX_PMAX]; };
static void reference_element(int P, Ref& r);

// forward: T = D - W^-1 R R^T (+ W^-1 L L^T in the first cell of a Dirichlet line); backward: -W^-1 T^T W; centred: mean
// The 113-bit derivation costs microseconds of host time; every launch needs the tables, so they are computed once.
static int make_dtables_uncached(int P, int flux, fx_dtables* d);
static int make_tables_uncached(int P, fx_tables* t);
static std::once_flag g_once;
static fx_tables g_tab[FX_PMAX + 1];
static fx_dtables g_dtab[FX_PMAX + 1][4];
static void fill_cache() {
    for (int P = 1; P <= FX_PMAX; ++P) {
        make_tables_uncached(P, &g_tab[P]);
        for (int f = 0; f < 4; ++f) make_dtables_uncached(P, f, &g_dtab[P][f]);
    }
}
extern "C" int fx_make_dtables(int P, int flux, fx_dtables* d) {
    if (P < 1 || P > FX_PMAX || flux < 0 || flux > 3) return -1;
    std::call_once(g_once, fill_cache);
    *d = g_dtab[P][flux];
    return 0;
}
extern "C" int fx_make_tables(int P, fx_tables* t) {
    if (P < 1 || P > FX_PMAX) return -1;
    std::call_once(g_once, fill_cache);
    *t = g_tab[P];
    return 0;
}

static int make_dtables_uncached(int P, int flux, fx_dtables* d) {
    if (P < 1 || P > FX_PMAX || flux < 0 || flux > 3) return -1;
    Ref r; reference_element(P, r);
    if (flux == 3) {             // the jump matrix: diagonal block R R^T + L L^T, neighbour traces with -R (next) and -L (previous)
        for (int v = 0; v < 2; ++v)
            for (int k = 0; k < P; ++k)
                for (int m = 0; m < P; ++m) d->TT[v][k][m] = rnd(r.R[k] * r.R[m] + r.L[k] * r.L[m]);
        for (int k = 0; k < P; ++k) { d->cN[k] = rnd(-r.R[k]); d->cP[k] = rnd(-r.L[k]); }
        return 0;
    }
    for (int v = 0; v < 2; ++v)
        for (int k = 0; k < P; ++k)
            for (int m = 0; m < P; ++m) {
                q tkm = r.D[k][m] - r.R[k] * r.R[m] / r.w[k], tmk = r.D[m][k] - r.R[m] * r.R[k] / r.w[m];
                if (v) { tkm += r.L[k] * r.L[m] / r.w[k]; tmk += r.L[m] * r.L[k] / r.w[m]; }
                const q f = tkm, b = -tmk * r.w[m] / r.w[k];
                d->TT[v][k][m] = rnd(flux == 0 ? f : flux == 1 ? b : (f + b) / 2);
            }
    for (int k = 0; k < P; ++k) {
        const q cn = r.R[k] / r.w[k], cp = -r.L[k] / r.w[k];
        d->cN[k] = flux == 0 ? rnd(cn) : flux == 1 ? 0.0 : rnd(cn / 2);
        d->cP[k] = flux == 0 ? 0.0 : flux == 1 ? rnd(cp) : rnd(cp / 2);
    }
    return 0;
}

static void reference_element(int P, Ref& r) {
    q lam[FX_PMAX];
    q (&xi)[FX_PMAX] = r.xi; q (&w)[FX_PMAX] = r.w; q (&L)[FX_PMAX] = r.L; q (&R)[FX_PMAX] = r.R; q (&D)[FX_PMAX][FX_PMAX] = r.D;
    gauss_legendre(P, xi, w);
    for (int m = 0; m < P; ++m) {                      // barycentric weights
        q d = 1;
        for (int j = 0; j < P; ++j) if (j != m) d *= (xi[m] - xi[j]);
        lam[m] = 1 / d;
    }
    for (int m = 0; m < P; ++m) {                      // l_m(-1), l_m(+1)
        q a = lam[m], b = lam[m];
        for (int j = 0; j < P; ++j) if (j != m) { a *= (-1 - xi[j]); b *= (1 - xi[j]); }
        L[m] = a; R[m] = b;
    }
    for (int k = 0; k < P; ++k) {                      // D[k][m] = l_m'(xi_k)
        q diag = 0;
        for (int m = 0; m < P; ++m) if (m != k) { D[k][m] = (lam[m] / lam[k]) / (xi[k] - xi[m]); diag -= D[k][m]; }
        D[k][k] = diag;
    }
}

static int make_tables_uncached(int P, fx_tables* t) {
    if (P < 1 || P > FX_PMAX) return -1;
    Ref r; reference_element(P, r);
    q (&xi)[FX_PMAX] = r.xi; q (&w)[FX_PMAX] = r.w; q (&L)[FX_PMAX] = r.L; q (&R)[FX_PMAX] = r.R; q (&D)[FX_PMAX][FX_PMAX] = r.D;
    t->P = P;
    for (int k = 0; k < P; ++k) {
        t->xi[k] = rnd(xi[k]); t->w[k] = (double)w[k]; t->L[k] = rnd(L[k]); t->R[k] = rnd(R[k]);
        t->B[k] = rnd(R[k] / w[k]);
        for (int m = 0; m < P; ++m) {
            q t0 = D[k][m] - R[k] * R[m] / w[k];
            t->T0[k][m] = rnd(t0);
            t->T0L[k][m] = rnd(t0 + L[k] * L[m] / w[k]);
            t->WW[k][m] = (double)(w[k] * w[m]);
            t->D[k][m] = rnd(D[k][m]);
        }
    }
    return 0;
}
