"""ctypes binding of oracle/liboracle.so (built from oracle/fxo.cpp).  TEST INFRASTRUCTURE.

Argument marshalling only; all arithmetic is in fxo.cpp.  numpy float64 arrays in, numpy out.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fxo.cpp")
_SO = os.path.join(_HERE, "liboracle.so")

PER, DIR = 0, 1
OK, MAXIT, EINVAL, EBREAKDOWN = 0, 1, -1, -4


class Grid(C.Structure):
    """grid{Nx,Ny,P,lx,ly,bcx,bcy}: domain [0,lx]x[0,ly] (Fig. 2)."""
    _fields_ = [("Nx", C.c_int32), ("Ny", C.c_int32), ("P", C.c_int32),
                ("lx", C.c_double), ("ly", C.c_double), ("bcx", C.c_int32), ("bcy", C.c_int32)]

    @property
    def n(self):
        return self.Nx * self.Ny * self.P * self.P

    @property
    def shape(self):
        return (self.Ny * self.P, self.Nx * self.P)


class Grid3(C.Structure):
    """3-D product grid (Q24): Nz planes of the 2-D grid, one node per plane in z"""
    _fields_ = [("Nx", C.c_int32), ("Ny", C.c_int32), ("Nz", C.c_int32), ("P", C.c_int32),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double), ("bcx", C.c_int32), ("bcy", C.c_int32)]

    @property
    def n(self):
        return self.Nx * self.Ny * self.Nz * self.P * self.P

    @property
    def plane(self):
        return Grid(self.Nx, self.Ny, self.P, self.lx, self.ly, self.bcx, self.bcy)


class CGInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("status", C.c_int32), ("rel_residual", C.c_double)]


def build(force=False):
    """Compile liboracle.so with g++ (contraction off, explicit fma only)."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=gnu++17", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-fPIC", "-shared",
           _SRC, "-o", _SO + ".tmp", "-lquadmath"]
    subprocess.run(cmd, check=True)
    os.replace(_SO + ".tmp", _SO)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp = C.POINTER(C.c_double)
        L.fxo_exdot.restype = C.c_double
        L.fxo_exdot.argtypes = [dp, dp, C.c_int64]
        L.fxo_exdot_digits.restype = C.c_double
        L.fxo_exdot_digits.argtypes = [dp, dp, C.c_int64, C.POINTER(C.c_uint64), C.POINTER(C.c_int32)]
        L.fxo_exdot3.restype = C.c_double
        L.fxo_exdot3.argtypes = [dp, dp, dp, C.c_int64]
        L.fxo_exdot_f32.restype = C.c_double
        L.fxo_exdot_f32.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int64]
        L.fxo_exsum.restype = C.c_double
        L.fxo_exsum.argtypes = [dp, C.c_int64]
        L.fxo_exdot_cancel_fill.restype = None
        L.fxo_exdot_cancel_fill.argtypes = [dp, dp, C.c_int64, C.c_int64, dp]
        L.fxo_round_digits.restype = C.c_double
        L.fxo_round_digits.argtypes = [C.POINTER(C.c_uint64)]
        L.fxo_axpby.restype = None
        L.fxo_axpby.argtypes = [C.c_double, dp, C.c_double, dp, C.c_int64]
        L.fxo_pointwise_dot.restype = None
        L.fxo_pointwise_dot.argtypes = [C.c_double, dp, dp, C.c_double, dp, C.c_int64]
        L.fxo_dg_tables.restype = C.c_int
        L.fxo_dg_tables.argtypes = [C.c_int32, dp]
        gp = C.POINTER(Grid)
        L.fxo_dg_weights.restype = C.c_int
        L.fxo_dg_weights.argtypes = [gp, dp, dp]
        L.fxo_dg_nodes.restype = C.c_int
        L.fxo_dg_nodes.argtypes = [gp, dp, dp]
        L.fxo_dg_matrix_1d.restype = C.c_int
        L.fxo_dg_matrix_1d.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_int32, dp, dp]
        L.fxo_dg_apply_definition.restype = C.c_int
        L.fxo_dg_apply_definition.argtypes = [gp, dp, dp, C.c_int32, dp, dp]
        L.fxo_dg_apply_canonical.restype = C.c_int
        L.fxo_dg_apply_canonical.argtypes = [gp, dp, dp, C.c_int32, dp]
        L.fxo_dg_dtables.restype = C.c_int
        L.fxo_dg_dtables.argtypes = [C.c_int32, C.c_int32, dp]
        L.fxo_dg_derivative_canonical.restype = C.c_int
        L.fxo_dg_derivative_canonical.argtypes = [gp, C.c_int32, C.c_int32, C.c_double, dp, C.c_double, dp]
        L.fxo_dg_derivative_matrix_1d.restype = C.c_int
        L.fxo_dg_derivative_matrix_1d.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_int32, dp]
        L.fxo_dg_derivative_definition.restype = C.c_int
        L.fxo_dg_derivative_definition.argtypes = [gp, C.c_int32, C.c_int32, C.c_double, dp, C.c_double, dp, dp, dp]
        L.fxo_pointwise_dot2.restype = None
        L.fxo_pointwise_dot2.argtypes = [C.c_double, dp, dp, C.c_double, dp, dp, C.c_double, dp, C.c_int64]
        L.fxo_arakawa.restype = C.c_int
        L.fxo_arakawa.argtypes = [gp, dp, dp, dp]
        L.fxo_cg_solve.restype = C.c_int
        L.fxo_cg_solve.argtypes = [gp, dp, dp, dp, C.c_double, C.c_int32, C.POINTER(CGInfo)]
        g3 = C.POINTER(Grid3)
        L.fxo_dg3_weights.restype = C.c_int
        L.fxo_dg3_weights.argtypes = [g3, dp, dp]
        L.fxo_dg3_apply_canonical.restype = C.c_int
        L.fxo_dg3_apply_canonical.argtypes = [g3, dp, dp, C.c_int32, dp]
        L.fxo_dg3_apply_definition.restype = C.c_int
        L.fxo_dg3_apply_definition.argtypes = [g3, dp, dp, C.c_int32, dp, dp]
        L.fxo_cg3_solve.restype = C.c_int
        L.fxo_cg3_solve.argtypes = [g3, dp, dp, dp, C.c_double, C.c_int32, C.POINTER(CGInfo)]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def exdot(x, y):
    x, y = _f64(x).ravel(), _f64(y).ravel()
    assert x.size == y.size
    return float(lib().fxo_exdot(_p(x), _p(y), x.size))


def exdot3(x, w, y):
    """weighted dot RN(sum RN(x_i*w_i)*y_i) (Q14)"""
    x, w, y = _f64(x).ravel(), _f64(w).ravel(), _f64(y).ravel()
    assert x.size == w.size == y.size
    return float(lib().fxo_exdot3(_p(x), _p(w), _p(y), x.size))


def exdot_f32(x, y):
    """RN_double(sum x_i*y_i) for float32 inputs"""
    x = np.ascontiguousarray(x, dtype=np.float32).ravel(); y = np.ascontiguousarray(y, dtype=np.float32).ravel()
    assert x.size == y.size
    fp = C.POINTER(C.c_float)
    return float(lib().fxo_exdot_f32(x.ctypes.data_as(fp), y.ctypes.data_as(fp), x.size))


def exsum(x):
    x = _f64(x).ravel()
    return float(lib().fxo_exsum(_p(x), x.size))


def exdot_digits(x, y):
    """-> (value, limbs uint64[68] two's complement with limb k weighing 2^(64k-2176), flags int32[3])"""
    x, y = _f64(x).ravel(), _f64(y).ravel()
    assert x.size == y.size
    limbs = np.zeros(68, dtype=np.uint64)
    flags = np.zeros(3, dtype=np.int32)
    v = lib().fxo_exdot_digits(_p(x), _p(y), x.size, limbs.ctypes.data_as(C.POINTER(C.c_uint64)),
                               flags.ctypes.data_as(C.POINTER(C.c_int32)))
    return float(v), limbs, flags


def exdot_cancel_fill(x, y, start, t):
    """Family B of config 1: y[j] = RN(RN(t[j] - RN(sum_{i<j} x_i y_i)) / x[j]) for j >= start, in place; -> y"""
    x, t = _f64(x).ravel(), _f64(t).ravel()
    y = np.array(y, dtype=np.float64).ravel()
    assert x.size == y.size == t.size and 0 <= start <= x.size
    lib().fxo_exdot_cancel_fill(_p(x), _p(y), int(start), x.size, _p(t))
    return y


def round_digits(limbs):
    limbs = np.ascontiguousarray(limbs, dtype=np.uint64)
    assert limbs.size == 68
    return float(lib().fxo_round_digits(limbs.ctypes.data_as(C.POINTER(C.c_uint64))))


def axpby(alpha, x, beta, y):
    """returns the updated copy of y:  y <- alpha*x + beta*y in canonical order"""
    x = _f64(x).ravel()
    y = np.array(y, dtype=np.float64).ravel().copy()
    assert x.size == y.size
    lib().fxo_axpby(alpha, _p(x), beta, _p(y), x.size)
    return y


def pointwise_dot(alpha, x1, x2, beta, y):
    x1, x2 = _f64(x1).ravel(), _f64(x2).ravel()
    y = np.array(y, dtype=np.float64).ravel().copy()
    assert x1.size == x2.size == y.size
    lib().fxo_pointwise_dot(alpha, _p(x1), _p(x2), beta, _p(y), y.size)
    return y


def dg_tables(P):
    """-> dict(xi,w,L,R,B: [P]; T0,T0L,WW,D: [P,P])"""
    out = np.zeros(5 * P + 4 * P * P)
    rc = lib().fxo_dg_tables(P, _p(out))
    if rc != 0:
        raise ValueError("P out of range")
    d, o = {}, 0
    for name in ("xi", "w", "L", "R", "B"):
        d[name] = out[o:o + P].copy(); o += P
    for name in ("T0", "T0L", "WW", "D"):
        d[name] = out[o:o + P * P].reshape(P, P).copy(); o += P * P
    return d


def dg_weights(g):
    W = np.zeros(g.n); V = np.zeros(g.n)
    if lib().fxo_dg_weights(C.byref(g), _p(W), _p(V)) != 0:
        raise ValueError("bad grid")
    return W, V


def dg_nodes(g):
    xs = np.zeros(g.Nx * g.P); ys = np.zeros(g.Ny * g.P)
    if lib().fxo_dg_nodes(C.byref(g), _p(xs), _p(ys)) != 0:
        raise ValueError("bad grid")
    return xs, ys


def dg_matrix_1d(N, P, h, bc):
    n = N * P
    F = np.zeros((n, n)); J = np.zeros((n, n))
    if lib().fxo_dg_matrix_1d(N, P, h, bc, _p(F), _p(J)) != 0:
        raise ValueError("bad arguments")
    return F, J


def dg_apply_definition(g, chi, x, normed=False):
    chi, x = _f64(chi).ravel(), _f64(x).ravel()
    assert chi.size == g.n and x.size == g.n
    y = np.zeros(g.n); s = np.zeros(g.n)
    if lib().fxo_dg_apply_definition(C.byref(g), _p(chi), _p(x), int(normed), _p(y), _p(s)) != 0:
        raise ValueError("bad grid")
    return y, s


def dg_apply_canonical(g, chi, x, normed=False):
    chi, x = _f64(chi).ravel(), _f64(x).ravel()
    assert chi.size == g.n and x.size == g.n
    y = np.zeros(g.n)
    if lib().fxo_dg_apply_canonical(C.byref(g), _p(chi), _p(x), int(normed), _p(y)) != 0:
        raise ValueError("bad grid")
    return y


FORWARD, BACKWARD, CENTERED = 0, 1, 2


def dg_dtables(P, flux):
    """-> dict(TT: [2,P,P] (interior / first cell of a DIR line), cN: [P], cP: [P])"""
    out = np.zeros(2 * P * P + 2 * P)
    if lib().fxo_dg_dtables(P, flux, _p(out)) != 0:
        raise ValueError("bad arguments")
    return dict(TT=out[:2 * P * P].reshape(2, P, P).copy(), cN=out[2 * P * P:2 * P * P + P].copy(), cP=out[2 * P * P + P:].copy())


def dg_derivative_canonical(g, direction, flux, alpha, x, beta, y):
    """y <- alpha * M x + beta * y in the canonical fp64 order (returns the updated copy of y)"""
    x = _f64(x).ravel()
    y = np.array(y, dtype=np.float64).ravel().copy()
    assert x.size == g.n and y.size == g.n
    if lib().fxo_dg_derivative_canonical(C.byref(g), direction, flux, alpha, _p(x), beta, _p(y)) != 0:
        raise ValueError("bad arguments")
    return y


def dg_derivative_matrix_1d(N, P, h, bc, flux):
    n = N * P
    M = np.zeros((n, n))
    if lib().fxo_dg_derivative_matrix_1d(N, P, h, bc, flux, _p(M)) != 0:
        raise ValueError("bad arguments")
    return M


def dg_derivative_definition(g, direction, flux, alpha, x, beta, y):
    """-> (alpha*M x + beta*y from explicit 113-bit matrices, error scale)"""
    x, y = _f64(x).ravel(), _f64(y).ravel()
    out = np.zeros(g.n); sc = np.zeros(g.n)
    if lib().fxo_dg_derivative_definition(C.byref(g), direction, flux, alpha, _p(x), beta, _p(y), _p(out), _p(sc)) != 0:
        raise ValueError("bad arguments")
    return out, sc


def pointwise_dot2(alpha, x1, y1, beta, x2, y2, gamma, z):
    """z <- alpha*x1*y1 + beta*x2*y2 + gamma*z in the canonical order (returns the updated copy of z)"""
    x1, y1, x2, y2 = (_f64(a).ravel() for a in (x1, y1, x2, y2))
    z = np.array(z, dtype=np.float64).ravel().copy()
    lib().fxo_pointwise_dot2(alpha, _p(x1), _p(y1), beta, _p(x2), _p(y2), gamma, _p(z), z.size)
    return z


def arakawa(g, f, gg):
    """Arakawa bracket {f,g} with centred dG derivatives (nine canonical calls)"""
    f, gg = _f64(f).ravel(), _f64(gg).ravel()
    out = np.zeros(g.n)
    if lib().fxo_arakawa(C.byref(g), _p(f), _p(gg), _p(out)) != 0:
        raise ValueError("bad grid")
    return out


def cg_solve(g, chi, rho, phi0, tol, maxit):
    """-> (phi, CGInfo)"""
    chi, rho = _f64(chi).ravel(), _f64(rho).ravel()
    phi = np.array(phi0, dtype=np.float64).ravel().copy()
    assert chi.size == g.n and rho.size == g.n and phi.size == g.n
    info = CGInfo()
    lib().fxo_cg_solve(C.byref(g), _p(chi), _p(rho), _p(phi), tol, maxit, C.byref(info))
    return phi, info


# ---- 3-D product grids (Q24) ----------------------------------------------------------------------------
def dg3_weights(g):
    W = np.empty(g.n); V = np.empty(g.n)
    assert lib().fxo_dg3_weights(C.byref(g), _p(W), _p(V)) == 0
    return W, V


def dg3_apply_canonical(g, chi, x, normed=False):
    chi, x = _f64(chi).ravel(), _f64(x).ravel()
    assert chi.size == x.size == g.n
    y = np.empty(g.n)
    assert lib().fxo_dg3_apply_canonical(C.byref(g), _p(chi), _p(x), 1 if normed else 0, _p(y)) == 0
    return y


def dg3_apply_definition(g, chi, x, normed=False):
    chi, x = _f64(chi).ravel(), _f64(x).ravel()
    assert chi.size == x.size == g.n
    y = np.empty(g.n); sc = np.empty(g.n)
    assert lib().fxo_dg3_apply_definition(C.byref(g), _p(chi), _p(x), 1 if normed else 0, _p(y), _p(sc)) == 0
    return y, sc


def cg3_solve(g, chi, rho, phi0, tol, maxit):
    chi, rho = _f64(chi).ravel(), _f64(rho).ravel()
    phi = np.array(phi0, dtype=np.float64).ravel().copy()
    assert chi.size == rho.size == phi.size == g.n
    info = CGInfo()
    lib().fxo_cg3_solve(C.byref(g), _p(chi), _p(rho), _p(phi), float(tol), int(maxit), C.byref(info))
    return phi, info
