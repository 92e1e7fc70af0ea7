"""paper_1807_01971_b200 -- thin Python binding of libfx.so (C ABI: include/fx.h).

Argument marshalling only: every step of the hot path (exact dot, axpby, pointwise_dot, dG elliptic apply, CG) runs in
the hand-written sm_100a kernels of csrc/.  torch is used for device memory and streams.  There is no CPU fallback and
nothing here imports oracle/: if the library cannot be built/loaded or no CUDA device is present, calls raise.
"""
import ctypes as C
import os

from . import build as _build

PER, DIR, NEU, DIR_NEU, NEU_DIR = 0, 1, 2, 3, 4      # fx_bc (include/fx.h)
OK, MAXIT, EINVAL, ECUDA, ENOMEM, EBREAKDOWN = 0, 1, -1, -2, -3, -4

_HERE = os.path.dirname(os.path.abspath(__file__))


class Grid(C.Structure):
    """fx_grid: Nx x Ny cells on [0,lx] x [0,ly], P Gauss-Legendre nodes per cell and direction (Fig. 2)."""
    _fields_ = [("Nx", C.c_int32), ("Ny", C.c_int32), ("P", C.c_int32),
                ("lx", C.c_double), ("ly", C.c_double), ("bcx", C.c_int32), ("bcy", C.c_int32)]

    @property
    def n(self):
        return self.Nx * self.Ny * self.P * self.P


class Grid3(C.Structure):
    """fx_grid3: 3-D product grid, Nz planes of the 2-D grid with one node per plane in z (include/fx.h; Q24)."""
    _fields_ = [("Nx", C.c_int32), ("Ny", C.c_int32), ("Nz", C.c_int32), ("P", C.c_int32),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double), ("bcx", C.c_int32), ("bcy", C.c_int32)]

    @property
    def n(self):
        return self.Nx * self.Ny * self.Nz * self.P * self.P


class CGInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("status", C.c_int32), ("rel_residual", C.c_double)]


class FxError(RuntimeError):
    pass


_lib = None
_vp, _dp = C.c_void_p, C.POINTER(C.c_double)

# name -> (restype, argtypes): every symbol include/fx.h declares
_SIGNATURES = {
    "fx_set_stream": (C.c_int, [_vp]),
    "fx_last_error": (C.c_char_p, []),
    "fx_shutdown": (None, []),
    "fx_set_launch": (C.c_int, [C.c_int32, C.c_int32, C.c_int32]),
    "fx_set_cg_fused": (C.c_int, [C.c_int32]),
    "fx_set_dg_path": (C.c_int, [C.c_int32]),
    "fx_exdot": (C.c_double, [_vp, _vp, C.c_int64]),
    "fx_exdot_async": (C.c_int, [_vp, _vp, C.c_int64, _vp]),
    "fx_exdot_static": (C.c_int, [_vp, _vp, C.c_int64, _vp, _vp]),
    "fx_exdot_digits": (C.c_int, [_vp, _vp, C.c_int64, _vp, _vp, _vp]),
    "fx_exdot_host": (C.c_double, [_vp, _vp, C.c_int64]),
    "fx_exdot3": (C.c_double, [_vp, _vp, _vp, C.c_int64]),
    "fx_exsum": (C.c_double, [_vp, C.c_int64]),
    "fx_exdot_f32": (C.c_double, [_vp, _vp, C.c_int64]),
    "fx_axpby": (C.c_int, [C.c_double, _vp, C.c_double, _vp, C.c_int64]),
    "fx_pointwise_dot": (C.c_int, [C.c_double, _vp, _vp, C.c_double, _vp, C.c_int64]),
    "fx_pointwise_dot2": (C.c_int, [C.c_double, _vp, _vp, C.c_double, _vp, _vp, C.c_double, _vp, C.c_int64]),
    "fx_arakawa": (C.c_int, [C.POINTER(Grid), _vp, _vp, _vp]),
    "fx_dg_elliptic_apply": (C.c_int, [C.POINTER(Grid), _vp, _vp, _vp]),
    "fx_dg_elliptic_apply_sym": (C.c_int, [C.POINTER(Grid), _vp, _vp, _vp]),
    "fx_dg_weights": (C.c_int, [C.POINTER(Grid), _vp, _vp]),
    "fx_dg_tables": (C.c_int, [C.c_int32, _dp]),
    "fx_dg_derivative": (C.c_int, [C.POINTER(Grid), C.c_int32, C.c_int32, C.c_double, _vp, C.c_double, _vp]),
    "fx_dg_dtables": (C.c_int, [C.c_int32, C.c_int32, _dp]),
    "fx_cg_solve": (C.c_int, [C.POINTER(Grid), _vp, _vp, _vp, C.c_double, C.c_int32, C.POINTER(CGInfo)]),
    "fx_cg_solve_host": (C.c_int, [C.POINTER(Grid), _vp, _vp, _vp, C.c_double, C.c_int32, C.POINTER(CGInfo)]),
    "fx_cg_profile": (C.c_int, [C.c_int32]),
    "fx_cg_last_profile": (C.c_int, [_dp, C.POINTER(C.c_int32)]),
    "fx_time_primitive": (C.c_int, [C.c_int32, C.POINTER(Grid), _vp, _vp, _vp, C.c_int64, C.c_int32, _dp]),
    "fx_launch_count": (C.c_int64, []),
    "fx_exdot_stats": (C.c_int, [_vp, C.c_int32]),
    "fx_dg3_elliptic_apply": (C.c_int, [C.POINTER(Grid3), _vp, _vp, _vp, C.c_int32]),
    "fx_dg3_weights": (C.c_int, [C.POINTER(Grid3), _vp, _vp]),
    "fx_cg3_solve": (C.c_int, [C.POINTER(Grid3), _vp, _vp, _vp, C.c_double, C.c_int32, C.POINTER(CGInfo)]),
    "fx_create": (C.c_int, [C.POINTER(_vp), C.c_int32, _vp]),
    "fx_destroy": (None, [_vp]),
}
# the context forms: NAME_ex(ctx, <the plain call's arguments> [, result_host for the value-returning reductions])
for _n in ("fx_dg3_elliptic_apply", "fx_dg3_weights", "fx_cg3_solve", "fx_exdot_stats", "fx_set_stream", "fx_set_launch", "fx_set_cg_fused", "fx_set_dg_path", "fx_exdot_async", "fx_exdot_digits", "fx_axpby",
           "fx_pointwise_dot", "fx_pointwise_dot2", "fx_arakawa", "fx_dg_elliptic_apply", "fx_dg_elliptic_apply_sym", "fx_dg_weights",
           "fx_dg_derivative", "fx_cg_solve", "fx_cg_solve_host", "fx_cg_profile", "fx_cg_last_profile", "fx_time_primitive"):
    _SIGNATURES[_n + "_ex"] = (C.c_int, [_vp] + _SIGNATURES[_n][1])
for _n in ("fx_exdot_host", "fx_exdot3", "fx_exsum", "fx_exdot_f32"):
    _SIGNATURES[_n + "_ex"] = (C.c_int, [_vp] + _SIGNATURES[_n][1] + [_dp])
_SIGNATURES["fx_exdot_ex"] = (C.c_int, [_vp, _vp, _vp, C.c_int64, _dp, _vp])


def lib_path():
    return os.path.join(_HERE, "libfx.so")


def lib():
    """Load libfx.so (building it in-tree first if it is missing or stale).  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError if the ABI lost a symbol
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc, what):
    if rc < 0:
        raise FxError("%s failed (%d): %s" % (what, rc, lib().fx_last_error().decode()))
    return rc


def _ptr(t, n=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    if n is not None and t.numel() != n:
        raise ValueError("tensor has %d elements, expected %d" % (t.numel(), n))
    return t.data_ptr()


def _use_torch_stream():
    import torch
    _check(lib().fx_set_stream(torch.cuda.current_stream().cuda_stream), "fx_set_stream")


class Context:
    """An explicit fx_ctx (include/fx.h "contexts"): one device, one stream, its own scratch.  The module-level functions use
    the default context of the current device; this class exposes the same calls on a context of its own."""

    def __init__(self, device=None, stream=None):
        import torch
        self._h = _vp()
        dev = torch.cuda.current_device() if device is None else int(device)
        st = stream.cuda_stream if hasattr(stream, "cuda_stream") else (stream or 0)
        _check(lib().fx_create(C.byref(self._h), dev, st), "fx_create")

    def destroy(self):
        if self._h:
            lib().fx_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_stream(self, stream):
        st = stream.cuda_stream if hasattr(stream, "cuda_stream") else (stream or 0)
        _check(lib().fx_set_stream_ex(self._h, st), "fx_set_stream_ex")

    def set_dg_path(self, path):
        _check(lib().fx_set_dg_path_ex(self._h, int(path)), "fx_set_dg_path_ex")

    def set_cg_fused(self, fused):
        _check(lib().fx_set_cg_fused_ex(self._h, int(fused)), "fx_set_cg_fused_ex")

    def exdot(self, x, y, out=None):
        """host float (synchronises) or, with `out` (a 1-element float64 CUDA tensor), the stream-ordered device form"""
        n = x.numel()
        if out is not None:
            _check(lib().fx_exdot_ex(self._h, _ptr(x), _ptr(y, n), n, None, _ptr(out, 1)), "fx_exdot_ex")
            return out
        v = C.c_double(0.0)
        _check(lib().fx_exdot_ex(self._h, _ptr(x), _ptr(y, n), n, C.byref(v), None), "fx_exdot_ex")
        return v.value

    def exsum(self, x):
        v = C.c_double(0.0)
        _check(lib().fx_exsum_ex(self._h, _ptr(x), x.numel(), C.byref(v)), "fx_exsum_ex")
        return v.value

    def axpby(self, alpha, x, beta, y):
        n = x.numel()
        _check(lib().fx_axpby_ex(self._h, float(alpha), _ptr(x), float(beta), _ptr(y, n), n), "fx_axpby_ex")

    def pointwise_dot(self, alpha, x1, x2, beta, y):
        n = x1.numel()
        _check(lib().fx_pointwise_dot_ex(self._h, float(alpha), _ptr(x1), _ptr(x2, n), float(beta), _ptr(y, n), n), "fx_pointwise_dot_ex")

    def dg_elliptic_apply(self, grid, chi, x, y, sym=False):
        fn = lib().fx_dg_elliptic_apply_sym_ex if sym else lib().fx_dg_elliptic_apply_ex
        _check(fn(self._h, C.byref(grid), _ptr(chi, grid.n), _ptr(x, grid.n), _ptr(y, grid.n)), "fx_dg_elliptic_apply_ex")

    def cg_solve(self, grid, chi, rho, phi, tol, maxit):
        info = CGInfo()
        rc = lib().fx_cg_solve_ex(self._h, C.byref(grid), _ptr(chi, grid.n), _ptr(rho, grid.n), _ptr(phi, grid.n), float(tol), int(maxit),
                                  C.byref(info))
        _check(rc, "fx_cg_solve_ex")
        return info


def make_grid(Nx, Ny, P, lx, ly, bcx, bcy):
    return Grid(int(Nx), int(Ny), int(P), float(lx), float(ly), int(bcx), int(bcy))


def set_launch(kernel_id, grid_dim=0, block_dim=0):
    _check(lib().fx_set_launch(kernel_id, grid_dim, block_dim), "fx_set_launch")


def set_cg_fused(fused):
    _check(lib().fx_set_cg_fused(int(fused)), "fx_set_cg_fused")


def set_dg_path(path):
    _check(lib().fx_set_dg_path(int(path)), "fx_set_dg_path")


def launch_count():
    return int(lib().fx_launch_count())


def exdot(x, y):
    """RN(sum x_i*y_i) as a Python float (synchronises).  PAPER.md:170-176."""
    _use_torch_stream()
    n = x.numel()
    v = lib().fx_exdot(_ptr(x), _ptr(y, n), n)
    if v != v and lib().fx_last_error():
        raise FxError(lib().fx_last_error().decode())
    return v


def exdot_stats(reset=False):
    """slow-path census of the exact reductions since the last reset (fx.h): dict(deposit_double, deposit_product, window_moves)"""
    out = (C.c_uint64 * 4)()
    _check(lib().fx_exdot_stats(out, 1 if reset else 0), "fx_exdot_stats")
    return dict(deposit_double=int(out[0]), deposit_product=int(out[1]), window_moves=int(out[2]))


def exdot3(x, w, y):
    """weighted dot RN(sum RN(x_i*w_i)*y_i) (Q14); synchronises"""
    _use_torch_stream()
    n = x.numel()
    v = lib().fx_exdot3(_ptr(x), _ptr(w, n), _ptr(y, n), n)
    if v != v and lib().fx_last_error():
        raise FxError(lib().fx_last_error().decode())
    return v


def exsum(x):
    """exactly rounded sum (EXSUM); synchronises"""
    _use_torch_stream()
    v = lib().fx_exsum(_ptr(x), x.numel())
    if v != v and lib().fx_last_error():
        raise FxError(lib().fx_last_error().decode())
    return v


def exdot_f32(x, y):
    """RN_double(sum x_i*y_i) for contiguous float32 CUDA tensors; synchronises"""
    import torch
    _use_torch_stream()
    assert x.is_cuda and y.is_cuda and x.dtype == torch.float32 and y.dtype == torch.float32 and x.is_contiguous() and y.is_contiguous()
    assert x.numel() == y.numel()
    v = lib().fx_exdot_f32(x.data_ptr(), y.data_ptr(), x.numel())
    if v != v and lib().fx_last_error():
        raise FxError(lib().fx_last_error().decode())
    return v


def exdot_async(x, y, out):
    """Stream-ordered form: writes the double into out[0] (a float64 CUDA tensor)."""
    _use_torch_stream()
    n = x.numel()
    _check(lib().fx_exdot_async(_ptr(x), _ptr(y, n), n, _ptr(out)), "fx_exdot_async")
    return out


EXDOT_STATIC_MAX_N = 1 << 28


def exdot_static(x, y, out, stream=None):
    """Allocation-free exact dot (fx_exdot_static): no context, no work space, scratch in a static device array of the
    library; n <= EXDOT_STATIC_MAX_N; writes out[0] (float64 CUDA tensor) on `stream` (default: torch's current stream).
    Calls that overlap on the GPU race on the shared scratch."""
    import torch
    st = torch.cuda.current_stream().cuda_stream if stream is None else (stream.cuda_stream if hasattr(stream, "cuda_stream") else stream)
    n = x.numel()
    _check(lib().fx_exdot_static(_ptr(x), _ptr(y, n), n, _ptr(out), st), "fx_exdot_static")
    return out


def exdot_digits(x, y):
    """-> (value, limbs uint64[68] numpy, flags int32[3] numpy): the long accumulator itself."""
    import numpy as np
    _use_torch_stream()
    n = x.numel()
    limbs = np.zeros(68, dtype=np.uint64)
    flags = np.zeros(3, dtype=np.int32)
    res = C.c_double(0.0)
    _check(lib().fx_exdot_digits(_ptr(x), _ptr(y, n), n, limbs.ctypes.data, flags.ctypes.data, C.addressof(res)), "fx_exdot_digits")
    return res.value, limbs, flags


def exdot_host(x, y):
    """x, y: CPU float64 tensors (pinned for full speed) or numpy arrays; copies inside the call."""
    n, px, py = _host_ptrs(x, y)
    v = lib().fx_exdot_host(px, py, n)
    if v != v and lib().fx_last_error():
        raise FxError(lib().fx_last_error().decode())
    return v


def _host_ptrs(*arrs):
    import numpy as np
    import torch
    ptrs, n = [], None
    for a in arrs:
        if isinstance(a, torch.Tensor):
            assert (not a.is_cuda) and a.dtype == torch.float64 and a.is_contiguous()
            ptrs.append(a.data_ptr()); m = a.numel()
        else:
            assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous
            ptrs.append(a.ctypes.data); m = a.size
        assert n is None or n == m
        n = m
    return (n, *ptrs)


def axpby(alpha, x, beta, y):
    """y <- alpha*x + beta*y in the canonical order of DESIGN.md 3.2 (in place; returns y).  PAPER.md:184-186."""
    _use_torch_stream()
    n = y.numel()
    _check(lib().fx_axpby(float(alpha), _ptr(x, n), float(beta), _ptr(y), n), "fx_axpby")
    return y


def pointwise_dot(alpha, x1, x2, beta, y):
    """y <- alpha*x1*x2 + beta*y (in place; returns y).  PAPER.md:238."""
    _use_torch_stream()
    n = y.numel()
    _check(lib().fx_pointwise_dot(float(alpha), _ptr(x1, n), _ptr(x2, n), float(beta), _ptr(y), n), "fx_pointwise_dot")
    return y


def pointwise_dot2(alpha, x1, y1, beta, x2, y2, gamma, z):
    """z <- alpha*x1*y1 + beta*x2*y2 + gamma*z (in place; returns z).  PAPER.md:414."""
    _use_torch_stream()
    n = z.numel()
    _check(lib().fx_pointwise_dot2(float(alpha), _ptr(x1, n), _ptr(y1, n), float(beta), _ptr(x2, n), _ptr(y2, n), float(gamma), _ptr(z), n),
           "fx_pointwise_dot2")
    return z


def arakawa(grid, f, g, out):
    """out = {f, g}: Arakawa bracket with centred dG derivatives (nine primitive calls).  PAPER.md:240, Fig. 6a."""
    _use_torch_stream()
    _check(lib().fx_arakawa(C.byref(grid), _ptr(f, grid.n), _ptr(g, grid.n), _ptr(out, grid.n)), "fx_arakawa")
    return out


def dg_elliptic_apply(grid, chi, x, y, sym=False):
    """y = A x (normed, default) or y = S x (sym=True): the dG discretisation of -div(chi grad .).  PAPER.md:73, 240."""
    _use_torch_stream()
    fn = lib().fx_dg_elliptic_apply_sym if sym else lib().fx_dg_elliptic_apply
    _check(fn(C.byref(grid), _ptr(chi, grid.n), _ptr(x, grid.n), _ptr(y, grid.n)), "fx_dg_elliptic_apply")
    return y


def make_grid3(Nx, Ny, Nz, P, lx, ly, lz, bcx, bcy):
    return Grid3(int(Nx), int(Ny), int(Nz), int(P), float(lx), float(ly), float(lz), int(bcx), int(bcy))


def dg3_elliptic_apply(grid, chi, x, y, sym=False):
    """3-D product grid (fx.h): y = A3 x, or S3 x = hz * S2 x plane by plane with sym=True"""
    _use_torch_stream()
    _check(lib().fx_dg3_elliptic_apply(C.byref(grid), _ptr(chi, grid.n), _ptr(x, grid.n), _ptr(y, grid.n), 1 if sym else 0), "fx_dg3_elliptic_apply")


def dg3_weights(grid, w=None, v=None):
    _use_torch_stream()
    _check(lib().fx_dg3_weights(C.byref(grid), _ptr(w, grid.n) if w is not None else None, _ptr(v, grid.n) if v is not None else None), "fx_dg3_weights")


def cg3_solve(grid, chi, rho, phi, tol, maxit):
    _use_torch_stream()
    info = CGInfo()
    rc = lib().fx_cg3_solve(C.byref(grid), _ptr(chi, grid.n), _ptr(rho, grid.n), _ptr(phi, grid.n), float(tol), int(maxit), C.byref(info))
    _check(rc, "fx_cg3_solve")
    return info


def dg_weights(grid, w=None, v=None):
    _use_torch_stream()
    _check(lib().fx_dg_weights(C.byref(grid), _ptr(w, grid.n) if w is not None else None,
                               _ptr(v, grid.n) if v is not None else None), "fx_dg_weights")
    return w, v


FORWARD, BACKWARD, CENTERED = 0, 1, 2


def dg_derivative(grid, direction, flux, alpha, x, beta, y):
    """y <- alpha * M x + beta * y, M = d/dx (direction 0) or d/dy (1), flux FORWARD/BACKWARD/CENTERED.  PAPER.md:240, 321."""
    _use_torch_stream()
    _check(lib().fx_dg_derivative(C.byref(grid), int(direction), int(flux), float(alpha), _ptr(x, grid.n), float(beta), _ptr(y, grid.n)),
           "fx_dg_derivative")
    return y


def dg_dtables(P, flux):
    """The derivative kernels' tables (host only): dict(TT: [2,P,P], cN: [P], cP: [P])."""
    import numpy as np
    out = np.zeros(2 * P * P + 2 * P)
    _check(lib().fx_dg_dtables(P, flux, out.ctypes.data_as(_dp)), "fx_dg_dtables")
    return dict(TT=out[:2 * P * P].reshape(2, P, P).copy(), cN=out[2 * P * P:2 * P * P + P].copy(), cP=out[2 * P * P + P:].copy())


def dg_tables(P):
    """The kernels' reference-element tables (host only, no GPU): dict(xi,w,L,R,B: [P]; T0,T0L,WW,D: [P,P])."""
    import numpy as np
    out = np.zeros(5 * P + 4 * P * P)
    _check(lib().fx_dg_tables(P, out.ctypes.data_as(_dp)), "fx_dg_tables")
    d, o = {}, 0
    for name in ("xi", "w", "L", "R", "B"):
        d[name] = out[o:o + P].copy(); o += P
    for name in ("T0", "T0L", "WW", "D"):
        d[name] = out[o:o + P * P].reshape(P, P).copy(); o += P * P
    return d


def cg_solve(grid, chi, rho, phi, tol, maxit):
    """Solve div(chi grad phi) = rho in place in phi (in: phi0).  Returns CGInfo.  PAPER.md:29, 75, 212."""
    _use_torch_stream()
    info = CGInfo()
    _check(lib().fx_cg_solve(C.byref(grid), _ptr(chi, grid.n), _ptr(rho, grid.n), _ptr(phi, grid.n), float(tol), int(maxit),
                             C.byref(info)), "fx_cg_solve")
    return info


TIME_KINDS = {"exdot": 0, "axpby": 1, "pointwise_dot": 2, "dg_apply_sym": 3, "dg_apply": 4, "exdot_host": 5, "axpy": 6, "exdot3": 7, "exsum": 8, "dx_forward": 9, "dy_forward": 10, "dx_centered": 11, "dy_centered": 12, "arakawa": 13, "fp64_fma": 14}
FP64_ROOF_FMAS_PER_SM = 8 * 256 * 8 * 4096          # fused multiply-adds one "fp64_fma" launch executes per SM (fx.h, kind 14)


def time_primitive(kind, a, b, c, reps, grid=None):
    """Average milliseconds per call of `reps` back-to-back calls of one primitive, timed on the device (fx.h)."""
    _use_torch_stream()
    ms = C.c_double(0.0)
    n = a.numel()
    _check(lib().fx_time_primitive(TIME_KINDS[kind], C.byref(grid) if grid is not None else None, _ptr(a), _ptr(b, n), _ptr(c, n), n,
                                   int(reps), C.byref(ms)), "fx_time_primitive")
    return ms.value


def cg_profile(enable):
    """enable: False/0 = off, True/1 = events around the kernels of every iteration, n > 1 = of every n-th iteration"""
    _check(lib().fx_cg_profile(int(enable)), "fx_cg_profile")


def cg_last_profile():
    """-> dict(loop_ms, k1_ms, k2_ms, k3_ms, iterations) of the most recent profiled fused solve (device times)."""
    ms = (C.c_double * 4)()
    it = C.c_int32(0)
    _check(lib().fx_cg_last_profile(ms, C.byref(it)), "fx_cg_last_profile")
    return dict(loop_ms=ms[0], k1_ms=ms[1], k2_ms=ms[2], k3_ms=ms[3], iterations=it.value)


def cg_solve_host(grid, chi, rho, phi, tol, maxit):
    """Same with HOST buffers (CPU tensors / numpy); phi is updated in place."""
    n, pc, pr, pp = _host_ptrs(chi, rho, phi)
    assert n == grid.n
    info = CGInfo()
    _check(lib().fx_cg_solve_host(C.byref(grid), pc, pr, pp, float(tol), int(maxit), C.byref(info)), "fx_cg_solve_host")
    return info
