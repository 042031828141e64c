"""ctypes access to the CPU oracle (oracle/sldg_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It does
argument marshalling only; every number comes out of the C code.
"""
import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

_pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_pf = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_pi = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_pl = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def _load():
    global _lib
    if _lib is not None:
        return _lib
    spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    lib = C.CDLL(mod.build())
    grid = [C.c_int, C.c_int, _pi, C.c_int, _pd, _pd]          # dx, dv, cells, o, lo, hi
    lib.oracle_gauss_legendre.argtypes = [C.c_int, _pd, _pd]
    lib.oracle_lagrange.argtypes = [C.c_int, _pd, C.c_int, C.c_double]
    lib.oracle_lagrange.restype = C.c_double
    lib.oracle_shift_split.argtypes = [C.c_double, C.POINTER(C.c_long), C.POINTER(C.c_double)]
    lib.oracle_shift_split.restype = None
    lib.oracle_assemble_AB.argtypes = [C.c_int, C.c_double, _pd, _pd]
    lib.oracle_node_coords.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _pd]
    lib.oracle_poisson_E.argtypes = [_pd, C.c_int, _pi, C.c_int, _pd, _pd, _pd]
    for suf, pt in (("f64", _pd), ("f32", _pf)):
        getattr(lib, "oracle_translate_line_" + suf).argtypes = [C.c_int, C.c_long, pt, pt, C.c_long, pt, pt]
        getattr(lib, "oracle_translate_" + suf).argtypes = [pt, C.c_int, _pl, C.c_int, C.c_int, _pd, C.c_int, _pi]
        getattr(lib, "oracle_advect_" + suf).argtypes = [pt] + grid + [C.c_int, C.c_double, C.c_void_p]
        getattr(lib, "oracle_rho_" + suf).argtypes = [pt] + grid + [_pd]
        getattr(lib, "oracle_step_" + suf).argtypes = [pt] + grid + [C.c_double]
        getattr(lib, "oracle_diagnostics_" + suf).argtypes = [pt] + grid + [C.POINTER(C.c_double)] * 3
        getattr(lib, "oracle_moments_" + suf).argtypes = [pt] + grid + [_pd, C.POINTER(C.c_double)]
    _lib = lib
    return lib


def _check(rc, what):
    if rc != 0:
        raise ValueError("oracle: %s failed (rc=%d)" % (what, rc))


def _suf(f):
    if f.dtype == np.float64:
        return "f64"
    if f.dtype == np.float32:
        return "f32"
    raise TypeError("f must be float64 or float32")


def num_threads():
    return int(_load().oracle_num_threads())


def gauss_legendre(o):
    xi, w = np.zeros(o), np.zeros(o)
    _check(_load().oracle_gauss_legendre(o, xi, w), "gauss_legendre")
    return xi, w


def lagrange(o, xi, j, x):
    return float(_load().oracle_lagrange(o, np.ascontiguousarray(xi, dtype=np.float64), j, float(x)))


def shift_split(sigma):
    m, th = C.c_long(), C.c_double()
    _load().oracle_shift_split(float(sigma), C.byref(m), C.byref(th))
    return int(m.value), float(th.value)


def assemble_AB(o, theta):
    A, B = np.zeros((o, o)), np.zeros((o, o))
    _check(_load().oracle_assemble_AB(o, float(theta), A, B), "assemble_AB")
    return A, B


def node_coords(n_cells, o, lo, hi):
    c = np.zeros(n_cells * o)
    _check(_load().oracle_node_coords(n_cells, o, float(lo), float(hi), c), "node_coords")
    return c


def translate_line(o, A, B, m, u_old):
    """One periodic 1-D line (O2/O7).  A, B, u_old share one dtype (already rounded)."""
    u_old = np.ascontiguousarray(u_old)
    suf = _suf(u_old)
    A = np.ascontiguousarray(A, dtype=u_old.dtype)
    B = np.ascontiguousarray(B, dtype=u_old.dtype)
    u_new = np.empty_like(u_old)
    fn = getattr(_load(), "oracle_translate_line_" + suf)
    _check(fn(o, u_old.size // o, A, B, int(m), u_old, u_new), "translate_line")
    return u_new


def translate(f, N, o, k, sigma, dep):
    """In-place sweep along dimension k of flat f (canonical layout, N[d] nodes per dim)."""
    assert f.flags["C_CONTIGUOUS"] and f.ndim == 1
    N = np.ascontiguousarray(N, dtype=np.int64)
    sigma = np.ascontiguousarray(sigma, dtype=np.float64)
    dep = np.ascontiguousarray(dep, dtype=np.int32)
    assert f.size == int(np.prod(N))
    assert sigma.size == int(np.prod(N[dep])) if dep.size else sigma.size == 1
    fn = getattr(_load(), "oracle_translate_" + _suf(f))
    _check(fn(f, len(N), N, o, k, sigma, len(dep), dep), "translate")
    return f


class Grid:
    """Arguments that describe the phase-space grid (S:section 8 Notation)."""

    def __init__(self, dx, dv, cells, o, lo, hi):
        self.dx, self.dv, self.o = int(dx), int(dv), int(o)
        self.cells = np.ascontiguousarray(cells, dtype=np.int32)
        self.lo = np.ascontiguousarray(lo, dtype=np.float64)
        self.hi = np.ascontiguousarray(hi, dtype=np.float64)
        assert self.cells.size == self.lo.size == self.hi.size == self.dx + self.dv
        self.N = self.cells.astype(np.int64) * self.o
        self.X = int(np.prod(self.N[: self.dx]))
        self.ndof = int(np.prod(self.N))

    def _args(self):
        return (self.dx, self.dv, self.cells, self.o, self.lo, self.hi)

    def coords(self, d):
        return node_coords(int(self.cells[d]), self.o, self.lo[d], self.hi[d])

    def advect(self, f, dim, tau, E=None):
        fn = getattr(_load(), "oracle_advect_" + _suf(f))
        Ep = None
        if E is not None:
            E = np.ascontiguousarray(E, dtype=np.float64)
            assert E.size == self.dx * self.X
            Ep = E.ctypes.data_as(C.c_void_p)
        _check(fn(f, *self._args(), dim, float(tau), Ep), "advect")
        return f

    def rho(self, f):
        rho = np.zeros(self.X)
        _check(getattr(_load(), "oracle_rho_" + _suf(f))(f, *self._args(), rho), "rho")
        return rho

    def poisson_E(self, rho):
        E = np.zeros(self.dx * self.X)
        rho = np.ascontiguousarray(rho, dtype=np.float64)
        _check(_load().oracle_poisson_E(rho, self.dx, self.cells, self.o, self.lo, self.hi, E), "poisson_E")
        return E.reshape(self.dx, self.X)

    def step(self, f, dt):
        _check(getattr(_load(), "oracle_step_" + _suf(f))(f, *self._args(), float(dt)), "step")
        return f

    def moments(self, f):
        """(momentum[dv], kinetic energy) -- NEXT-4 invariants."""
        P, k = np.zeros(self.dv), C.c_double()
        _check(getattr(_load(), "oracle_moments_" + _suf(f))(f, *self._args(), P, C.byref(k)), "moments")
        return P, k.value

    def diagnostics(self, f):
        m, l2, ee = C.c_double(), C.c_double(), C.c_double()
        fn = getattr(_load(), "oracle_diagnostics_" + _suf(f))
        _check(fn(f, *self._args(), C.byref(m), C.byref(l2), C.byref(ee)), "diagnostics")
        return m.value, l2.value, ee.value
