"""Python binding of the C-ABI library (include/sldg.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of libsldg.so.  PyTorch provides device
memory and the stream.  Importing this module loads libsldg.so and raises if it has not
been built; there is no CPU fallback.
"""
import ctypes as C
import os

import numpy as np

SLDG_F64, SLDG_F32 = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsldg.so")

EXPORTS = [
    "sldg_create", "sldg_destroy", "sldg_last_error", "sldg_num_dofs", "sldg_num_x",
    "sldg_node_coords", "sldg_set_initial", "sldg_get_f", "sldg_current", "sldg_fill_uniform",
    "sldg_translate", "sldg_translate_dev", "sldg_advect", "sldg_advect_pair", "sldg_translate_pair_dev", "sldg_advect_triple", "sldg_translate_triple_dev", "sldg_compute_rho", "sldg_poisson_E",
    "sldg_set_E", "sldg_advect_x_rho", "sldg_advect_x_twice", "sldg_step", "sldg_step_n", "sldg_diagnostics", "sldg_moments", "sldg_invariants", "sldg_launch_count",
    "sldg_rho_noalloc", "sldg_wide_shift_seen",
]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libsldg.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
            "(or python -m paper_1907_08316_b200.build).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.sldg_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, ip, C.c_int, dp, dp, C.c_int, vp, vp, vp]
    lib.sldg_destroy.argtypes = [vp]
    lib.sldg_last_error.argtypes = [vp]
    lib.sldg_last_error.restype = C.c_char_p
    lib.sldg_num_dofs.argtypes = [vp]
    lib.sldg_num_dofs.restype = C.c_size_t
    lib.sldg_num_x.argtypes = [vp]
    lib.sldg_num_x.restype = C.c_size_t
    lib.sldg_node_coords.argtypes = [vp, C.c_int, dp]
    lib.sldg_set_initial.argtypes = [vp, vp, C.c_int]
    lib.sldg_get_f.argtypes = [vp, vp, C.c_int]
    lib.sldg_current.argtypes = [vp]
    lib.sldg_current.restype = vp
    lib.sldg_fill_uniform.argtypes = [vp, C.c_ulonglong, C.c_uint]
    lib.sldg_translate.argtypes = [vp, C.c_int, dp, C.c_size_t]
    lib.sldg_translate_dev.argtypes = [vp, C.c_int, vp, C.c_size_t]
    lib.sldg_advect.argtypes = [vp, C.c_int, C.c_double]
    lib.sldg_advect_pair.argtypes = [vp, C.c_int, C.c_int, C.c_double]
    lib.sldg_translate_pair_dev.argtypes = [vp, C.c_int, vp, C.c_size_t, C.c_int, vp, C.c_size_t]
    lib.sldg_advect_triple.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double]
    lib.sldg_translate_triple_dev.argtypes = [vp] + [C.c_int, vp, C.c_size_t] * 3
    lib.sldg_compute_rho.argtypes = [vp, vp]
    lib.sldg_poisson_E.argtypes = [vp, vp]
    lib.sldg_set_E.argtypes = [vp, vp, C.c_int]
    lib.sldg_step.argtypes = [vp, C.c_double]
    lib.sldg_advect_x_rho.argtypes = [vp, C.c_double, vp]
    lib.sldg_advect_x_twice.argtypes = [vp, C.c_double]
    lib.sldg_step_n.argtypes = [vp, C.c_double, C.c_int]
    lib.sldg_diagnostics.argtypes = [vp, dp, dp, dp]
    lib.sldg_moments.argtypes = [vp, dp, dp]
    lib.sldg_invariants.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.sldg_launch_count.argtypes = [vp]
    lib.sldg_launch_count.restype = C.c_ulonglong
    lib.sldg_wide_shift_seen.argtypes = [vp, ip, C.c_int]
    lib.sldg_rho_noalloc.argtypes = [vp, C.c_int, C.c_size_t, C.c_size_t, vp, vp, vp, C.c_char_p, C.c_size_t]
    return lib


_lib = _load()


class SldgError(RuntimeError):
    pass


def rho_noalloc(f, X, V, Wv, rho, stream=None):
    """sldg_rho_noalloc: rho[x] = -sum_v Wv[v] f[v*X + x] with no device allocation inside the library.

    For callers that may not call cudaMalloc (a host code whose pool owns the whole device heap, a callback in
    another program's time loop, a fixed memory budget): there is no context, the caller brings every buffer --
    f (X*V values, float64 or float32), Wv (V float64) and rho (X float64, written), all CUDA tensors on the
    current device -- and the partial sums sit in a fixed 4 MiB array inside libsldg.so.  X may not exceed
    SLDG_RHO_NOALLOC_MAX_X (524288).  Calls on one device share that array: keep them on one stream.  The first
    call on a device also looks the array up; make it outside any stream capture.  Marshalling only."""
    import torch
    assert f.is_cuda and Wv.is_cuda and rho.is_cuda and f.is_contiguous() and Wv.is_contiguous() and rho.is_contiguous()
    assert Wv.dtype == torch.float64 and rho.dtype == torch.float64 and f.dtype in (torch.float64, torch.float32)
    assert f.numel() == X * V and Wv.numel() == V and rho.numel() == X
    if stream is None:
        stream = torch.cuda.current_stream(f.device)
    err = C.create_string_buffer(512)
    with torch.cuda.device(f.device):
        rc = _lib.sldg_rho_noalloc(f.data_ptr(), SLDG_F64 if f.dtype == torch.float64 else SLDG_F32, int(X), int(V),
                                   Wv.data_ptr(), rho.data_ptr(), stream.cuda_stream, err, len(err))
    if rc != 0:
        raise SldgError("sldg_rho_noalloc failed (%d): %s" % (rc, err.value.decode()))
    return rho


class Sldg:
    """One solver context.  Allocates the two f buffers as torch CUDA tensors (caller-owned
    memory in the sense of sldg.h) and forwards every call to the library."""

    def __init__(self, dx, dv, cells, order, lo, hi, dtype="f64", device="cuda:0", stream=None, buffers=None):
        import torch
        if not torch.cuda.is_available():
            raise SldgError("no CUDA device: the SLDG library has no CPU path")
        self.torch = torch
        self.dx, self.dv, self.order = int(dx), int(dv), int(order)
        D = self.dx + self.dv
        self.cells = tuple(int(c) for c in cells)
        self.N = tuple(c * self.order for c in self.cells)
        self.X = int(np.prod(self.N[: self.dx]))
        self.ndof = int(np.prod(self.N))
        self.dtype = {"f64": SLDG_F64, "f32": SLDG_F32}[dtype]
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.npdtype = np.float64 if dtype == "f64" else np.float32
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        if buffers is None:
            self.buf = [torch.empty(self.ndof, dtype=self.tdtype, device=self.device) for _ in range(2)]
        else:       # caller-owned device buffers (two contiguous CUDA tensors of N values each)
            self.buf = list(buffers)
            for b in self.buf:
                assert b.is_cuda and b.dtype == self.tdtype and b.numel() == self.ndof and b.is_contiguous()
        cells_a = (C.c_int * D)(*self.cells)
        lo_a = (C.c_double * D)(*[float(x) for x in lo])
        hi_a = (C.c_double * D)(*[float(x) for x in hi])
        h = C.c_void_p()
        rc = _lib.sldg_create(C.byref(h), self.dx, self.dv, cells_a, self.order, lo_a, hi_a, self.dtype,
                              self.buf[0].data_ptr(), self.buf[1].data_ptr(), self.stream.cuda_stream)
        if rc != 0:
            raise SldgError("sldg_create failed (%d): %s" % (rc, _lib.sldg_last_error(None).decode()))
        self.h = h

    @classmethod
    def from_config(cls, cfg, dtype="f64", **kw):
        return cls(cfg.dx, cfg.dv, cfg.cells, cfg.order, cfg.lo, cfg.hi, dtype=dtype, **kw)

    def _chk(self, rc, what):
        if rc != 0:
            raise SldgError("%s failed (%d): %s" % (what, rc, _lib.sldg_last_error(self.h).decode()))

    def close(self):
        if getattr(self, "h", None):
            _lib.sldg_destroy(self.h)
            self.h = None
            self.buf = None          # release the two f buffers

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- data in / out
    def node_coords(self, dim):
        out = np.zeros(self.N[dim], dtype=np.float64)
        self._chk(_lib.sldg_node_coords(self.h, dim, out.ctypes.data_as(C.POINTER(C.c_double))), "node_coords")
        return out

    def set_initial(self, f):
        """f: numpy array (host) or torch CUDA tensor, N values of the context's dtype."""
        if isinstance(f, np.ndarray):
            f = np.ascontiguousarray(f, dtype=self.npdtype).reshape(-1)
            assert f.size == self.ndof
            self._chk(_lib.sldg_set_initial(self.h, f.ctypes.data, 0), "set_initial")
        elif f.is_cuda:
            assert f.dtype == self.tdtype and f.numel() == self.ndof and f.is_contiguous()
            self._chk(_lib.sldg_set_initial(self.h, f.data_ptr(), 1), "set_initial")
        else:   # host torch tensor (e.g. pinned)
            assert f.dtype == self.tdtype and f.numel() == self.ndof and f.is_contiguous()
            self._chk(_lib.sldg_set_initial(self.h, f.data_ptr(), 0), "set_initial")

    def get_f(self, out=None):
        """Copy f to host: into `out` (numpy or host torch tensor) or a new numpy array."""
        if out is None:
            out = np.empty(self.ndof, dtype=self.npdtype)
        ptr = out.ctypes.data if isinstance(out, np.ndarray) else out.data_ptr()
        self._chk(_lib.sldg_get_f(self.h, ptr, 0), "get_f")
        return out

    def current(self):
        """The torch tensor (view of the caller-owned buffer) that holds f now."""
        p = _lib.sldg_current(self.h)
        return self.buf[0] if p == self.buf[0].data_ptr() else self.buf[1]

    def fill_uniform(self, seed, tag=0):
        self._chk(_lib.sldg_fill_uniform(self.h, int(seed), int(tag)), "fill_uniform")

    # ---- the path
    def translate(self, dim, shift_cells):
        if isinstance(shift_cells, np.ndarray):
            s = np.ascontiguousarray(shift_cells, dtype=np.float64).reshape(-1)
            self._chk(_lib.sldg_translate(self.h, dim, s.ctypes.data_as(C.POINTER(C.c_double)), s.size), "translate")
        else:
            assert shift_cells.is_cuda and shift_cells.dtype == self.torch.float64 and shift_cells.is_contiguous()
            self._chk(_lib.sldg_translate_dev(self.h, dim, shift_cells.data_ptr(), shift_cells.numel()), "translate_dev")

    def advect(self, dim, dt):
        self._chk(_lib.sldg_advect(self.h, dim, float(dt)), "advect")

    def advect_pair(self, dim1, dim2, dt):
        self._chk(_lib.sldg_advect_pair(self.h, dim1, dim2, float(dt)), "advect_pair")

    def translate_pair(self, dim1, shift1, dim2, shift2):
        """Fused pair of raw sweeps; shift tables are fp64 CUDA tensors."""
        for t in (shift1, shift2):
            assert t.is_cuda and t.dtype == self.torch.float64 and t.is_contiguous()
        self._chk(_lib.sldg_translate_pair_dev(self.h, dim1, shift1.data_ptr(), shift1.numel(),
                                               dim2, shift2.data_ptr(), shift2.numel()), "translate_pair_dev")

    def advect_triple(self, d1, d2, d3, dt):
        self._chk(_lib.sldg_advect_triple(self.h, d1, d2, d3, float(dt)), "advect_triple")

    def translate_triple(self, d1, s1, d2, s2, d3, s3):
        for t in (s1, s2, s3):
            assert t.is_cuda and t.dtype == self.torch.float64 and t.is_contiguous()
        self._chk(_lib.sldg_translate_triple_dev(self.h, d1, s1.data_ptr(), s1.numel(), d2, s2.data_ptr(),
                                                 s2.numel(), d3, s3.data_ptr(), s3.numel()), "translate_triple_dev")

    def compute_rho(self, out=True):
        """rho into the context; with out=True also returned as a new device tensor."""
        if not out:
            self._chk(_lib.sldg_compute_rho(self.h, None), "compute_rho")
            return None
        rho = self.torch.empty(self.X, dtype=self.torch.float64, device=self.device)
        self._chk(_lib.sldg_compute_rho(self.h, rho.data_ptr()), "compute_rho")
        return rho

    def poisson_E(self, out=True):
        if not out:
            self._chk(_lib.sldg_poisson_E(self.h, None), "poisson_E")
            return None
        E = self.torch.empty((self.dx, self.X), dtype=self.torch.float64, device=self.device)
        self._chk(_lib.sldg_poisson_E(self.h, E.data_ptr()), "poisson_E")
        return E

    def set_E(self, E):
        if isinstance(E, np.ndarray):
            E = np.ascontiguousarray(E, dtype=np.float64).reshape(-1)
            assert E.size == self.dx * self.X
            self._chk(_lib.sldg_set_E(self.h, E.ctypes.data, 0), "set_E")
        else:
            assert E.is_cuda and E.dtype == self.torch.float64 and E.numel() == self.dx * self.X
            self._chk(_lib.sldg_set_E(self.h, E.data_ptr(), 1), "set_E")

    def advect_x_rho(self, tau, out=True):
        """x half-step + rho of the result in one pass (rho returned as a new device tensor if out)."""
        if not out:
            self._chk(_lib.sldg_advect_x_rho(self.h, float(tau), None), "advect_x_rho")
            return None
        rho = self.torch.empty(self.X, dtype=self.torch.float64, device=self.device)
        self._chk(_lib.sldg_advect_x_rho(self.h, float(tau), rho.data_ptr()), "advect_x_rho")
        return rho

    def advect_x_twice(self, tau):
        self._chk(_lib.sldg_advect_x_twice(self.h, float(tau)), "advect_x_twice")

    def step_n(self, dt, nsteps):
        """nsteps Strang steps with the x half-steps of consecutive steps merged into one pass."""
        self._chk(_lib.sldg_step_n(self.h, float(dt), int(nsteps)), "step_n")

    def step(self, dt):
        self._chk(_lib.sldg_step(self.h, float(dt)), "step")

    def diagnostics(self):
        m, l2, ee = C.c_double(), C.c_double(), C.c_double()
        self._chk(_lib.sldg_diagnostics(self.h, C.byref(m), C.byref(l2), C.byref(ee)), "diagnostics")
        return m.value, l2.value, ee.value

    def moments(self):
        """(momentum[dv] as numpy array, kinetic energy)."""
        P = (C.c_double * self.dv)()
        k = C.c_double()
        self._chk(_lib.sldg_moments(self.h, P, C.byref(k)), "moments")
        return np.array(list(P)), k.value

    def invariants(self):
        """(mass, l2, electric energy, momentum[dv], kinetic energy) from one read of f."""
        m, l2, ee, k = C.c_double(), C.c_double(), C.c_double(), C.c_double()
        P = (C.c_double * self.dv)()
        self._chk(_lib.sldg_invariants(self.h, C.byref(m), C.byref(l2), C.byref(ee), P, C.byref(k)), "invariants")
        return m.value, l2.value, ee.value, np.array(list(P)), k.value

    def wide_shift_seen(self, reset=False):
        """True when a fused v-sweep met a line shifted by a cell or more since create / the last reset
        (it then ran its slow per-block fallback: shorten dt or issue single sweeps).  Synchronises the stream."""
        seen = C.c_int(0)
        self._chk(_lib.sldg_wide_shift_seen(self.h, C.byref(seen), 1 if reset else 0), "wide_shift_seen")
        return bool(seen.value)

    def launch_count(self):
        return int(_lib.sldg_launch_count(self.h))
