"""sldg_rho_noalloc -- the rho pass for callers that may not allocate device memory -- against the
existing path, sldg_compute_rho.

Why the entry point exists: everything else in the library hangs off sldg_create, which cudaMallocs its
tables.  A host code that has handed the whole device heap to its own pool, a callback inside somebody
else's time loop (an allocation can synchronise the device under them) or a job with a fixed, audited
memory budget cannot use that.  sldg_rho_noalloc takes plain device pointers, keeps its partial sums in
a fixed 4 MiB array inside libsldg.so and allocates nothing, at the price of a size limit
(X <= SLDG_RHO_NOALLOC_MAX_X = 524288 x-nodes) and of all calls on a device sharing that one array.

What is checked: the new call gives sldg_compute_rho's rho within 1e-13 of max|rho| (the bound the rho
tests of test_gpu_physics.py use; the two paths add the same fp64 terms in a different order), on two
calls in a row and then on a differently shaped problem -- the array still holds the earlier call's
partial sums by then, and none of them may leak into the result.  The file sorts last on purpose: the
suite runs with pytest -x, and a failure here must not hide the tests of the main path.  It does not depend
on them either: each test builds its own inputs, so it passes alone in a fresh process as well.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1907_08316_b200 import sldg as S
from paper_1907_08316_b200 import workloads as W

from tests.gpu_util import NPDT, make_solver, rel_err

RHO_TOL = 1e-13          # as test_rho_poisson_diagnostics: |rho - rho_ref| <= RHO_TOL * max|rho_ref|
MAX_X = 524288           # SLDG_RHO_NOALLOC_MAX_X in include/sldg.h


def _v_weights(cfg):
    """W_v = prod_a h_a w_j over the v-dimensions (v_1 fastest), w the Gauss-Legendre weights on [0, 1]."""
    w = np.polynomial.legendre.leggauss(cfg.order)[1] / 2.0
    Wv = np.ones(1)
    for a in range(cfg.dx, cfg.dx + cfg.dv):
        h = (cfg.hi[a] - cfg.lo[a]) / cfg.cells[a]
        Wv = np.multiply.outer(np.tile(w * h, cfg.cells[a]), Wv).reshape(-1)    # later dimensions are slower
    return Wv


def _problem(dx, dv, cells, order, dtype, seed):
    lo = (0.0,) * dx + (-4.0,) * dv
    hi = tuple(2 * np.pi * (1 + 0.5 * a) for a in range(dx)) + (4.0,) * dv
    cfg = W.Config("noalloc", dx, dv, cells, order, lo, hi)
    f0 = np.random.default_rng(seed).uniform(0.0, 1.0, cfg.ndof).astype(NPDT[dtype])
    return cfg, f0


def _both_paths(cfg, f0, dtype, repeats):
    """rho of f0 through sldg_compute_rho (existing path) and `repeats` times through sldg_rho_noalloc."""
    import torch
    s = make_solver(cfg, dtype)
    s.set_initial(f0)
    ref = s.compute_rho().cpu().numpy()
    f = s.current()
    Wv = torch.from_numpy(_v_weights(cfg)).cuda()
    V = cfg.ndof // s.X
    outs = []
    for _ in range(repeats):
        rho = torch.full((s.X,), float("nan"), dtype=torch.float64, device="cuda")
        S.rho_noalloc(f, s.X, V, Wv, rho)
        outs.append(rho.cpu().numpy())
    s.close()
    return ref, outs


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rho_noalloc_matches_compute_rho_on_two_calls_in_a_row(dtype):
    # ragged 2+2 D grid: several blocks along x, several v-splits, a short last split
    cfg, f0 = _problem(2, 2, (23, 19, 17, 13), 3, dtype, seed=11)
    ref, (first, second) = _both_paths(cfg, f0, dtype, repeats=2)
    assert np.all(np.isfinite(first)) and np.all(np.isfinite(second))
    assert rel_err(first, ref) <= RHO_TOL
    assert rel_err(second, ref) <= RHO_TOL
    assert np.array_equal(first, second)          # same inputs, same launch geometry, fixed summation order
    # a different shape next: fewer x-nodes, so more v-splits land on scratch the calls above filled
    for shape in ((1, 1, (9, 7), 3), (3, 3, (4, 3, 5, 3, 4, 3), 2), (1, 2, (5, 6, 7), 3)):
        cfg2, f2 = _problem(shape[0], shape[1], shape[2], shape[3], dtype, seed=12)
        ref2, (again,) = _both_paths(cfg2, f2, dtype, repeats=1)
        assert rel_err(again, ref2) <= RHO_TOL, shape


@pytest.mark.gpu
def test_rho_noalloc_odd_pitch_and_unaligned_views():
    """X odd (scalar loads) and an f that starts 8 bytes into an allocation (no 16-byte vector loads)."""
    import torch
    X, V = 45, 301
    rng = np.random.default_rng(3)
    f = torch.from_numpy(rng.uniform(0.0, 1.0, X * V + 1)).cuda()
    Wv = torch.from_numpy(rng.uniform(0.5, 1.5, V)).cuda()
    want = -(Wv.cpu().numpy()[:, None] * f.cpu().numpy()[1:].reshape(V, X)).sum(axis=0)
    for _ in range(2):
        rho = torch.empty(X, dtype=torch.float64, device="cuda")
        S.rho_noalloc(f[1:], X, V, Wv, rho)
        assert rel_err(rho.cpu().numpy(), want) <= 1e-13
    X2 = 64
    f2 = torch.from_numpy(rng.uniform(0.0, 1.0, X2 * V + 1)).cuda()
    want2 = -(Wv.cpu().numpy()[:, None] * f2.cpu().numpy()[1:].reshape(V, X2)).sum(axis=0)
    rho2 = torch.empty(X2, dtype=torch.float64, device="cuda")
    S.rho_noalloc(f2[1:], X2, V, Wv, rho2)
    assert rel_err(rho2.cpu().numpy(), want2) <= 1e-13


def test_rho_noalloc_rejects_sizes_beyond_its_scratch():
    """No GPU needed: the size and argument checks come before any CUDA call, and nothing is dereferenced."""
    lib = C.CDLL(S.LIB_PATH)
    lib.sldg_rho_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_size_t, C.c_size_t, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_char_p, C.c_size_t]
    err = C.create_string_buffer(512)
    fake = 4096                                    # non-null, aligned, never touched
    rc = lib.sldg_rho_noalloc(fake, S.SLDG_F64, MAX_X + 1, 8, fake, fake, None, err, len(err))
    assert rc == -1 and b"SLDG_RHO_NOALLOC_MAX_X" in err.value and str(MAX_X + 1).encode() in err.value
    assert lib.sldg_rho_noalloc(None, S.SLDG_F64, 16, 8, fake, fake, None, err, len(err)) == -1
    assert lib.sldg_rho_noalloc(fake, S.SLDG_F64, 0, 8, fake, fake, None, err, len(err)) == -1
    assert lib.sldg_rho_noalloc(fake, 7, 16, 8, fake, fake, None, None, 0) == -2
    text = open(S.LIB_PATH.replace("paper_1907_08316_b200/libsldg.so", "include/sldg.h")).read()
    assert "#define SLDG_RHO_NOALLOC_MAX_X %d" % MAX_X in text
