"""Helpers shared by the -m gpu parity tests (not a test module)."""
import numpy as np

TOL = {"f64": 1e-12, "f32": 2e-5}          # BASELINE.json north_star: max|f_gpu - f_cpu| <= tol * max|f|
NPDT = {"f64": np.float64, "f32": np.float32}


def dep_of(cfg_dx, dim):
    """Dimensions the shift of a sweep along `dim` depends on (D:R8)."""
    return [cfg_dx + dim] if dim < cfg_dx else list(range(cfg_dx))


def rel_err(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def make_solver(cfg, dtype):
    from paper_1907_08316_b200.sldg import Sldg
    return Sldg.from_config(cfg, dtype=dtype)
