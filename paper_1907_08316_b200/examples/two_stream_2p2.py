"""The paper's validation run (section 8, eq. (2)): 2+2 D two-stream
instability in double AND single precision side by side on one B200, reporting what the paper
reports: the differences between the two in f (infinity norm), in E (infinity norm) and in the
electric energy (relative), which the paper states are "below 2e-4" for 60^4 cells, o = 4, t <= 100,
plus the invariants of its Fig. 15 (mass, total energy, L2 norm) for both precisions.

    python -m paper_1907_08316_b200.examples.two_stream_2p2 [--cells 60] [--t-end 100] [--dt 0.1]

Every step runs in the CUDA library (sldg_step, sldg_diagnostics, sldg_moments); torch is used only
to subtract the two device buffers for the infinity norms.  The paper does not print its time step;
dt is this build's choice (default 0.1).
"""
import argparse
import json

import numpy as np

from .. import workloads as W
from ..sldg import Sldg


def run(cells=60, t_end=100.0, dt=0.1, sample_every=10, order=4, verbose=False):
    import torch
    cfg = W.PAPER_TWOSTREAM.scaled((cells,) * 4)
    cfg = W.Config(cfg.name, cfg.dx, cfg.dv, cfg.cells, order, cfg.lo, cfg.hi, dt, int(round(t_end / dt)),
                   cfg.kind, cfg.eps, cfg.k, dict(cfg.extra))
    s64 = Sldg.from_config(cfg, dtype="f64")
    s32 = Sldg.from_config(cfg, dtype="f32")
    coords = [s64.node_coords(d) for d in range(4)]
    gx, gv = W.initial_factors(cfg, coords)
    f0 = torch.outer(torch.from_numpy(gv).cuda(), torch.from_numpy(gx).cuda()).reshape(-1).contiguous()
    s64.set_initial(f0)
    s32.set_initial(f0.to(torch.float32))
    del f0

    def sample(step):
        m64, l64, e64 = s64.diagnostics()
        m32, l32, e32 = s32.diagnostics()
        E64, E32 = s64.poisson_E(), s32.poisson_E()          # E of the rho the diagnostics just computed
        P64, K64 = s64.moments()
        P32, K32 = s32.moments()
        a, b = s64.current(), s32.current()
        df, fmax = 0.0, 0.0
        chunk = 1 << 28                                      # bounded temporaries
        for i in range(0, a.numel(), chunk):
            x = a[i:i + chunk]
            df = max(df, float((x - b[i:i + chunk].double()).abs().max()))
            fmax = max(fmax, float(x.abs().max()))
        return {"t": step * dt, "ee64": e64, "ee32": e32, "mass64": m64, "mass32": m32, "l2_64": l64,
                "l2_32": l32, "energy64": K64 + e64, "energy32": K32 + e32,
                "df_inf": df, "f_max": fmax, "dE_inf": float((E64 - E32).abs().max()),
                "E_max": float(E64.abs().max())}

    trace = [sample(0)]
    for n in range(1, cfg.steps + 1):
        s64.step(dt)
        s32.step(dt)
        if n % sample_every == 0 or n == cfg.steps:
            trace.append(sample(n))
            if verbose:
                print(json.dumps(trace[-1]), flush=True)
    s64.close()
    s32.close()
    ee64 = np.array([r["ee64"] for r in trace])
    ee32 = np.array([r["ee32"] for r in trace])
    out = {
        "config": {"cells": cells, "order": order, "dt": dt, "t_end": t_end, "ndof": cfg.ndof},
        "max_df_inf": max(r["df_inf"] for r in trace),
        "max_df_inf_rel_to_fmax": max(r["df_inf"] for r in trace) / max(r["f_max"] for r in trace),
        "max_dE_inf": max(r["dE_inf"] for r in trace),
        "max_E_inf": max(r["E_max"] for r in trace),
        "max_rel_ee_diff_vs_trace_max": float(np.max(np.abs(ee64 - ee32)) / np.max(ee64)),
        "max_rel_ee_diff_pointwise": float(np.max(np.abs(ee64 - ee32) / ee64)),
        "ee_growth": float(np.max(ee64) / ee64[0]),
        "mass_drift64": float(max(abs(r["mass64"] - trace[0]["mass64"]) for r in trace) / trace[0]["mass64"]),
        "mass_drift32": float(max(abs(r["mass32"] - trace[0]["mass32"]) for r in trace) / trace[0]["mass32"]),
        "energy_drift64": float(max(abs(r["energy64"] - trace[0]["energy64"]) for r in trace) / trace[0]["energy64"]),
        "energy_drift32": float(max(abs(r["energy32"] - trace[0]["energy32"]) for r in trace) / trace[0]["energy32"]),
        "l2_drop64": float(1.0 - trace[-1]["l2_64"] / trace[0]["l2_64"]),
        "l2_drop32": float(1.0 - trace[-1]["l2_32"] / trace[0]["l2_32"]),
        "paper_claim": "differences in f (inf-norm), E (inf-norm) and relative electric energy below 2e-4 "
                       "(60^4 cells, o=4, t<=100; PAPER.md line 235)",
    }
    return out, trace


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", type=int, default=60)
    ap.add_argument("--t-end", type=float, default=100.0)
    ap.add_argument("--dt", type=float, default=0.1)
    ap.add_argument("--order", type=int, default=4)
    ap.add_argument("--sample-every", type=int, default=10)
    ap.add_argument("--verbose", action="store_true")
    a = ap.parse_args()
    out, _ = run(a.cells, a.t_end, a.dt, a.sample_every, a.order, a.verbose)
    print(json.dumps(out))


if __name__ == "__main__":
    main()
