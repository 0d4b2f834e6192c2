"""Device times of the film configs (BASELINE.json configs 1, 3, 5), which `bench.py` does not time.

    python -m paper_2411_11725_b200.config_timing [--steps 200]

One JSON line per config: CUDA-event times (ms, after warm-up, on the launching stream) of one
`nm_llg_rhs`, one RK4 step, one Dormand-Prince step (config 3's integrator), one adjoint RK4 step
(config 5's backward pass), the launches of one right-hand side, and whether steps were replayed
as CUDA graphs (`NM_GRAPH`).  Inputs are the seeded synthetic workloads of
`workloads.py`; nothing here is a parity check (tests/) or the bench contract (bench.py).
"""
import argparse
import json
import os

import numpy as np
import torch

from . import binding as nm
from . import workloads as wl


def _dev(a, td):
    return torch.from_numpy(wl.to_abi(a)).to(device="cuda:0", dtype=td).contiguous()


def _mesh(w, td):
    mat = {k: (float(getattr(w, k)) if np.isscalar(getattr(w, k)) else _dev(getattr(w, k), td))
           for k in ("Ms", "A", "Ku")}
    return nm.Mesh(w.n_cells, w.dx, dtype=td, terms=w.terms, gamma=w.gamma, alpha=w.alpha,
                   ku_axis=w.ku_axis, **mat)


def _zeeman(w, td):
    if not (w.terms & wl.TERM_ZEEMAN):
        return None
    hp = _dev(w.h_pulse, td) if w.h_pulse is not None else None
    amp = (lambda t: wl.sinc_pulse(t, **w.pulse)) if (w.pulse and hp is not None) else None
    return nm.Zeeman(h_uniform=w.h_uniform, h_pulse=hp, amp=amp)


def _time(fn, n):
    for _ in range(10):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=200)
    args = ap.parse_args()
    cases = (("config1_tiny_film", wl.config1_tiny_film(), torch.float64),
             ("config3_thin_film", wl.config3_thin_film(512), torch.float32),
             ("config5_inverse", wl.config5_inverse(), torch.float64))
    for name, w, td in cases:
        mesh = _mesh(w, td)
        z = _zeeman(w, td)
        nd = np.float64 if td == torch.float64 else np.float32
        m = _dev(wl.round_to(w.m0, nd), td)
        dt = w.dt if w.dt > 0 else 1e-13
        l0 = mesh.nm_launch_count()
        mesh.nm_llg_rhs(0.0, m, z)
        per_rhs = mesh.nm_launch_count() - l0
        y, a = m.clone(), m.clone()
        u = torch.zeros(mesh.cell_shape_abi, dtype=td, device="cuda:0")
        out = {
            "config": name, "n_cells": list(w.n_cells), "dtype": "f64" if td == torch.float64 else "f32",
            "launches_per_rhs": per_rhs,
            "graph_replay": os.environ.get("NM_GRAPH", "auto"),
            "host_amplitude_callback": bool(z is not None and z._keep[2] is not None),
            "llg_rhs_ms": _time(lambda: mesh.nm_llg_rhs(0.0, m, z), args.steps),
            "rk4_step_ms": _time(lambda: mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, y, z), args.steps),
            "dopri5_step_ms": _time(lambda: mesh.nm_rk_step(nm.NM_DOPRI5, 0.0, dt, y, z), args.steps),
            "adjoint_rk4_step_ms": _time(lambda: mesh.nm_adjoint_rk4_step(0.0, dt, y, a, u, z), args.steps),
        }
        out["mcells_per_s_rhs"] = float(np.prod(w.n_cells)) / out["llg_rhs_ms"] / 1e3
        print(json.dumps(out), flush=True)
        mesh.close()


if __name__ == "__main__":
    main()
