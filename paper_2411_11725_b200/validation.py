"""Physics validation runs through the C-ABI (Sec. VI).

The paper validates on MuMag standard problem #4 (3-D against 2-D discretisation, Fig. 5) and on the
two-phase domain-wall depinning problem of its ref. 21 (Table I).  Neither problem file is in this
container, so the runs here are stand-ins of the same kind, with their own stated parameters, and
checks that need no reference data:

  film_reversal     a thin-film element (BASELINE.json config 1's cell and materials, 160 x 40 x 1
                    cells = 500 x 125 x 3 nm) is relaxed at alpha = 1 and then switched by a field
                    applied 170 degrees from +x; run on the 3-D nodal basis and on the 2-D basis of
                    Sec. III C; the check of PAPER.md:311 is that both give the same <m>(t).
  depinning_field   a 1-D two-phase rod (1-D basis of Eq. 24) with the uniaxial anisotropy constant
                    jumping from 0 to K at the interface, equal A and Ms, no demag: the field at
                    which a wall pushed from the soft phase breaks into the hard phase, by a
                    quasi-static field ramp.  For this special case the sharp-interface theory gives
                    H_p = H_K / 4 = K / (2 mu0 Ms)  (the "K" row of the paper's Table I is this kind).

Host loop control only; every field evaluation and time step runs in libnm.so.
"""
import math

import numpy as np
import torch

from . import binding as nm
from .drivers import integrate_dopri5

MU0 = 4.0e-7 * math.pi


def _to_dev(a, dtype, device):
    """(3, n1, n2, n3) paper order -> ABI order device tensor."""
    return torch.from_numpy(np.ascontiguousarray(np.asarray(a).transpose(0, 3, 2, 1))).to(
        device="cuda:%d" % device, dtype=dtype).contiguous()


def film_reversal(basis=3, n_cells=(160, 40, 1), cell=(3.125e-9, 3.125e-9, 3e-9), Ms=8e5, A=1.3e-11,
                  alpha=0.02, h_mag=2.0e4, h_angle_deg=170.0, t_relax=1.0e-9, t_run=1.0e-9, dtype=torch.float64,
                  device=0, rtol=1e-5, atol=1e-5):
    """Relax (alpha = 1) from a tilted uniform state, then apply a uniform field of h_mag A/m at
    h_angle_deg from +x in the film plane and integrate for t_run with Dormand-Prince.

    Returns a dict: times, <m> per accepted step, energies sampled along the run, step counts and
    max | |m| - 1 |."""
    n = tuple(int(v) for v in n_cells)
    nodes = (n[0] + 1, n[1] + 1 if basis >= 2 else 1, n[2] + 1 if basis >= 3 else 1)
    m0 = np.zeros((3,) + nodes)
    m0[0], m0[1], m0[2] = 1.0, 0.3, 0.05
    m0 /= np.sqrt((m0 ** 2).sum(axis=0))
    m = _to_dev(m0, dtype, device)
    terms = nm.NM_TERM_EXCHANGE | nm.NM_TERM_DEMAG | nm.NM_TERM_ZEEMAN
    relax = nm.Mesh(n, cell, dtype=dtype, device=device, terms=terms, alpha=1.0, Ms=Ms, A=A, basis=basis)
    zero = nm.Zeeman(h_uniform=(0.0, 0.0, 0.0))
    _, _, acc0, rej0 = integrate_dopri5(relax, m, 0.0, t_relax, 1e-13, zero, rtol=rtol, atol=atol)
    m_relaxed = m.mean(dim=(1, 2, 3)).cpu().numpy()
    del relax
    run = nm.Mesh(n, cell, dtype=dtype, device=device, terms=terms, alpha=alpha, Ms=Ms, A=A, basis=basis)
    ang = math.radians(h_angle_deg)
    hu = (h_mag * math.cos(ang), h_mag * math.sin(ang), 0.0)
    z = nm.Zeeman(h_uniform=hu)
    # L-weighted energy E = -1/2 sum L m.(H - H_ext) - sum L m.H_ext on the device (nodal weights of the lumped mass)
    V = cell[0] * cell[1] * cell[2]
    w1 = [np.ones(k) if k == 1 else np.concatenate(([0.5], np.ones(k - 2), [0.5])) for k in nodes]
    ncell_per_node = 2 ** basis
    lw = (w1[0][:, None, None] * w1[1][None, :, None] * w1[2][None, None, :]) * ncell_per_node
    L = MU0 * (V / ncell_per_node) * Ms * lw
    Ld = torch.from_numpy(np.ascontiguousarray(L.transpose(2, 1, 0))).to(device=m.device, dtype=dtype)
    hext = torch.tensor(hu, dtype=dtype, device=m.device).view(3, 1, 1, 1)

    def energy():
        H = run.nm_heff(0.0, m, z)
        return float((-0.5 * (Ld * (m * (H - hext)).sum(dim=0)).sum() - (Ld * (m * hext).sum(dim=0)).sum()).item())

    ts, avg, en = [0.0], [m.mean(dim=(1, 2, 3)).cpu().numpy()], [(0.0, energy())]
    state = {"k": 0}

    def on_step(t, h, err):
        ts.append(t)
        avg.append(m.mean(dim=(1, 2, 3)).cpu().numpy())
        state["k"] += 1
        if state["k"] % 50 == 0:
            en.append((t, energy()))

    _, _, acc, rej = integrate_dopri5(run, m, 0.0, t_run, 1e-13, z, rtol=rtol, atol=atol, on_step=on_step)
    nrm = torch.sqrt((m * m).sum(dim=0))
    return {"basis": basis, "t": np.array(ts), "m_avg": np.array(avg), "energy": np.array(en),
            "m_relaxed": m_relaxed, "relax_steps": (acc0, rej0), "run_steps": (acc, rej),
            "norm_defect": float((nrm - 1).abs().max().item()), "launches": run.nm_launch_count()}


def depinning_field(n_cells=400, cell=0.5e-9, Ms=1.0e6, A=1.0e-11, K=1.0e6, alpha=1.0, h_start=0.90, h_stop=1.10,
                    h_step=0.0025, t_hold=1.0e-10, dt=4.0e-14, dtype=torch.float64, device=0):
    """Quasi-static depinning of a wall at a soft (Ku = 0) / hard (Ku = K) interface of a rod of
    n_cells cells on the 1-D basis; easy axis z, field along -z raised from h_start to h_stop times
    H_K / 4 in steps of h_step, held t_hold each (RK4 steps of dt, alpha = 1).

    Returns a dict with the analytic H_p = K / (2 mu0 Ms) and, in units of it, the last field at which
    the far half of the hard phase was untouched (`held`), the first at which the wall had entered it
    (`moved`: its mean m_z below 0.999) and the first at which it had reversed (`broke`: mean m_z < 0)."""
    N = int(n_cells)
    Ku = np.zeros((N, 1, 1))
    Ku[N // 2:] = K
    Kd = torch.from_numpy(np.ascontiguousarray(Ku.transpose(2, 1, 0))).to(device="cuda:%d" % device, dtype=dtype)
    terms = nm.NM_TERM_EXCHANGE | nm.NM_TERM_ANISO | nm.NM_TERM_ZEEMAN
    mesh = nm.Mesh((N, 1, 1), (cell, cell, cell), dtype=dtype, device=device, terms=terms, alpha=alpha, Ms=Ms, A=A,
                   Ku=Kd, ku_axis=(0.0, 0.0, 1.0), basis=1)
    # wall in the soft phase, two wall widths before the interface: m = (sech, 0, tanh) profile
    x = (np.arange(N + 1) - N // 2) * cell
    delta = math.sqrt(A / K)
    th = np.tanh((x + 6 * delta) / (2 * delta))
    m0 = np.zeros((3, N + 1, 1, 1))
    m0[2, :, 0, 0] = th
    m0[0, :, 0, 0] = np.sqrt(np.maximum(0.0, 1 - th ** 2))
    m = _to_dev(m0, dtype, device)
    h_p = K / (2.0 * MU0 * Ms)
    steps = int(round(t_hold / dt))
    held, moved, broke = None, None, None
    f = h_start
    history = []
    while f <= h_stop + 1e-12:
        z = nm.Zeeman(h_uniform=(0.0, 0.0, -f * h_p))
        for s in range(steps):
            mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, m, z)
        mz_hard = float(m[2, 0, 0, N // 2 + N // 4:].mean().item())
        history.append((f, mz_hard))
        if mz_hard < 0.999 and moved is None:
            moved = f
        if mz_hard < 0.0:
            broke = f
            break
        if moved is None:
            held = f
        f += h_step
    return {"h_p_analytic": h_p, "held": held, "moved": moved, "broke": broke, "history": history,
            "launches": mesh.nm_launch_count()}
