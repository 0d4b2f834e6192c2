#!/usr/bin/env python
"""bench.py -- throughput of the nodal-FD LLG hot path on B200 (contract: see the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--grid 256] [--dtype f32|f64]
    python bench.py --impl reference ...        # the CPU oracle, as it stands, on host cores

One *step* is one pass of the whole hot path over one grid:
  one RK4 step through nm_rk_step   = 4 fused right-hand sides (node->cell average, 5 FFT passes
                                      with the tensor multiply, cell->node average, exchange,
                                      LLG cross products, stage combination, renormalisation)
  one nm_llg_adjoint_rhs            = 2 more field evaluations (demag convolutions of m and of
                                      b/(S Ms), two node passes, the Ms-gradient cell pass)
so a step is 6 field evaluations; the metric is cells x field evaluations per second (Mcells/s),
BASELINE.json's "H_eff + LLG RHS evals/s (Mcells/s)".  Workload at N = 1: config 4's largest grid,
256^3 cells, fp32, exchange + demag, seeded random unit m (the grid north_star's target is quoted
on).  N > 1: replicas only: every rank runs the same grid on its own GPU with no
data-path collective; value = cells processed by all ranks / max-over-ranks time.

Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "llg_field_evaluations_mcells_per_s"
UNIT = "Mcells/s"
EVALS_PER_STEP = 6          # 4 (RK4) + 2 (adjoint right-hand side)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--grid", type=int, default=256, help="N of the N^3 config-4 grid")
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sample-grid", type=int, default=0, help="oracle sample grid (0 = auto)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the config-4 / film sweep block")
    ap.add_argument("--config3", type=float, default=0.0, metavar="NS",
                    help="instead of the bench: run config 3's stated recipe (512x512x1, fp32, Dormand-Prince) "
                         "for NS nanoseconds (10 = the full run) and print its wall time as one JSON line")
    ap.add_argument("--traffic-from", default="", metavar="NCU_REP",
                    help="instead of the bench: read dram bytes per launch of the hot kernels from an "
                         "`ncu --set full` report of this command and write profiles/traffic.json")
    return ap.parse_args()


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch of each kernel class come from
# profiles/traffic.json, written by `bench.py --traffic-from <ncu report>` from one `ncu --set full`
# capture of this command and stamped with the hash of the kernel sources it was captured on; a
# capture of other sources than the ones in the tree is reported as stale (traffic = null).
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")
KERNEL_CLASS = (("k_pz_mid", "mid"), ("k_fz_mid", "mid"), ("k_py_fwd", "y_fwd"), ("k_fy_fwd", "y_fwd"),
                ("k_py_inv", "y_inv"), ("k_fy_inv", "y_inv"), ("k_px_fwd", "x_fwd"), ("k_px_inv", "x_inv"),
                ("k_node", "node"))     # split further by the epilogue mode, see node_class()


def node_class(kernel_name):
    """'node' / 'node_rk' / 'node_adj' from the epilogue mode in a node kernel's template arguments
    (k_node_col<T, RY, CS, CM, ...>: CM 0-1 H / f, 2-4 Runge-Kutta stage, 5-6 adjoint passes)."""
    import re
    m = re.match(r"k_node_col<[^,]+,\s*\d+,\s*\d+,\s*(\d+)", kernel_name)
    if not m:
        return "node"
    cm = int(m.group(1))
    return "node" if cm <= 1 else "node_rk" if cm <= 4 else "node_adj"


def csrc_hash():
    import hashlib
    d = os.path.join(ROOT, "paper_2411_11725_b200", "csrc")
    h = hashlib.sha1()
    for f in sorted(os.listdir(d)):
        h.update(f.encode())
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def load_traffic(N, dtype):
    """(bytes per launch by kernel class or {}, source string)."""
    try:
        t = json.load(open(TRAFFIC_JSON))
    except Exception:
        return {}, "no profiles/traffic.json"
    if t.get("csrc_sha1") != csrc_hash():
        return {}, "profiles/traffic.json is stale (captured on other kernel sources, commit %s)" % t.get("commit")
    if (t.get("grid"), t.get("dtype")) != (N, dtype):
        return {}, "profiles/traffic.json is for %s^3 %s" % (t.get("grid"), t.get("dtype"))
    return t["bytes_per_launch"], "profiles/traffic.json (ncu --set full, per launch, commit %s)" % t.get("commit")


def write_traffic(rep, N, dtype):
    """Parse `ncu -i rep --page raw --csv` and write profiles/traffic.json."""
    import csv
    import io
    import re
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    idx = {h: i for i, h in enumerate(rows[0])}
    units = rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc = {}
    for r in rows[2:]:
        name = r[idx["Kernel Name"]]
        mk = re.search(r"\bk_[a-z0-9_]+.*", name)          # "void <unnamed>::k_pz_mid<0>(float2 *, ...)" -> "k_pz_mid<0>(..."
        base = mk.group(0) if mk else name
        cls = next((c for k, c in KERNEL_CLASS if base.startswith(k)), None)
        if cls is None:
            continue
        if cls == "node":
            cls = node_class(base)
        b = 0.0
        for col in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            b += float(r[idx[col]].replace(",", "")) * scale[units[idx[col]]]
        acc.setdefault(cls, []).append(b)
    commit = subprocess.run(["git", "rev-parse", "--short", "HEAD"], capture_output=True, text=True, cwd=ROOT).stdout.strip()
    doc = {"commit": commit or None, "csrc_sha1": csrc_hash(), "grid": N, "dtype": dtype, "report": os.path.basename(rep),
           "bytes_per_launch": {k: int(sum(v) / len(v)) for k, v in acc.items()},
           "launches_averaged": {k: len(v) for k, v in acc.items()}}
    json.dump(doc, open(TRAFFIC_JSON, "w"), indent=1)
    print(json.dumps(doc))


def peaks():
    """Measured HBM peak of this pool (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


# --------------------------------------------------------------------------------------------------
# algorithmic bytes per launch of each kernel class
def algorithmic_bytes(N1, N2, N3, s):
    nodes = (N1 + 1) * (N2 + 1) * (N3 + 1)
    cells = N1 * N2 * N3
    C1 = N1 + 1 if N1 > 1 else 1
    P2 = 2 * N2 if N2 > 1 else 1
    cx = 2 * s
    spec_a = 3 * cx * C1 * N2 * N3          # spectrum after the x pass
    spec_b = 3 * cx * C1 * P2 * N3          # after the y pass (3-D only)
    tensor = 6 * s * C1 * (N2 + 1) * (N3 + 1) if N3 > 1 else 4 * s * C1 * (N2 + 1)
    b = {
        "x_fwd": 3 * s * nodes + s * cells + spec_a,
        "x_inv": spec_a + 3 * s * cells,
        # node pass: m (3 nodal) + H^cell (3 cell) + materials (2 cell) in, then what the epilogue moves:
        "node": 3 * s * nodes + 5 * s * cells + 3 * s * nodes,                  # H or f out
        # Runge-Kutta stage (a10), mean over the four stages of RK4: the start-of-step state and stage states
        # in (0, 3, 3, 9 nodal arrays: stage 1 reads y0 as m), the next stage state out (3)
        "node_rk": 3 * s * nodes + 5 * s * cells + (3.75 + 3) * s * nodes,
        # adjoint passes (a11), mean of the two: pass 1 reads a, writes f, d, q (3 each) and w (1); pass 2
        # reads d and writes da/dt
        "node_adj": 3 * s * nodes + 5 * s * cells + (3 + 6.5) * s * nodes,
    }
    if N3 > 1:
        b["y_fwd"] = spec_a + spec_b
        b["y_inv"] = spec_a + spec_b
        b["mid"] = 2 * spec_b + tensor
    else:
        b["mid"] = 2 * spec_a + tensor
    return b


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.25] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
# the CPU oracle as it stands (cpu_baseline leg and --impl reference arm)
def oracle_sample_grid(n_steps_total, grid, forced=0):
    """Largest config-4 sample grid whose `n_steps_total` oracle steps finish in about two minutes
    (measured on 8 host cores: 10.7 s per step at 64^3, 1.2 s at 32^3, 0.15 s at 16^3)."""
    if forced:
        return forced
    for n, sec in ((64, 10.7), (32, 1.2), (16, 0.15)):
        if n <= grid and sec * n_steps_total <= 130.0:
            return n
    return min(16, grid)


def oracle_run(sample_n, dtype_name, steps, warmup, fft_workers=1):
    """Times `steps` oracle steps (rk4_step + adjoint_rhs, fp64 arithmetic on inputs rounded to the
    build precision) on the sample grid; the demag tensor setup is outside the timed region, like
    nm_mesh_create on the GPU side.  Returns (seconds, cells per step, threads)."""
    import numpy as np

    from oracle import adjoint, llg
    from paper_2411_11725_b200 import workloads as wl

    nd = np.float32 if dtype_name == "f32" else np.float64
    w = wl.config4_sweep(sample_n)
    r = lambda v: wl.round_to(w.cell_array(v), nd)
    p = llg.Problem(tuple(w.n_cells), tuple(w.dx), r(w.Ms), r(w.A), r(w.Ku), tuple(w.ku_axis),
                    float(w.gamma), float(w.alpha), int(w.terms))
    p.Nt                                    # setup (not timed)
    m = wl.round_to(w.m0, nd)
    a = wl.round_to(np.random.default_rng(99).standard_normal(m.shape), nd)

    def step(mm):
        mm = llg.rk4_step(p, 0.0, w.dt, mm)
        adjoint.adjoint_rhs(p, 0.0, mm, a)
        return mm

    def run():
        mm = m
        for _ in range(warmup):
            mm = step(mm)
        t0 = time.perf_counter()
        for _ in range(steps):
            mm = step(mm)
        return time.perf_counter() - t0

    if fft_workers <= 1:
        # numpy elementwise loops and numpy.fft (pocketfft) run on one thread; no BLAS call is made
        return run(), sample_n ** 3, 1
    # BASELINE.md 4's second line: the same oracle with its library FFT calls (numpy.fft.rfftn / irfftn,
    # the only routines it calls there) served by scipy.fft on `fft_workers` threads; everything else
    # in it stays single-threaded numpy.  The oracle's source is not touched: the two names are
    # swapped in numpy.fft for the duration of this leg.
    import scipy.fft as sfft
    keep = (np.fft.rfftn, np.fft.irfftn)
    np.fft.rfftn = lambda a, s=None, axes=None: sfft.rfftn(a, s=s, axes=axes, workers=fft_workers)
    np.fft.irfftn = lambda a, s=None, axes=None: sfft.irfftn(a, s=s, axes=axes, workers=fft_workers)
    try:
        return run(), sample_n ** 3, fft_workers
    finally:
        np.fft.rfftn, np.fft.irfftn = keep


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = oracle_sample_grid(args.steps + args.warmup, args.grid, args.sample_grid)
    sec, cells, threads = oracle_run(n, args.dtype, args.steps, args.warmup)
    value = EVALS_PER_STEP * cells * args.steps / sec / 1e6
    sample = ("config-4 recipe at %d^3 cells (the oracle cannot hold %d^3 in minutes); each step = "
              "oracle rk4_step + adjoint_rhs, tensor setup untimed" % (n, args.grid))
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "config4_sweep N=%d (sampled at %d^3)" % (args.grid, n),
                   "terms": "exchange+demag", "evals_per_step": EVALS_PER_STEP, "input_dtype": args.dtype},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


# --------------------------------------------------------------------------------------------------
# the other configurations, timed after the bench's own region (CUDA events, this process, one GPU)
def _dev_mesh(w, td):
    import numpy as np
    import torch

    from paper_2411_11725_b200 import binding as nm
    from paper_2411_11725_b200 import workloads as wl
    put = lambda a: torch.from_numpy(wl.to_abi(a)).to(device="cuda", dtype=td).contiguous()
    mat = {k: (float(getattr(w, k)) if np.isscalar(getattr(w, k)) else put(getattr(w, k))) for k in ("Ms", "A", "Ku")}
    mesh = nm.Mesh(w.n_cells, w.dx, dtype=td, device=torch.cuda.current_device(), terms=w.terms, gamma=w.gamma,
                   alpha=w.alpha, ku_axis=w.ku_axis, **mat)
    z = None
    if w.terms & wl.TERM_ZEEMAN:
        hp = put(w.h_pulse) if w.h_pulse is not None else None
        amp = (lambda t: wl.sinc_pulse(t, **w.pulse)) if (w.pulse and hp is not None) else None
        z = nm.Zeeman(h_uniform=w.h_uniform, h_pulse=hp, amp=amp)
    nd = np.float64 if td == torch.float64 else np.float32
    return mesh, z, put(wl.round_to(w.m0, nd))


def _event_ms(fn, n, warm=5):
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def _wall_ms(fn, n, warm=3):
    """Host wall clock per call, the stream drained on both sides (the paper's protocol: integration
    wall time divided by the number of field evaluations)."""
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(n):
        fn()
    torch.cuda.synchronize()
    return 1e3 * (time.perf_counter() - t0) / n


def sweep_block(peak):
    """nm_llg_rhs (and the steps each config is stated with) at the other points of config 4 and at the
    film configs 1, 3, 5: ms per call by CUDA events after warm-up, Mcells/s, and the fraction of the
    HBM peak over the algorithmic bytes of one evaluation (grids that fit the 126 MB L2 are marked)."""
    import torch

    from paper_2411_11725_b200 import binding as nm
    from paper_2411_11725_b200 import workloads as wl
    rows = []
    pts = [(wl.config4_sweep(n), td) for n, td in ((16, "f32"), (32, "f32"), (64, "f32"), (128, "f32"), (192, "f32"),
                                                    (64, "f64"), (128, "f64"), (192, "f64"), (256, "f64"))]
    pts += [(wl.config1_tiny_film(), "f64"), (wl.config2_cube(64), "f32"), (wl.config3_thin_film(512), "f32"),
            (wl.config5_inverse(), "f64")]
    for w, prec in pts:
        td = torch.float32 if prec == "f32" else torch.float64
        s = 4 if prec == "f32" else 8
        mesh, z, m = _dev_mesh(w, td)
        N1, N2, N3 = w.n_cells
        cells = N1 * N2 * N3
        big = cells >= 128 ** 3
        reps = 10 if big else 100
        out = torch.empty_like(m)
        l0 = mesh.nm_launch_count()
        mesh.nm_llg_rhs(0.0, m, z, out)
        per_rhs = mesh.nm_launch_count() - l0
        t_rhs = _event_ms(lambda: mesh.nm_llg_rhs(0.0, m, z, out), reps)
        y = m.clone()
        dt = w.dt if w.dt > 0 else 1e-13
        row = {"workload": w.name, "n_cells": [N1, N2, N3], "dtype": prec, "llg_rhs_ms": t_rhs,
               "mcells_per_s": cells / t_rhs / 1e3, "launches_per_rhs": per_rhs,
               "demag_path": mesh.nm_debug_demag_path(),
               "rk4_step_ms": _event_ms(lambda: mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, y, z), max(3, reps // 2))}
        # the paper's own protocol (Fig. 6): wall time of a fixed-step integration / field evaluations
        row["paper_protocol_ms_per_eval"] = _wall_ms(lambda: mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, y, z), max(5, reps)) / 4.0
        byts = sum(v for k, v in algorithmic_bytes(N1, N2, N3, s).items() if k not in ("node_rk", "node_adj"))
        row["algorithmic_bytes"] = byts
        row["frac"] = byts / (t_rhs * 1e-3) / 1e9 / peak
        row["l2_resident"] = byts < 126e6
        if w.name.startswith("config3"):
            y.copy_(m)
            row["dopri5_step_ms"] = _event_ms(lambda: mesh.nm_rk_step(nm.NM_DOPRI5, 1e-10, dt, y, z), 50)
            row["host_amplitude_callback"] = True
        if w.name.startswith("config5") or w.name.startswith("config1"):
            a = m.clone()
            u = torch.zeros(mesh.cell_shape_abi, dtype=td, device=m.device)
            row["adjoint_rk4_step_ms"] = _event_ms(lambda: mesh.nm_adjoint_rk4_step(0.0, dt, y, a, u, z), 50)
        rows.append(row)
        mesh.close()
        mesh.workspace = None
        del m, out, y
        torch.cuda.empty_cache()
    return rows


def run_config3(args):
    """Config 3 as BASELINE.json states it: 512x512x1 cells, fp32, stripe pulse, Dormand-Prince with
    rtol = atol = 1e-5 from 0 to args.config3 ns through drivers.integrate_dopri5 (one host read of the
    error norm per trial step).  Prints wall time, step counts, |m| and the internal energy."""
    import numpy as np
    import torch

    from paper_2411_11725_b200 import drivers
    from paper_2411_11725_b200 import workloads as wl
    w = wl.config3_thin_film(512)
    td = torch.float32
    mesh, z, y = _dev_mesh(w, td)

    def energy():
        H = mesh.nm_heff(0.0, y).double()
        cnt = []
        for N in w.n_cells:
            c = torch.full((N + 1,), 2.0, dtype=torch.float64, device=y.device)
            c[0] = c[-1] = 1.0
            cnt.append(c)
        L = cnt[2][:, None, None] * cnt[1][None, :, None] * cnt[0][None, None, :]
        L = L * (4e-7 * np.pi * float(w.Ms) * float(np.prod(w.dx)) / 8.0)
        return -0.5 * float((L * (y.double() * H).sum(0)).sum())

    E0 = energy()
    T = args.config3 * 1e-9
    l0 = mesh.nm_launch_count()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    t, dt, acc, rej = drivers.integrate_dopri5(mesh, y, 0.0, T, 1e-13, z)
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    evals = 7 * (acc + rej)
    print(json.dumps({
        "what": "config 3 stated recipe", "n_cells": list(w.n_cells), "dtype": "f32", "t_end_s": t,
        "wall_s": sec, "accepted": acc, "rejected": rej, "rhs_evaluations": evals, "last_dt_s": dt,
        "ms_per_trial_step": 1e3 * sec / (acc + rej), "mcells_per_s": evals * float(np.prod(w.n_cells)) / sec / 1e6,
        "gpu_launches": mesh.nm_launch_count() - l0,
        "max_abs_norm_minus_1": float((y.double().norm(dim=0) - 1).abs().max()),
        "finite": bool(torch.isfinite(y).all()), "energy_J": {"t0": E0, "t_end": energy()},
        "rtol": 1e-5, "atol": 1e-5}))


# --------------------------------------------------------------------------------------------------
# the CUDA path through the C-ABI
def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2411_11725_b200 import binding as nm
    from paper_2411_11725_b200 import replicas
    from paper_2411_11725_b200 import workloads as wl

    nm.lib()                                 # fails loudly if libnm.so is missing (no fallback)
    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    td = torch.float32 if args.dtype == "f32" else torch.float64
    s = 4 if args.dtype == "f32" else 8
    N = args.grid

    # seeded synthetic input, config 4's recipe (replica r uses seed 4 + N + r)
    w = wl.config4_sweep(N)
    if rank:
        w.m0 = wl.random_unit_field(w.node_shape, replicas.replica_seed(N, rank))
    m_host = torch.from_numpy(wl.to_abi(w.m0)).to(td).pin_memory()
    a_host = torch.from_numpy(wl.to_abi(
        np.random.default_rng(99 + rank).standard_normal((3,) + w.node_shape))).to(td).pin_memory()
    mesh = nm.Mesh(w.n_cells, w.dx, dtype=td, device=local, terms=w.terms, gamma=w.gamma, alpha=w.alpha,
                   Ms=float(w.Ms), A=float(w.A), Ku=0.0)
    m = m_host.to(dev)
    a = a_host.to(dev)
    f_out = torch.empty_like(m)
    dadt = torch.empty_like(m)
    dudt = torch.empty(mesh.cell_shape_abi, dtype=td, device=dev)
    dt = w.dt
    L = nm.lib()
    import ctypes
    vp = ctypes.c_void_p

    def step():
        mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, m)
        nm._check(L.nm_llg_adjoint_rhs(mesh.handle, 0.0, vp(m.data_ptr()), vp(a.data_ptr()), None,
                                       vp(f_out.data_ptr()), vp(dadt.data_ptr()), vp(dudt.data_ptr()),
                                       nm._stream(local)))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n):
        """CUDA-event time of n back-to-back calls of fn on the current stream, seconds."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        barrier()
        return e0.elapsed_time(e1) * 1e-3

    def over_ranks(sec):
        return replicas.max_over_ranks(sec, dev)

    for _ in range(args.warmup):
        step()
    # ---- the timed region: K steps, per-kernel events on (roofline), clocks sampled ----
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = mesh.nm_launch_count()
    mesh.nm_profile_begin()
    w0 = time.time()
    sec = over_ranks(timed(step, args.steps))
    w1 = time.time()
    prof = mesh.nm_profile_end()
    mesh_dropped = mesh.nm_profile_dropped()
    launches = mesh.nm_launch_count() - launches0
    clocks = sampler.stop(w0, w1) if sampler else None
    # the same K steps without the per-kernel events (what the events cost)
    sec_plain = over_ranks(timed(step, args.steps))

    cells = N ** 3
    value = replicas.job_value(world, EVALS_PER_STEP, cells, args.steps, sec)

    # ---- breakdown: the three calls of BASELINE.json's metric, timed alone ----
    H = torch.empty_like(m)
    reps = max(5, args.steps)
    _timed = timed

    def timed(fn, n):       # one untimed call first: a kernel variant's first launch loads its module
        fn()
        return _timed(fn, n)
    t_heff = over_ranks(timed(lambda: mesh.nm_heff(0.0, m, None, H), reps)) / reps
    t_rhs = over_ranks(timed(lambda: mesh.nm_llg_rhs(0.0, m, None, H), reps)) / reps
    t_rk4 = over_ranks(timed(lambda: mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, m), reps)) / reps
    t_paper = _wall_ms(lambda: mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, m), reps) / 4.0
    t_adj = over_ranks(timed(lambda: nm._check(L.nm_llg_adjoint_rhs(
        mesh.handle, 0.0, vp(m.data_ptr()), vp(a.data_ptr()), None, vp(f_out.data_ptr()),
        vp(dadt.data_ptr()), vp(dudt.data_ptr()), nm._stream(local))), reps)) / reps

    # ---- end to end: host buffers, copies inside the timed region ----
    m_back = torch.empty_like(m_host).pin_memory()
    da_back = torch.empty_like(m_host).pin_memory()
    du_back = torch.empty(mesh.cell_shape_abi, dtype=td).pin_memory()

    # Steps are independent jobs (each brings its own m and a from the host), so the copies of
    # neighbouring steps overlap the kernels: inputs of step i + 1 go up on a copy stream while step i
    # computes on the main stream, and the results of step i - 1 come down on a third stream.  Every
    # step still moves all of its inputs and results inside the timed region; three sets of device
    # buffers rotate (with two, the upload of step i + 1 would wait for the download of step i - 1 out
    # of the same set, and the two copy directions would run one after the other), and events order
    # copy -> compute -> copy per set.
    cur = torch.cuda.current_stream(dev)
    s_up, s_down = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    buf = [dict(m=torch.empty_like(m), a=torch.empty_like(a), dadt=torch.empty_like(m),
                dudt=torch.empty_like(dudt), up=torch.cuda.Event(), done=torch.cuda.Event(),
                down=torch.cuda.Event()) for _ in range(3)]
    state = {"i": 0}

    def step_e2e():
        b = buf[state["i"] % 3]
        state["i"] += 1
        s_up.wait_event(b["down"])                  # the previous results of this buffer have left it
        with torch.cuda.stream(s_up):
            b["m"].copy_(m_host, non_blocking=True)
            b["a"].copy_(a_host, non_blocking=True)
            b["up"].record(s_up)
        cur.wait_event(b["up"])
        mesh.nm_rk_step(nm.NM_RK4, 0.0, dt, b["m"])
        nm._check(L.nm_llg_adjoint_rhs(mesh.handle, 0.0, vp(b["m"].data_ptr()), vp(b["a"].data_ptr()), None,
                                       vp(f_out.data_ptr()), vp(b["dadt"].data_ptr()), vp(b["dudt"].data_ptr()),
                                       nm._stream(local)))
        b["done"].record(cur)
        s_down.wait_event(b["done"])
        with torch.cuda.stream(s_down):
            m_back.copy_(b["m"], non_blocking=True)
            da_back.copy_(b["dadt"], non_blocking=True)
            du_back.copy_(b["dudt"], non_blocking=True)
            b["down"].record(s_down)

    def timed_e2e(n):
        """As timed(), closing the region only when the last results are back on the host."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(n):
            step_e2e()
        cur.wait_stream(s_down)
        cur.wait_stream(s_up)
        e1.record()
        barrier()
        return e0.elapsed_time(e1) * 1e-3

    for _ in range(3):
        step_e2e()
    sec_e2e = over_ranks(timed_e2e(args.steps))
    h2d = 2 * m_host.numel() * s
    d2h = (2 * m_host.numel() + du_back.numel()) * s
    e2e_value = replicas.job_value(world, EVALS_PER_STEP, cells, args.steps, sec_e2e)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (largest share of the timed region) ----
    peak, peak_src = peaks()
    traffic, traffic_src = load_traffic(N, args.dtype)
    alg = algorithmic_bytes(N, N, N, s)
    shares = {k: v[0] for k, v in prof.items() if v[1] > 0}
    tot_ms = sum(shares.values())
    dom = max((k for k in shares if k in alg), key=lambda k: shares[k])
    dom_ms, dom_n = prof[dom]
    achieved = alg[dom] / (dom_ms * 1e-3 / dom_n) / 1e9
    eval_bytes = sum(v for k, v in alg.items() if k not in ("node_rk", "node_adj"))   # one nm_llg_rhs
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic.get(dom),
                "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg[dom], "launches": dom_n,
                "avg_launch_ms": dom_ms / dom_n, "share_of_step": dom_ms / tot_ms}
    # The z pass is as close to the FP32 pipe as to HBM: the same launch against the
    # arithmetic peak.  Lane operations per launch from the committed ncu capture (packed
    # FADD2/FMUL2/FFMA2 = 64 per warp instruction, scalar = 32; profiles/r1d_packed.md); peak =
    # 128 FP32 lanes per clock and SM at the maximum SM clock.
    roofline_alu = None
    if dom == "mid" and (N, args.dtype) == (256, "f32"):
        lane_ops = 1.32e10
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        alu_peak = 128.0 * sm_count * float((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6
        alu_ach = lane_ops / (dom_ms * 1e-3 / dom_n)
        roofline_alu = {"bound": "alu", "kernel": dom, "achieved": alu_ach / 1e12, "peak": alu_peak / 1e12,
                        "unit": "T FP32 lane-op/s", "frac": alu_ach / alu_peak,
                        "lane_ops_per_launch": lane_ops, "source": "profiles/r1d_packed.md"}
    per_kernel = {k: {"ms_per_launch": prof[k][0] / prof[k][1], "launches": prof[k][1],
                      "share": prof[k][0] / tot_ms,
                      "GBps": (alg[k] / (prof[k][0] * 1e-3 / prof[k][1]) / 1e9) if k in alg else None}
                  for k in shares}
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": "config4_sweep N=%d: %d^3 cells, 2 nm, exchange+demag, seeded random unit m"
                               % (N, N), "evals_per_step": EVALS_PER_STEP,
                   "step": "nm_rk_step(RK4) + nm_llg_adjoint_rhs", "parallelism": "replicas x%d" % world,
                   "l2": "inputs larger than L2" if 9 * (N + 1) ** 3 * s > 126e6 else "L2-resident grid",
                   "workspace_bytes": mesh.workspace_bytes},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * sec_e2e / args.steps,
                "how": "host pinned buffers; per step H2D of m and a, D2H of m, da/dt, du/dt; copies of "
                       "neighbouring steps overlap the kernels (3 streams, three rotating sets of device arrays)"},
        "gpu_launches": launches,
        "clocks": clocks,
        "roofline": roofline,
        "roofline_alu": roofline_alu,
        "roofline_eval": {"what": "one fused nm_llg_rhs: algorithmic bytes of all passes / its time",
                          "bytes": eval_bytes, "ms": 1e3 * t_rhs, "achieved": eval_bytes / t_rhs / 1e9,
                          "frac": eval_bytes / t_rhs / 1e9 / peak, "frac_of_8TBps_nominal":
                          eval_bytes / t_rhs / 1e9 / 8000.0},
        "kernels": per_kernel,
        "breakdown": {"heff_ms": 1e3 * t_heff, "heff_mcells_per_s": cells / t_heff / 1e6,
                      "llg_rhs_ms": 1e3 * t_rhs, "llg_rhs_mcells_per_s": cells / t_rhs / 1e6,
                      "rk4_step_ms": 1e3 * t_rk4, "rk4_steps_per_s": 1.0 / t_rk4,
                      "paper_protocol_ms_per_eval": t_paper,      # RK4 integration wall time / field evaluations
                      "adjoint_rhs_ms": 1e3 * t_adj,
                      "ms_per_step_without_kernel_events": 1e3 * sec_plain / args.steps},
    }
    if not args.no_sweep and world == 1:
        mesh.close()
        mesh.workspace = None            # the bench mesh's 5.4 GB go back before the sweep's meshes come
        buf.clear()
        torch.cuda.empty_cache()
        out["sweep"] = sweep_block(peak)
    if out["kernels"] and mesh_dropped:
        out["profile_dropped_launches"] = mesh_dropped
    if not args.no_cpu_baseline and world == 1:
        n = args.sample_grid or min(64, N)
        csteps = 3                  # about 15 s of CPU work at 64^3 on the GPU box's host
        csec, ccells, threads = oracle_run(n, args.dtype, csteps, 0)
        out["cpu_baseline"] = {
            "value": EVALS_PER_STEP * ccells * csteps / csec / 1e6, "unit": UNIT, "cores": threads,
            "kind": "oracle", "host_cores": os.cpu_count(),
            "sample": "%d oracle steps (rk4_step + adjoint_rhs) of the config-4 recipe at %d^3 cells, "
                      "%.1f s, tensor setup untimed" % (csteps, n, csec)}
        # the same sample with the oracle's FFT calls on every host core
        tsec, _, tthreads = oracle_run(n, args.dtype, csteps, 0, fft_workers=os.cpu_count() or 1)
        out["cpu_baseline"]["threaded_fft"] = {
            "value": EVALS_PER_STEP * ccells * csteps / tsec / 1e6, "unit": UNIT, "cores": tthreads,
            "how": "numpy.fft.rfftn / irfftn served by scipy.fft(workers=%d); the rest of the oracle is "
                   "single-threaded numpy; %.1f s" % (tthreads, tsec)}
    else:
        out["cpu_baseline"] = None
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a_ = parse()
    if a_.traffic_from:
        write_traffic(a_.traffic_from, a_.grid, a_.dtype)
    elif a_.impl == "reference":
        run_reference(a_)
    elif a_.config3 > 0:
        run_config3(a_)
    else:
        run_b200(a_)
