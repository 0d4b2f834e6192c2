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
    return ap.parse_args()


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch of each kernel class from the
# committed `ncu --set full` capture of this command (profiles/r1e_final.md); only for the workload
# that capture was taken on (256^3, fp32)
NCU_TRAFFIC = {(256, "f32"): {"mid": 2025138896, "y_fwd": 1195136896, "y_inv": 1215810952,
                              "x_fwd": 569166424, "x_inv": 586457048, "node": 808990384}}


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
        "node": 3 * s * nodes + 2 * s * cells + 3 * s * cells + 3 * s * nodes,
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


def oracle_run(sample_n, dtype_name, steps, warmup):
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

    for _ in range(warmup):
        m = step(m)
    t0 = time.perf_counter()
    for _ in range(steps):
        m = step(m)
    sec = time.perf_counter() - t0
    # numpy elementwise loops and numpy.fft (pocketfft) run on one thread; no BLAS call is made
    return sec, sample_n ** 3, 1


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
    alg = algorithmic_bytes(N, N, N, s)
    shares = {k: v[0] for k, v in prof.items() if v[1] > 0}
    tot_ms = sum(shares.values())
    dom = max((k for k in shares if k in alg), key=lambda k: shares[k])
    dom_ms, dom_n = prof[dom]
    achieved = alg[dom] / (dom_ms * 1e-3 / dom_n) / 1e9
    eval_bytes = sum(alg.values())
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC.get((N, args.dtype), {}).get(dom),
                "traffic_source": "profiles/r1e_final.md (ncu --set full, per launch)", "peak_source": peak_src,
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
                      "adjoint_rhs_ms": 1e3 * t_adj,
                      "ms_per_step_without_kernel_events": 1e3 * sec_plain / args.steps},
    }
    if not args.no_cpu_baseline and world == 1:
        n = args.sample_grid or min(64, N)
        csteps = 3                  # about 15 s of CPU work at 64^3 on the GPU box's host
        csec, ccells, threads = oracle_run(n, args.dtype, csteps, 0)
        out["cpu_baseline"] = {
            "value": EVALS_PER_STEP * ccells * csteps / csec / 1e6, "unit": UNIT, "cores": threads,
            "kind": "oracle", "host_cores": os.cpu_count(),
            "sample": "%d oracle steps (rk4_step + adjoint_rhs) of the config-4 recipe at %d^3 cells, "
                      "%.1f s, tensor setup untimed" % (csteps, n, csec)}
    else:
        out["cpu_baseline"] = None
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a_ = parse()
    if a_.impl == "reference":
        run_reference(a_)
    else:
        run_b200(a_)
