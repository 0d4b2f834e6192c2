"""Whole-step CUDA-graph replay (nm_api.cu `run_step`) against plain launches and the oracle.

Small meshes are launch-latency-bound, so `nm_rk_step` / `nm_adjoint_rk4_step` replay a time step
as one CUDA graph once the same arguments (scheme, dt, state pointers, tolerances, Zeeman arrays)
arrive twice in a row.  NM_GRAPH = 0 / 1 (read at nm_mesh_create) forces plain launches / replay.
The replayed step launches the same kernels with the same arguments, so its results must be
bit-identical to the plain launches: across a change of dt, of the state buffer, of Ms
(nm_mesh_set_Ms invalidates the cached step) and of the integration scheme; and the replayed
trajectory is held to the fp64 oracle like any other (a10, a11).
"""
import os

import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import dev, gpu_mesh, gpu_zeeman, host, np_dtype, oracle_problem, oracle_zeeman, rel_l2

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


def _mesh(w, td, graph):
    old = os.environ.get("NM_GRAPH")
    os.environ["NM_GRAPH"] = "1" if graph else "0"
    try:
        return gpu_mesh(w, td)
    finally:
        if old is None:
            os.environ.pop("NM_GRAPH", None)
        else:
            os.environ["NM_GRAPH"] = old


def _case(n, seed=5):
    """All four terms, cell-wise Ms with a vacuum block, uniform + static nodal Zeeman field, no
    time-dependent pulse (a host amplitude callback keeps a step on plain launches)."""
    w, hs = wl.varied_case(n, vacuum=True, seed=seed)
    w.pulse = None
    w.h_pulse = None
    return w, hs


def _m0(w, td, seed=3):
    return wl.round_to(wl.random_unit_field(w.node_shape, seed), np_dtype(td))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(12, 6, 4), (32, 32, 32), (48, 24, 1)])
def test_rk4_replay_bit_identical_and_oracle(n, prec):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = _case(n)
    m0 = _m0(w, td)
    out = {}
    for graph in (False, True):
        mesh = _mesh(w, td, graph)
        gz = gpu_zeeman(w, td, h_static=hs)
        assert gz is None or gz._keep[2] is None
        y = dev(m0, td)
        for s in range(5):
            mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
        a = y.clone()
        for s in range(3):                              # another step size
            mesh.nm_rk_step(0, 0.0, 0.5 * w.dt, y, gz)
        b = y.clone()
        y2 = dev(m0, td)                                # another state buffer, no renormalisation
        for s in range(3):
            mesh.nm_rk_step(0, 0.0, w.dt, y2, gz, renormalise=False)
        for s in range(3):                              # and without the external field
            mesh.nm_rk_step(0, 0.0, w.dt, y2, None)
        out[graph] = (a, b, y2.clone(), mesh.nm_launch_count())
        mesh.close()
    for u, v in zip(out[False][:3], out[True][:3]):
        assert torch.equal(u, v)
    assert out[False][3] == out[True][3]                # replayed kernels are counted like launched ones
    if n == (12, 6, 4):
        p = oracle_problem(w, nd)
        z = oracle_zeeman(w, nd, hs)
        ref = m0
        for s in range(5):
            ref = llg.rk4_step(p, s * w.dt, w.dt, ref, z)
        assert rel_l2(host(out[True][0]), ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_dopri5_replay_bit_identical(prec):
    td = DT[prec]
    w, hs = _case((16, 12, 3))
    m0 = _m0(w, td)
    out = {}
    for graph in (False, True):
        mesh = _mesh(w, td, graph)
        gz = gpu_zeeman(w, td, h_static=hs)
        y = dev(m0, td)
        errs = []
        for dt in (2e-14, 2e-14, 2e-14, 2e-14, 2e-13, 2e-13, 2e-13, 4e-14):   # 2e-13: rejected steps
            errs.append(mesh.nm_rk_step(1, 0.0, dt, y, gz, rtol=1e-5, atol=1e-5, want_err=True))
        for _ in range(3):                              # no read-back of the error norm
            mesh.nm_rk_step(1, 0.0, 3e-14, y, gz, rtol=1e-5, atol=1e-5)
        for _ in range(3):                              # RK4 in between keeps its own cached step
            mesh.nm_rk_step(0, 0.0, 3e-14, y, gz)
        out[graph] = (y.clone(), errs)
        mesh.close()
    assert torch.equal(out[False][0], out[True][0])
    assert out[False][1] == out[True][1]
    assert out[True][1][4] > 1.0 and out[True][1][0] <= 1.0


def test_adjoint_rk4_replay_bit_identical_and_set_Ms_fp64():
    from oracle import adjoint
    td = torch.float64
    w = wl.config5_inverse((32, 8, 1), n_steps=12)
    m0 = _m0(w, td)
    aT = wl.objective_weights(w)
    Ms2 = wl.round_to(w.cell_array(w.Ms) * 1.1, np.float64)
    out = {}
    for graph in (False, True):
        mesh = _mesh(w, td, graph)
        gz = gpu_zeeman(w, td)
        y = dev(m0, td)
        for s in range(w.n_steps):
            mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
        yT = y.clone()
        a = dev(aT, td)
        u = torch.zeros(mesh.cell_shape_abi, dtype=td, device="cuda:0")
        for s in range(w.n_steps, 0, -1):
            mesh.nm_adjoint_rk4_step(s * w.dt, w.dt, y, a, u, gz)
        first = (yT, y.clone(), a.clone(), u.clone())
        # other Ms on the same mesh, same buffers: the cached steps must not be replayed as they are
        mesh.nm_mesh_set_Ms(dev(Ms2, td))
        for s in range(4):
            mesh.nm_rk_step(0, 0.0, w.dt, y, gz)
        for s in range(4):
            mesh.nm_adjoint_rk4_step(0.0, w.dt, y, a, u, gz)
        out[graph] = first + (y.clone(), a.clone(), u.clone())
        mesh.close()
    for p_, q_ in zip(out[False], out[True]):
        assert torch.equal(p_, q_)
    # and the replayed backward pass against the oracle
    p = oracle_problem(w)
    z = oracle_zeeman(w)
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=0)
    assert rel_l2(host(out[True][0]), mT_ref) <= 1e-11
    # no checkpoints: the backward pass integrates m backwards itself (reading C8)
    _, a0_ref, u0_ref = adjoint.backward_rk4(p, mT_ref, aT, w.dt, w.n_steps, z, checkpoints=None)
    assert rel_l2(host(out[True][2]), a0_ref) <= 1e-11
    assert rel_l2(wl.from_abi(out[True][3].cpu().numpy()), u0_ref) <= 1e-11


def test_steps_inside_a_graph_the_caller_captures():
    """A caller that captures its own CUDA graph (here: torch.cuda.graph) around nm_rk_step gets plain
    launches recorded into that graph: the library neither starts a capture of its own nor launches
    its cached step while the caller's stream is capturing, and replaying the caller's graph
    advances the state like the steps themselves."""
    td = torch.float64
    w, hs = _case((12, 6, 4))
    mesh = _mesh(w, td, True)
    gz = gpu_zeeman(w, td, h_static=hs)
    y = dev(_m0(w, td), td)
    mesh.nm_rk_step(0, 0.0, w.dt, y, gz)                # these arguments have been seen once
    want = y.clone()
    for _ in range(4):
        mesh.nm_rk_step(0, 0.0, w.dt, want, gz)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        mesh.nm_rk_step(0, 0.0, w.dt, y, gz)            # would be the library's own capture
        mesh.nm_rk_step(0, 0.0, w.dt, y, gz)
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(y, want)
    mesh.nm_rk_step(0, 0.0, w.dt, y, gz)                # and the library's replay still works afterwards
    mesh.nm_rk_step(0, 0.0, w.dt, y, gz)
    for _ in range(2):
        mesh.nm_rk_step(0, 0.0, w.dt, want, gz)
    assert torch.equal(y, want)
    mesh.close()
