"""GPU parity of the three node-kernel forms against the fp64 oracle (a5-a11).

With uniform A and Ku the library evaluates the local terms through separable operators, either
in the column-marching kernel (k_node_col: whole node rows per CTA, a ring of plane stages fed by a
producer warp with bulk copies when N1 is 128 or 256, else -- or with NM_NODE_PATH=ring -- by cp.async
of every thread; grids with 96 <= N1 + 1 <= 320) or in the patch kernel (k_node_sep); cell-wise A / Ku
use the 27-point kernel (k_node).  NM_NODE_PATH selects a form for the meshes created while it is set, so each form
is held to the same oracle on the same inputs: every mode of the epilogue (H, f, RK4 stages,
Dormand-Prince stages with the error norm, both adjoint passes), cell-wise Ms with a vacuum block
and scalar Ms, grids whose z extent spans several z chunks and whose last row tile is ragged.
"""
import os

import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import assert_parity, dev, gpu_mesh, gpu_zeeman, host, np_dtype, oracle_problem, oracle_zeeman, rel_l2

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


@pytest.fixture(params=["auto", "ring", "sep", "generic"])
def node_path(request):
    old = os.environ.get("NM_NODE_PATH")
    if request.param == "auto":
        os.environ.pop("NM_NODE_PATH", None)
    else:
        os.environ["NM_NODE_PATH"] = request.param
    yield request.param
    if old is None:
        os.environ.pop("NM_NODE_PATH", None)
    else:
        os.environ["NM_NODE_PATH"] = old


def _case(n, uniform_ms, seed=21):
    """varied_case with scalar A and Ku (the separable operators' precondition) and no nodal field."""
    w, _ = wl.varied_case(n, vacuum=not uniform_ms, seed=seed)
    w.A = 1.1e-11
    w.Ku = 3e5
    if uniform_ms:
        w.Ms = 7e5
    return w


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("uniform_ms", [False, True])
@pytest.mark.parametrize("n", [(96, 9, 4), (128, 16, 16), (108, 4, 48), (243, 2, 3), (256, 5, 42), (128, 1, 1)])
def test_heff_and_rhs(n, uniform_ms, prec, node_path):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w = _case(n, uniform_ms)
    p = oracle_problem(w, nd)
    m = wl.round_to(w.m0, nd)
    z = oracle_zeeman(w, nd)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    H = host(mesh.nm_heff(0.0, dev(m, td), gz))
    ref = llg.effective_field(p, m, z(0.0))
    assert_parity(H, ref, TOL[prec], 'H')
    f = host(mesh.nm_llg_rhs(0.0, dev(m, td), gz))
    assert_parity(f, llg.llg_rhs(p, 0.0, m, z), TOL[prec], 'f')
    if not uniform_ms:
        from oracle.mesh import scatter_cells_to_nodes
        vac = scatter_cells_to_nodes(w.cell_array(w.Ms)) == 0
        assert vac.any() and np.all(H[:, vac] == 0)          # reading C3(iii)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("uniform_ms", [False, True])
def test_exchange_only_and_demag_only(uniform_ms, prec, node_path):
    """Term subsets: no demag (no cell tiles in the stage ring) and demag alone."""
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    for terms in (wl.TERM_EXCHANGE | wl.TERM_ANISO, wl.TERM_DEMAG, wl.TERM_EXCHANGE | wl.TERM_ZEEMAN):
        w = _case((144, 3, 6), uniform_ms)
        w.terms = terms
        p = oracle_problem(w, nd)
        m = wl.round_to(w.m0, nd)
        z = oracle_zeeman(w, nd)
        H = host(gpu_mesh(w, td).nm_heff(0.0, dev(m, td), gpu_zeeman(w, td)))
        assert_parity(H, llg.effective_field(p, m, z(0.0) if z else None), TOL[prec], 'terms %d' % terms)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("uniform_ms", [False, True])
def test_rk4_and_dopri5(uniform_ms, prec, node_path):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w = _case((96, 6, 48), uniform_ms)
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    m = wl.round_to(w.m0, nd)
    ref = m.copy()
    y = dev(m, td)
    for s in range(3):
        ref = llg.rk4_step(p, s * w.dt, w.dt, ref, z)
        mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
    assert rel_l2(host(y), ref) <= TOL[prec]
    ref2 = llg.rk4_step(p, 0.0, w.dt, m, z, renormalise=False)
    y2 = dev(m, td)
    mesh.nm_rk_step(0, 0.0, w.dt, y2, gz, renormalise=False)
    assert rel_l2(host(y2), ref2) <= TOL[prec]
    for dt, expect in ((5e-14, True), (4e-13, False)):
        out, err_ref, acc = llg.dopri5_step(p, 0.0, dt, m, z, rtol=1e-5, atol=1e-5)
        assert acc == expect
        y = dev(m, td)
        err = mesh.nm_rk_step(1, 0.0, dt, y, gz, rtol=1e-5, atol=1e-5, want_err=True)
        assert abs(err - err_ref) <= (1e-8 * err_ref if prec == "f64" else 2e-2 * err_ref + 1e-4)
        assert rel_l2(host(y), out) <= TOL[prec]
        if not expect:
            assert np.array_equal(host(y), m)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("uniform_ms", [False, True])
def test_adjoint_rhs(uniform_ms, prec, node_path):
    from oracle import adjoint
    td = DT[prec]
    nd = np_dtype(td)
    w = _case((96, 6, 4), uniform_ms)
    if not uniform_ms:
        w.Ms = np.where(w.Ms == 0, 5e5, w.Ms)     # S Ms > 0 everywhere: the Ms gradient is defined at every cell
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd)
    m = wl.round_to(w.m0, nd)
    a = wl.round_to(np.random.default_rng(78).standard_normal(m.shape), nd)
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a, z)
    mesh = gpu_mesh(w, td)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, td), dev(a, td), gpu_zeeman(w, td))
    assert rel_l2(host(f), f_ref) <= TOL[prec]
    assert rel_l2(host(da), da_ref) <= TOL[prec]
    assert rel_l2(host(du), du_ref) <= TOL[prec]
