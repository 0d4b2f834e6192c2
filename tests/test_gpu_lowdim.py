"""GPU parity of the reduced 2-D / 1-D nodal bases (Eqs. 23-24):
nm_mesh_desc.basis = 2 (films, N3 = 1) and 1 (rods, N2 = N3 = 1) against oracle/lowdim.py, through
the C-ABI, and the paper's own check: the 3-D and the 2-D discretisation of a film give
the same trajectory."""
import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import (assert_parity, dev, gpu_mesh, gpu_zeeman, host, np_dtype, oracle_problem, oracle_zeeman,
                    reduce_nodal, rel_l2)

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


def _reduced(w, hs, D):
    """The workload on the D-dimensional basis: nodal inputs restricted to the basis nodes."""
    w.m0 = reduce_nodal(w.m0, D)
    if w.h_pulse is not None:
        w.h_pulse = reduce_nodal(w.h_pulse, D)
    return w, (reduce_nodal(hs, D) if hs is not None else None)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,D", [((24, 12, 1), 2), ((9, 35, 1), 2), ((1, 6, 1), 2), ((64, 64, 1), 2),
                                 ((50, 1, 1), 1), ((16, 1, 1), 1), ((1, 1, 1), 1), ((1, 1, 1), 2)])
def test_heff_and_rhs_all_terms_reduced_basis(n, D, prec):
    """Every term on, cell-wise random Ms (vacuum block), A, Ku, tilted axis, nodal static field."""
    from oracle import llg
    td, nd = DT[prec], np_dtype(DT[prec])
    w, hs = _reduced(*wl.varied_case(n, vacuum=(n[0] >= 6)), D)
    p = oracle_problem(w, nd, basis=D)
    z = oracle_zeeman(w, nd, hs)
    m = wl.round_to(w.m0, nd)
    mesh = gpu_mesh(w, td, basis=D)
    assert mesh.node_shape_abi == (3,) + tuple(reversed(p.node_shape))
    gz = gpu_zeeman(w, td, h_static=hs)
    ref = llg.effective_field(p, m, z(0.0))
    got = host(mesh.nm_heff(0.0, dev(m, td), gz))
    assert_parity(got, ref, TOL[prec], "H")
    vac = p.L == 0
    assert np.all(got[:, vac] == 0)
    assert_parity(host(mesh.nm_llg_rhs(0.0, dev(m, td), gz)), llg.llg_rhs(p, 0.0, m, z), TOL[prec], "f")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_heff_term_by_term_on_a_film(prec):
    from oracle import llg
    td, nd = DT[prec], np_dtype(DT[prec])
    for term in (wl.TERM_EXCHANGE, wl.TERM_DEMAG, wl.TERM_ANISO, wl.TERM_ZEEMAN):
        w, hs = _reduced(*wl.varied_case((12, 6, 1)), 2)
        w.terms = term
        p = oracle_problem(w, nd, basis=2)
        z = oracle_zeeman(w, nd, hs)
        m = wl.round_to(w.m0, nd)
        ref = llg.effective_field(p, m, z(0.0) if z else None)
        got = host(gpu_mesh(w, td, basis=2).nm_heff(0.0, dev(m, td), gpu_zeeman(w, td, h_static=hs)))
        assert_parity(got, ref, TOL[prec], "term %d" % term)


def test_config1_film_on_the_2d_basis_trajectory_fp64():
    """Config 1 (32x8x1, exchange + demag, 200 RK4 steps of 1e-13 s) with the film basis: 33x9 nodes
    instead of 33x9x2."""
    from oracle import llg
    w, _ = _reduced(wl.config1_tiny_film(), None, 2)
    td = torch.float64
    p = oracle_problem(w, basis=2)
    ref = w.m0.copy()
    mesh = gpu_mesh(w, td, basis=2)
    y = dev(ref, td)
    assert y.shape == (3, 1, 9, 33)
    worst = 0.0
    for s in range(w.n_steps):
        ref = llg.rk4_step(p, s * w.dt, w.dt, ref)
        mesh.nm_rk_step(0, s * w.dt, w.dt, y)
        if s % 50 == 49:
            worst = max(worst, rel_l2(host(y), ref))
    assert worst <= 1e-11
    assert np.max(np.abs(np.sqrt(np.sum(host(y) ** 2, axis=0)) - 1.0)) < 1e-14


def test_3d_and_2d_discretisation_of_a_film_agree_fp64():
    """the full 3-D discretisation and the 2-D one of Sec. III C give the same averaged
    magnetisation over time.  Config 1 from a state that is uniform through the thickness: the 3-D run
    (two node layers) stays uniform through the thickness and equals the 2-D run node by node."""
    w3 = wl.config1_tiny_film()
    w3.m0 = np.repeat(reduce_nodal(w3.m0, 2), 2, axis=3)
    w2, _ = _reduced(wl.config1_tiny_film(), None, 2)
    td = torch.float64
    m3, m2 = gpu_mesh(w3, td), gpu_mesh(w2, td, basis=2)
    y3, y2 = dev(w3.m0, td), dev(w2.m0, td)
    for s in range(w3.n_steps):
        m3.nm_rk_step(0, s * w3.dt, w3.dt, y3)
        m2.nm_rk_step(0, s * w2.dt, w2.dt, y2)
        if s % 40 == 39:
            a3 = y3.mean(dim=(1, 2, 3))
            a2 = y2.mean(dim=(1, 2, 3))
            assert float((a3 - a2).abs().max()) <= 1e-12
    assert float((y3[:, 0] - y3[:, 1]).abs().max()) <= 1e-12
    assert float((y3[:, :1] - y2).abs().max()) <= 1e-11
    assert float((y2 - dev(w2.m0, td)).abs().max()) > 1e-3        # the state did move


def test_dormand_prince_on_a_2d_film_with_the_stripe_pulse_fp32():
    """Config 3's recipe (stripe pulse through the weak form, Dormand-Prince) on a 64x64x1 film with
    the 2-D basis: 25 accepted steps replayed by the oracle."""
    from oracle import llg
    from paper_2411_11725_b200 import drivers
    w, _ = _reduced(wl.config3_thin_film(64), None, 2)
    td = torch.float32
    p = oracle_problem(w, np.float32, basis=2)
    z = oracle_zeeman(w, np.float32)
    mesh = gpu_mesh(w, td, basis=2)
    gz = gpu_zeeman(w, td)
    ref = wl.round_to(w.m0, np.float32)
    y = dev(ref, td)
    t, dt, accepted = w.pulse["t0"] - 2e-12, 1e-13, 0
    for _ in range(60):
        err = mesh.nm_rk_step(1, t, dt, y, gz, rtol=1e-5, atol=1e-5, want_err=True)
        out, err_ref, acc = llg.dopri5_step(p, t, dt, ref, z, rtol=1e-5, atol=1e-5)
        assert abs(err - err_ref) <= 2e-2 * err_ref + 1e-4
        if err <= 1.0:
            assert acc or abs(err_ref - 1.0) < 1e-2
            ref = out if acc else ref
            t += dt
            accepted += 1
        dt = drivers.dopri5_next_dt(dt, err)
        if accepted >= 25:
            break
    assert accepted >= 10
    assert_parity(host(y), ref, 1e-5, "film state")


def test_reduced_basis_boundary_behaviour():
    from paper_2411_11725_b200 import binding as nm
    for n, basis in (((8, 8, 2), 2), ((8, 2, 1), 1), ((8, 8, 1), 4)):
        with pytest.raises(nm.NmError) as e:
            nm.Mesh(n, (1e-9,) * 3, terms=1, Ms=8e5, A=1e-11, Ku=0.0, basis=basis)
        assert e.value.status == nm.NM_EINVAL
    # basis = 0 means the full basis
    full = nm.Mesh((8, 8, 1), (1e-9,) * 3, dtype=torch.float64, terms=3, Ms=8e5, A=1e-11, Ku=0.0, basis=0)
    assert full.node_shape_abi == (3, 2, 9, 9)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,D", [((24, 12, 1), 2), ((9, 35, 1), 2), ((50, 1, 1), 1), ((1, 1, 1), 2)])
def test_adjoint_entry_points_on_reduced_bases(n, D, prec):
    """SURVEY 8(f) rows 1 x 2: the adjoint right-hand side and every gradient on the 2-D / 1-D bases against the oracle
    (oracle/adjoint.py with the operators of oracle/lowdim.py): f, -(df/dm)^T a, -(df/dMs)^T a with every term on, a
    vacuum block and a nodal static field; the uniform- and nodal-field gradients; the A_c / Ku_c gradients; then the
    backward pass of (m, a, u, u_h, u_A, u_Ku, u_hn) over 20 RK4 steps with a checkpoint."""
    from oracle import adjoint
    from paper_2411_11725_b200 import drivers
    td, nd = DT[prec], np_dtype(DT[prec])
    w, hs = _reduced(*wl.varied_case(n, vacuum=(n[0] >= 6)), D)
    p = oracle_problem(w, nd, basis=D)
    z = oracle_zeeman(w, nd, hs)
    m = wl.round_to(w.m0, nd)
    a = wl.round_to(np.random.default_rng(61).standard_normal(m.shape), nd)
    mesh = gpu_mesh(w, td, basis=D)
    gz = gpu_zeeman(w, td, h_static=hs)
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a, z)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, td), dev(a, td), gz)
    assert_parity(host(f), f_ref, TOL[prec], "f")
    assert_parity(host(da), da_ref, TOL[prec], "da/dt")
    # the Ms gradient is a sum of pieces that cancel: fp32 bound as for the 3-D basis
    assert rel_l2(wl.from_abi(du.cpu().double().numpy()), du_ref) <= (1e-11 if prec == "f64" else 1e-5)
    uh = mesh.nm_llg_adjoint_rhs_hext(dev(m, td), dev(a, td)).cpu().numpy()
    uh_ref = adjoint.adjoint_rhs_hext(p, 0.0, m, a)
    assert np.max(np.abs(uh - uh_ref)) <= (1e-11 if prec == "f64" else 1e-5) * max(np.max(np.abs(uh_ref)), 1e-300)
    assert_parity(host(mesh.nm_llg_adjoint_rhs_hnodal(dev(m, td), dev(a, td))), adjoint.adjoint_rhs_hnodal(p, 0.0, m, a),
                  TOL[prec], "nodal-field gradient")
    gA, gKu = mesh.nm_llg_adjoint_rhs_materials(dev(m, td), dev(a, td))
    gA_ref, gKu_ref = adjoint.adjoint_rhs_materials(p, 0.0, m, a)
    assert rel_l2(wl.from_abi(gA.cpu().double().numpy()), gA_ref) <= TOL[prec]
    assert rel_l2(wl.from_abi(gKu.cpu().double().numpy()), gKu_ref) <= TOL[prec]
    # backward pass
    dt, nst = 2e-14, 20
    wT = wl.round_to(np.random.default_rng(62).standard_normal(m.shape), nd)
    mT_ref, ck = adjoint.forward_rk4(p, m, dt, nst, z, checkpoint_every=10)
    ref = adjoint.backward_rk4(p, mT_ref, wT, dt, nst, z, checkpoints=ck, with_hext=True, with_materials=True,
                               with_hnodal=True)
    gT = dev(wT, td)
    out = drivers.adjoint_gradient(mesh, dev(m, td), lambda mm: gT, dt, nst, gz, checkpoint_every=10, with_hext=True,
                                   with_materials=True, with_hnodal=True)
    assert rel_l2(host(out[0]), mT_ref) <= TOL[prec]
    assert rel_l2(host(out[1]), ref[1]) <= TOL[prec]
    for k, name in ((2, "u"), (4, "u_A"), (5, "u_Ku")):
        assert rel_l2(wl.from_abi(out[k].cpu().double().numpy()), ref[k]) <= TOL[prec], name
    assert np.max(np.abs(out[3].cpu().numpy() - ref[3])) <= TOL[prec] * np.max(np.abs(ref[3]))
    assert_parity(host(out[6]), ref[6], TOL[prec], "u_hn(0)")
