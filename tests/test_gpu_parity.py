"""GPU parity: libnm.so (through the C-ABI binding) against the fp64 CPU oracle, element by element
on the same seeded inputs.  Tolerances are north_star's: relative L2 <= 1e-5 (fp32), 1e-11 (fp64).
"""
import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import (assert_parity, dev, gpu_mesh, gpu_zeeman, host, np_dtype, oracle_problem, oracle_zeeman,
                    rel_l2)

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


def _m0(w, td):
    return wl.round_to(w.m0, np_dtype(td))


# ---- demag tensor (reading C4): library setup vs the oracle's __float128 closed form -------------
@pytest.mark.parametrize("n,dx", [((12, 8, 6), (2e-9, 3e-9, 2.5e-9)),
                                  ((32, 8, 1), (3.125e-9, 3.125e-9, 3e-9)),
                                  ((48, 48, 48), (2e-9, 2e-9, 2e-9)),
                                  ((1, 1, 1), (1e-9, 2e-9, 0.5e-9)),
                                  ((64, 2, 1), (1e-9, 4e-9, 8e-9))])
def test_tensor_matches_oracle(n, dx):
    from oracle import demag
    from paper_2411_11725_b200 import binding as nm
    mesh = nm.Mesh(n, dx, dtype=torch.float64, terms=wl.TERM_DEMAG, Ms=1.0, A=0.0, Ku=0.0)
    got = mesh.nm_debug_get_tensor()            # [6][N3][N2][N1]
    ref = wl.to_abi(demag.demag_tensor(n, dx))  # oracle [6][N1][N2][N3] -> ABI order
    assert got.shape == ref.shape
    assert np.max(np.abs(got - ref)) <= 1e-13


# ---- H_eff ---------------------------------------------------------------------------------------
def _heff_case(w, prec, h_static=None):
    td = DT[prec]
    nd = np_dtype(td)
    p = oracle_problem(w, nd)
    m = _m0(w, td)
    z = oracle_zeeman(w, nd, h_static)
    from oracle import llg
    ref = llg.effective_field(p, m, z(0.0) if z else None)
    mesh = gpu_mesh(w, td)
    got = host(mesh.nm_heff(0.0, dev(m, td), gpu_zeeman(w, td, h_static=h_static)))
    return got, ref, mesh, p, m


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_heff_config1_tiny_film(prec):
    got, ref, *_ = _heff_case(wl.config1_tiny_film(), prec)
    assert_parity(got, ref, TOL[prec])


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_heff_config2_cube64(prec):
    got, ref, *_ = _heff_case(wl.config2_cube(64), prec)
    assert_parity(got, ref, TOL[prec])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(24, 12, 6), (6, 18, 48), (16, 1, 1), (1, 16, 4), (1, 1, 1),
                               (2, 2, 2), (96, 4, 3), (9, 27, 2)])
def test_heff_ragged_all_terms(n, prec):
    w, hs = wl.varied_case(n, vacuum=(n[0] >= 6))
    got, ref, *_ = _heff_case(w, prec, hs)
    assert_parity(got, ref, TOL[prec])
    # vacuum nodes (S Ms = 0) get exactly H = 0 (reading C3(iii))
    from oracle.mesh import scatter_cells_to_nodes
    vac = scatter_cells_to_nodes(w.cell_array(w.Ms)) == 0
    assert np.all(got[:, vac] == 0)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(16, 32, 64), (64, 16, 32), (32, 64, 16), (128, 16, 16), (16, 128, 32),
                               (32, 16, 128), (256, 16, 16), (16, 256, 16), (32, 32, 256)])
def test_heff_fast_path_sizes(n, prec):
    """Grids of the register-FFT fast path (every N_d = 16 M_d), all terms, cell-wise materials."""
    w, hs = wl.varied_case(n, vacuum=True)
    got, ref, mesh, *_ = _heff_case(w, prec, hs)
    assert_parity(got, ref, TOL[prec])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(20, 10, 5), (14, 7, 1), (5, 35, 6), (40, 24, 1), (50, 1, 1), (7, 7, 7),
                               (10, 28, 45)])
def test_heff_radix_5_7_sizes(n, prec, monkeypatch):
    """N_d with factors 5 and 7 (general path: radix-5 / 7 stages by the DFT sum in the x, y and z
    passes, mixed with the radix-8/4/3/2 stages); all terms, cell-wise materials, vacuum block."""
    monkeypatch.setenv("NM_DEMAG_PATH", "generic")      # not the zero-extended fast path
    w, hs = wl.varied_case(n, vacuum=(n[0] >= 6))
    got, ref, mesh, *_ = _heff_case(w, prec, hs)
    assert mesh.nm_debug_demag_path() == 0
    assert_parity(got, ref, TOL[prec])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(36, 128, 112), (68, 96, 100), (52, 64, 40), (100, 32, 24)])
def test_heff_embedded_fast_path_sizes(n, prec):
    """Grids the fast path serves on the zero-extended mesh (some N_d below the next 16 * 2^k, not
    necessarily 2^a 3^b), non-pipelined y / z kernels, both precisions; all terms, cell-wise
    materials, vacuum block."""
    w, hs = wl.varied_case(n, vacuum=True)
    got, ref, mesh, *_ = _heff_case(w, prec, hs)
    assert mesh.nm_debug_demag_path() == 2
    assert_parity(got, ref, TOL[prec])


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_heff_term_by_term(prec):
    """Each term alone against the oracle's part (a dropped or mis-signed term cannot hide)."""
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    base, hs = wl.varied_case((12, 6, 4))
    for term in (wl.TERM_EXCHANGE, wl.TERM_DEMAG, wl.TERM_ANISO, wl.TERM_ZEEMAN):
        w, _ = wl.varied_case((12, 6, 4))
        w.terms = term
        p = oracle_problem(w, nd)
        m = _m0(w, td)
        z = oracle_zeeman(w, nd, hs)
        ref = llg.effective_field(p, m, z(0.0) if z else None)
        got = host(gpu_mesh(w, td).nm_heff(0.0, dev(m, td), gpu_zeeman(w, td, h_static=hs)))
        assert_parity(got, ref, TOL[prec], 'term %d' % term)


def test_cell_demag_field_matches_direct_sum():
    """Cell field from the FFT passes vs the oracle's brute-force O(N^2) sum (no FFT on that side)."""
    from oracle import demag
    w, _ = wl.varied_case((6, 4, 3))
    w.terms = wl.TERM_DEMAG
    td = torch.float64
    p = oracle_problem(w)
    m = _m0(w, td)
    mesh = gpu_mesh(w, td)
    mesh.nm_heff(0.0, dev(m, td))
    got = host(mesh.nm_debug_get_cell_field())
    ref = demag.demag_field_cells_direct(demag.cell_magnetization(m, p.Ms), p.Nt)
    assert rel_l2(got, ref) <= 1e-12


# ---- LLG right-hand side and Runge-Kutta ---------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_llg_rhs(prec):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((12, 6, 4), vacuum=True)
    p = oracle_problem(w, nd)
    m = _m0(w, td)
    ref = llg.llg_rhs(p, 0.0, m, oracle_zeeman(w, nd, hs))
    got = host(gpu_mesh(w, td).nm_llg_rhs(0.0, dev(m, td), gpu_zeeman(w, td, h_static=hs)))
    assert_parity(got, ref, TOL[prec])


def test_rk4_trajectory_config1_fp64():
    """Config 1: 200 fixed RK4 steps of 1e-13 s in fp64, whole trajectory end state."""
    from oracle import llg
    w = wl.config1_tiny_film()
    td = torch.float64
    p = oracle_problem(w)
    m = _m0(w, td)
    mesh = gpu_mesh(w, td)
    y = dev(m, td)
    ref = m.copy()
    worst = 0.0
    for s in range(w.n_steps):
        ref = llg.rk4_step(p, s * w.dt, w.dt, ref)
        mesh.nm_rk_step(0, s * w.dt, w.dt, y)
        if s % 50 == 49:
            worst = max(worst, rel_l2(host(y), ref))
    assert worst <= 1e-11
    assert np.max(np.abs(np.sqrt(np.sum(host(y) ** 2, axis=0)) - 1.0)) < 1e-14


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_rk4_steps_all_terms(prec):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((12, 6, 4))
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd, hs)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td, h_static=hs)
    ref = _m0(w, td)
    y = dev(ref, td)
    for s in range(5):
        ref = llg.rk4_step(p, s * w.dt, w.dt, ref, z)
        mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
    assert rel_l2(host(y), ref) <= TOL[prec]
    # without renormalisation
    ref2 = llg.rk4_step(p, 0.0, w.dt, _m0(w, td), z, renormalise=False)
    y2 = dev(_m0(w, td), td)
    mesh.nm_rk_step(0, 0.0, w.dt, y2, gz, renormalise=False)
    assert rel_l2(host(y2), ref2) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_dopri5_step_accept_and_reject(prec):
    from oracle import llg
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((12, 6, 4))
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd, hs)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td, h_static=hs)
    m = _m0(w, td)
    for dt, expect in ((2e-14, True), (1e-13, True), (2e-13, False)):
        ref, err_ref, acc = llg.dopri5_step(p, 0.0, dt, m, z, rtol=1e-5, atol=1e-5)
        assert acc == expect
        y = dev(m, td)
        err = mesh.nm_rk_step(1, 0.0, dt, y, gz, rtol=1e-5, atol=1e-5, want_err=True)
        # fp32: the embedded error is a cancelling sum of stage derivatives, so its rounding floor
        # (~1e-5 of the scaled norm) is absolute, not relative
        assert abs(err - err_ref) <= (1e-8 * err_ref if prec == "f64" else 2e-2 * err_ref + 1e-4)
        assert rel_l2(host(y), ref) <= TOL[prec]
        if not expect:
            assert np.array_equal(host(y), m)      # rejected step leaves m untouched


def test_dopri5_replay_config3_small_fp32():
    """Config 3's recipe on a 64x64x1 film: the GPU runs the adaptive controller in fp32, the
    oracle replays the GPU's accepted/rejected dt sequence in fp64."""
    from oracle import llg
    from paper_2411_11725_b200 import drivers
    w = wl.config3_thin_film(64)
    td = torch.float32
    p = oracle_problem(w, np.float32)
    z = oracle_zeeman(w, np.float32)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    ref = _m0(w, td)
    y = dev(ref, td)
    t, dt = 0.0, 1e-13
    accepted = 0
    for _ in range(60):
        err = mesh.nm_rk_step(1, t, dt, y, gz, rtol=1e-5, atol=1e-5, want_err=True)
        out, err_ref, acc = llg.dopri5_step(p, t, dt, ref, z, rtol=1e-5, atol=1e-5)
        if err <= 1.0:
            assert acc or abs(err_ref - 1.0) < 1e-2
            ref = out if acc else ref
            t += dt
            accepted += 1
        dt = drivers.dopri5_next_dt(dt, err)
        if accepted >= 25:
            break
    assert accepted >= 10
    assert rel_l2(host(y), ref) <= 1e-5


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_vacuum_nodes_with_zero_magnetisation_stay_zero(prec):
    """The usual convention m = (0,0,0) at vacuum nodes (all adjacent cells Ms = 0): H = 0 there
    (reading C3(iii)), and renormalisation leaves a zero vector zero instead of 0 * inf = NaN, which
    the next cell average and the FFT would spread over the whole field.  RK4 steps, a Dormand-Prince
    step and the backward RK4 of (m, a, u), all with renormalise = 1, against the oracle."""
    from oracle import adjoint, llg
    from oracle.mesh import scatter_cells_to_nodes
    from paper_2411_11725_b200 import drivers
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((12, 6, 4), vacuum=True)
    vac = scatter_cells_to_nodes(w.cell_array(w.Ms)) == 0
    assert vac.any()
    m0 = _m0(w, td)
    m0[:, vac] = 0.0
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd, hs)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td, h_static=hs)
    ref = m0.copy()
    y = dev(m0, td)
    for s in range(4):
        ref = llg.rk4_step(p, s * w.dt, w.dt, ref, z)
        mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
    got = host(y)
    assert np.all(np.isfinite(got)) and np.all(got[:, vac] == 0) and np.all(ref[:, vac] == 0)
    assert_parity(got, ref, TOL[prec])
    ref5, err_ref, acc = llg.dopri5_step(p, 0.0, 5e-14, ref, z, rtol=1e-5, atol=1e-5)
    err = mesh.nm_rk_step(1, 0.0, 5e-14, y, gz, rtol=1e-5, atol=1e-5, want_err=True)
    assert acc and err <= 1.0 and np.isfinite(err)
    got = host(y)
    assert np.all(np.isfinite(got)) and np.all(got[:, vac] == 0)
    assert rel_l2(got, ref5) <= TOL[prec]
    # backward pass of (m, a, u) over 4 steps from m0
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, 4, z, checkpoint_every=2)
    aT = wl.round_to(np.random.default_rng(5).standard_normal(m0.shape), nd)
    _, a0_ref, u0_ref = adjoint.backward_rk4(p, mT_ref, aT, w.dt, 4, z, checkpoints=ck)
    g = dev(aT, td)
    mT, a0, u0 = drivers.adjoint_gradient(mesh, dev(m0, td), lambda m_: g, w.dt, 4, gz, checkpoint_every=2)
    assert bool(torch.isfinite(a0).all()) and bool(torch.isfinite(u0).all())
    assert rel_l2(host(mT), mT_ref) <= TOL[prec]
    assert rel_l2(host(a0), a0_ref) <= TOL[prec]
    assert rel_l2(wl.from_abi(u0.cpu().double().numpy()), u0_ref) <= (1e-11 if prec == "f64" else TOL[prec])


# ---- adjoint -------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("nodal_zeeman", [False, True])
def test_adjoint_rhs(prec, nodal_zeeman):
    from oracle import adjoint
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((12, 6, 4))
    if not nodal_zeeman:
        hs = None
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd, hs)
    m = _m0(w, td)
    a = wl.round_to(np.random.default_rng(77).standard_normal(m.shape), nd)
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a, z)
    mesh = gpu_mesh(w, td)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, td), dev(a, td), gpu_zeeman(w, td, h_static=hs))
    assert rel_l2(host(f), f_ref) <= TOL[prec]
    assert rel_l2(host(da), da_ref) <= TOL[prec]
    assert rel_l2(wl.from_abi(du.cpu().double().numpy()), du_ref) <= TOL[prec]


def test_adjoint_rk4_backward_small_config5_fp64():
    """Config 5's recipe on a 32x8x1 film, 40 steps, checkpoints every 10: u(0) = dJ/dMs."""
    from oracle import adjoint
    w = wl.config5_inverse((32, 8, 1), n_steps=40)
    td = torch.float64
    p = oracle_problem(w)
    z = oracle_zeeman(w)
    gz = gpu_zeeman(w, td)
    m0 = _m0(w, td)
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=10)
    aT = wl.objective_weights(w)
    _, a0_ref, u0_ref = adjoint.backward_rk4(p, mT_ref, aT, w.dt, w.n_steps, z, checkpoints=ck)

    mesh = gpu_mesh(w, td)
    y = dev(m0, td)
    gck = {}
    for s in range(w.n_steps):
        if s % 10 == 0:
            gck[s] = y.clone()
        mesh.nm_rk_step(0, s * w.dt, w.dt, y, gz)
    assert rel_l2(host(y), mT_ref) <= 1e-11
    a = dev(aT, td)
    u = torch.zeros(mesh.cell_shape_abi, dtype=td, device="cuda:0")
    for s in range(w.n_steps, 0, -1):
        mesh.nm_adjoint_rk4_step(s * w.dt, w.dt, y, a, u, gz)
        if (s - 1) in gck:
            y.copy_(gck[s - 1])
    assert rel_l2(host(a), a0_ref) <= 1e-11
    assert rel_l2(wl.from_abi(u.cpu().numpy()), u0_ref) <= 1e-11


def test_adjoint_gradient_driver_vs_finite_differences_config5_small_fp64():
    """Config 5's check on a 32x8x1 film, 40 steps: dJ/dMs from drivers.adjoint_gradient against
    central finite differences of J (GPU forward solves with Ms_c +- h) on 8 seeded cells
    (C8: <= 1e-3 relative; the adjoint-state gradient is the continuous problem's)."""
    from paper_2411_11725_b200 import drivers
    w = wl.config5_inverse((32, 8, 1), n_steps=40)
    td = torch.float64
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    m0 = dev(_m0(w, td), td)
    g = dev(wl.objective_weights(w), td)
    _, _, u0 = drivers.adjoint_gradient(mesh, m0, lambda mT: g, w.dt, w.n_steps, gz, checkpoint_every=10)
    grad = wl.from_abi(u0.cpu().numpy())

    def J(Ms):
        mesh.nm_mesh_set_Ms(dev(Ms, td))
        y = m0.clone()
        drivers.forward_rk4(mesh, y, w.dt, w.n_steps, gz)
        return float((g * y).sum())

    for c in wl.fd_cells(w, 8, 6):
        h = 1e-4 * w.Ms[c]
        Mp, Mm = w.Ms.copy(), w.Ms.copy()
        Mp[c] += h
        Mm[c] -= h
        fd = (J(Mp) - J(Mm)) / (2 * h)
        assert abs(grad[c] - fd) <= 1e-3 * abs(fd), (c, grad[c], fd)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_adjoint_gradient_objectives_at_several_times(prec):
    """L = w1 . m(T1) + w2 . m(T2) + wT . m(T) on a 32x8x1 film (config 5's recipe, 36
    steps, checkpoints every 12): drivers.adjoint_gradient with objectives_at (the jumps go through
    nm_adjoint_add_objective) against the oracle's backward pass with the same jumps."""
    from oracle import adjoint
    from paper_2411_11725_b200 import drivers
    td = DT[prec]
    nd = np_dtype(td)
    w = wl.config5_inverse((32, 8, 1), n_steps=36)
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd)
    m0 = _m0(w, td)
    rng = np.random.default_rng(23)
    w1, w2 = (wl.round_to(rng.standard_normal(m0.shape), nd) for _ in range(2))
    wT = wl.round_to(wl.objective_weights(w), nd)
    s1, s2 = 10, 24
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=12)
    _, a0_ref, u0_ref = adjoint.backward_rk4(p, mT_ref, wT, w.dt, w.n_steps, z, checkpoints=ck,
                                             a_jumps={s1: w1, s2: w2})
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    g1, g2, gT = dev(w1, td), dev(w2, td), dev(wT, td)
    mT, a0, u0 = drivers.adjoint_gradient(mesh, dev(m0, td), lambda m: gT, w.dt, w.n_steps, gz,
                                          checkpoint_every=12,
                                          objectives_at={s1: lambda m: g1, s2: lambda m: g2})
    assert rel_l2(host(mT), mT_ref) <= TOL[prec]
    assert rel_l2(host(a0), a0_ref) <= TOL[prec]
    assert rel_l2(wl.from_abi(u0.cpu().double().numpy()), u0_ref) <= TOL[prec]
    # the jump itself: a <- a + scale g, and overlapping arguments are refused
    from paper_2411_11725_b200 import binding as nm
    a = g1.clone()
    mesh.nm_adjoint_add_objective(a, g2, scale=-0.5)
    assert torch.equal(a, g1 + (-0.5) * g2)
    with pytest.raises(nm.NmError) as e:
        mesh.nm_adjoint_add_objective(a, a)
    assert e.value.status == nm.NM_EINVAL


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_hext_gradient_rhs_and_backward_pass(prec):
    """Gradient with respect to a uniform external field: nm_llg_adjoint_rhs_hext
    against oracle adjoint_rhs_hext on a ragged all-terms mesh with a vacuum block (several reduction
    blocks), and u_h(0) of drivers.adjoint_gradient(with_hext=True) against the oracle's backward pass
    on a film with anisotropy and a uniform field."""
    from oracle import adjoint
    from paper_2411_11725_b200 import drivers
    td = DT[prec]
    nd = np_dtype(td)
    # (1) single right-hand side
    w, hs = wl.varied_case((24, 12, 6), vacuum=True)
    p = oracle_problem(w, nd)
    m = _m0(w, td)
    a = wl.round_to(np.random.default_rng(31).standard_normal(m.shape), nd)
    ref = adjoint.adjoint_rhs_hext(p, 0.0, m, a)
    mesh = gpu_mesh(w, td)
    got = mesh.nm_llg_adjoint_rhs_hext(dev(m, td), dev(a, td)).cpu().numpy()
    # a sum of nodes of mixed sign: error relative to the sum of magnitudes, not to the result
    scale = p.gamma * np.sum(np.abs(a))
    assert np.max(np.abs(got - ref)) <= (1e-13 if prec == "f64" else 1e-6) * scale
    assert np.max(np.abs(got - ref)) <= (1e-11 if prec == "f64" else 1e-4) * np.max(np.abs(ref))
    # a mesh without the Zeeman term does not depend on h
    w0 = wl.config4_sweep(16)
    assert torch.all(gpu_mesh(w0, td).nm_llg_adjoint_rhs_hext(dev(_m0(w0, td), td), dev(_m0(w0, td), td)) == 0)
    # (2) backward integration
    w = wl.config5_inverse((32, 8, 1), n_steps=30)
    w.terms = wl.TERM_EXCHANGE | wl.TERM_DEMAG | wl.TERM_ANISO | wl.TERM_ZEEMAN
    w.Ku = 2e4
    w.ku_axis = (0.0, 0.6, 0.8)
    w.h_uniform = (1e3, 2e3, -1.5e3)
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd)
    m0 = _m0(w, td)
    wT = wl.round_to(wl.objective_weights(w), nd)
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=10)
    _, a0_ref, u0_ref, uh_ref = adjoint.backward_rk4(p, mT_ref, wT, w.dt, w.n_steps, z, checkpoints=ck,
                                                     with_hext=True)
    assert np.max(np.abs(uh_ref)) > 0
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    gT = dev(wT, td)
    out = {}
    for graph in ("0", "1"):
        import os
        old = os.environ.get("NM_GRAPH")
        os.environ["NM_GRAPH"] = graph
        try:
            mesh = gpu_mesh(w, td)
        finally:
            if old is None:
                os.environ.pop("NM_GRAPH", None)
            else:
                os.environ["NM_GRAPH"] = old
        mT, a0, u0, uh = drivers.adjoint_gradient(mesh, dev(m0, td), lambda m_: gT, w.dt, w.n_steps, gz,
                                                  checkpoint_every=10, with_hext=True)
        out[graph] = (a0.clone(), u0.clone(), uh.clone())
        assert rel_l2(host(a0), a0_ref) <= TOL[prec]
        assert rel_l2(wl.from_abi(u0.cpu().double().numpy()), u0_ref) <= TOL[prec]
        assert rel_l2(uh.cpu().numpy(), uh_ref) <= TOL[prec]
    for x, y in zip(out["0"], out["1"]):                # replayed steps accumulate u_h identically
        assert torch.equal(x, y)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_materials_gradient_rhs_and_backward_pass(prec):
    """VJPs with respect to the cell-wise A and Ku: nm_llg_adjoint_rhs_materials against the oracle on a
    ragged all-terms mesh with a vacuum block, zero for terms a mesh does not have, and (u_A, u_Ku, u_h)
    of drivers.adjoint_gradient(with_materials=True) against the oracle's backward pass."""
    from oracle import adjoint
    from paper_2411_11725_b200 import drivers
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((24, 12, 6), vacuum=True)
    p = oracle_problem(w, nd)
    m = _m0(w, td)
    a = wl.round_to(np.random.default_rng(41).standard_normal(m.shape), nd)
    gA_ref, gKu_ref = adjoint.adjoint_rhs_materials(p, 0.0, m, a)
    mesh = gpu_mesh(w, td)
    gA, gKu = mesh.nm_llg_adjoint_rhs_materials(dev(m, td), dev(a, td))
    tol = TOL[prec]
    assert rel_l2(wl.from_abi(gA.cpu().double().numpy()), gA_ref) <= tol
    assert rel_l2(wl.from_abi(gKu.cpu().double().numpy()), gKu_ref) <= tol
    only_A, none_Ku = mesh.nm_llg_adjoint_rhs_materials(dev(m, td), dev(a, td), want_Ku=False)
    assert none_Ku is None and torch.equal(only_A, gA)
    w0 = wl.config4_sweep(16)                             # exchange + demag: nothing depends on Ku
    m0_ = dev(_m0(w0, td), td)
    gA0, gKu0 = gpu_mesh(w0, td).nm_llg_adjoint_rhs_materials(m0_, m0_.flip(0).contiguous())
    assert torch.all(gKu0 == 0) and float(gA0.abs().max()) > 0
    # backward integration: film with cell-wise A and Ku
    w = wl.config5_inverse((32, 8, 1), n_steps=30)
    rng = np.random.default_rng(43)
    w.terms = wl.TERM_EXCHANGE | wl.TERM_DEMAG | wl.TERM_ANISO | wl.TERM_ZEEMAN
    w.A = rng.uniform(3e-12, 4e-12, size=w.n_cells)
    w.Ku = rng.uniform(1e4, 3e4, size=w.n_cells)
    w.ku_axis = (0.0, 0.6, 0.8)
    w.h_uniform = (1e3, 2e3, -1.5e3)
    p = oracle_problem(w, nd)
    z = oracle_zeeman(w, nd)
    m0 = _m0(w, td)
    wT = wl.round_to(wl.objective_weights(w), nd)
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=10)
    ref = adjoint.backward_rk4(p, mT_ref, wT, w.dt, w.n_steps, z, checkpoints=ck, with_hext=True,
                               with_materials=True)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td)
    gT = dev(wT, td)
    got = drivers.adjoint_gradient(mesh, dev(m0, td), lambda m_: gT, w.dt, w.n_steps, gz, checkpoint_every=10,
                                   with_hext=True, with_materials=True)
    cell = lambda x: wl.from_abi(x.cpu().double().numpy())
    lo = TOL[prec]
    assert rel_l2(host(got[1]), ref[1]) <= TOL[prec]
    assert rel_l2(cell(got[2]), ref[2]) <= lo
    assert rel_l2(got[3].cpu().numpy(), ref[3]) <= lo
    assert rel_l2(cell(got[4]), ref[4]) <= lo
    assert rel_l2(cell(got[5]), ref[5]) <= lo


def test_field_angle_problem_gradient_and_descent_fp64():
    """Sec. VII (Eqs. 31-33) on a small single-domain particle (8x4x2 cells, exchange +
    anisotropy + external field, Eq. 32): dL/dtheta, dL/dphi from one forward and one backward solve
    against central differences of GPU forward solves, and a few gradient-descent steps lower the
    objective L = mean_n |m_n(T) - m_target| (Eq. 33 with equal nodal weights)."""
    from paper_2411_11725_b200 import binding as nm, drivers
    td = torch.float64
    mesh = nm.Mesh((8, 4, 2), (3e-9, 3e-9, 3e-9), dtype=td, terms=wl.TERM_EXCHANGE | wl.TERM_ANISO | wl.TERM_ZEEMAN,
                   gamma=2.211e5, alpha=0.5, ku_axis=(0.0, 0.0, 1.0), Ms=8e5, A=1.3e-11, Ku=1e5)
    rng = np.random.default_rng(51)
    v = 0.05 * rng.standard_normal(mesh.node_shape_abi)
    v[0] += 1.0
    m0 = torch.from_numpy(v / np.sqrt(np.sum(v * v, axis=0))).to("cuda:0")
    target = torch.zeros_like(m0)
    target[1] = 1.0
    nn = m0[0].numel()

    def loss(mT):
        return float(torch.sqrt(((mT - target) ** 2).sum(0)).sum() / nn)

    def loss_grad(mT):
        d = mT - target
        return d / torch.sqrt((d ** 2).sum(0)) / nn

    Hc, th, ph, dt, nst = 2e5, 1.2, 0.4, 1e-13, 60

    def L_of(a, b):
        y = m0.clone()
        drivers.forward_rk4(mesh, y, dt, nst, nm.Zeeman(h_uniform=drivers.field_from_angles(Hc, a, b)))
        return loss(y)

    mT, dth, dph = drivers.field_angle_gradient(mesh, m0, loss_grad, Hc, th, ph, dt, nst, checkpoint_every=20)
    assert abs(loss(mT) - L_of(th, ph)) < 1e-14
    e = 1e-4
    fd_th = (L_of(th + e, ph) - L_of(th - e, ph)) / (2 * e)
    fd_ph = (L_of(th, ph + e) - L_of(th, ph - e)) / (2 * e)
    scale = max(abs(fd_th), abs(fd_ph))
    assert scale > 1e-3
    assert abs(dth - fd_th) < 2e-3 * scale and abs(dph - fd_ph) < 2e-3 * scale
    th1, ph1, hist = drivers.optimise_field_angles(mesh, m0, loss, loss_grad, Hc, th, ph, dt, nst,
                                                   rate=0.5, iterations=6, checkpoint_every=20)
    assert L_of(th1, ph1) < hist[0] - 1e-3
    assert all(b <= a + 1e-12 for a, b in zip(hist, hist[1:]))


# ---- boundary behaviour --------------------------------------------------------------------------
def test_errors_are_statuses_not_crashes():
    from paper_2411_11725_b200 import binding as nm
    with pytest.raises(nm.NmError) as e:
        nm.Mesh((11, 4, 4), (1e-9,) * 3, terms=wl.TERM_DEMAG, Ms=1.0, A=0.0, Ku=0.0)
    assert e.value.status == nm.NM_EUNSUPPORTED
    with pytest.raises(nm.NmError) as e:
        nm.Mesh((0, 4, 4), (1e-9,) * 3, terms=1, Ms=1.0, A=1.0, Ku=0.0)
    assert e.value.status == nm.NM_EINVAL
    # exchange-only meshes accept any size
    mesh = nm.Mesh((5, 7, 3), (1e-9,) * 3, dtype=torch.float64, terms=1, Ms=8e5, A=1.3e-11, Ku=0.0)
    m = torch.zeros(mesh.node_shape_abi, dtype=torch.float64, device="cuda:0")
    m[0] = 1.0
    assert float(mesh.nm_heff(0.0, m).abs().max()) == 0.0   # uniform m: exchange field vanishes
    assert mesh.nm_launch_count() > 0


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_nodal_hext_gradient_rhs_and_backward_pass(prec):
    """Gradient with respect to a NODAL external field (SURVEY.md 8(f) row 2, H^ext): nm_llg_adjoint_rhs_hnodal
    against oracle adjoint_rhs_hnodal on a ragged all-terms mesh with a vacuum block, its sum over the nodes
    against the uniform-field gradient, and u_hn(0) of drivers.adjoint_gradient(with_hnodal=True) against the
    oracle's backward pass on a film with a nodal static field."""
    from oracle import adjoint
    from paper_2411_11725_b200 import drivers
    td = DT[prec]
    nd = np_dtype(td)
    w, hs = wl.varied_case((24, 12, 6), vacuum=True)
    p = oracle_problem(w, nd)
    m = _m0(w, td)
    a = wl.round_to(np.random.default_rng(31).standard_normal(m.shape), nd)
    ref = adjoint.adjoint_rhs_hnodal(p, 0.0, m, a)
    mesh = gpu_mesh(w, td)
    got = host(mesh.nm_llg_adjoint_rhs_hnodal(dev(m, td), dev(a, td)))
    assert_parity(got, ref, TOL[prec], "nodal-field gradient")
    vac = p.L == 0
    assert vac.any()
    uni = mesh.nm_llg_adjoint_rhs_hext(dev(m, td), dev(a, td)).cpu().numpy()
    assert np.max(np.abs(got.sum(axis=(1, 2, 3)) - uni)) <= (1e-10 if prec == "f64" else 1e-4) * np.max(np.abs(uni))
    w0 = wl.config4_sweep(16)
    assert torch.all(gpu_mesh(w0, td).nm_llg_adjoint_rhs_hnodal(dev(_m0(w0, td), td), dev(_m0(w0, td), td)) == 0)
    # backward integration with a nodal static field
    w = wl.config5_inverse((32, 8, 1), n_steps=30)
    w.h_uniform = (1e3, 2e3, -1.5e3)
    p = oracle_problem(w, nd)
    hs = wl.round_to(1e3 * np.random.default_rng(8).standard_normal((3,) + w.node_shape), nd)
    z = oracle_zeeman(w, nd, hs)
    m0 = _m0(w, td)
    wT = wl.round_to(wl.objective_weights(w), nd)
    mT_ref, ck = adjoint.forward_rk4(p, m0, w.dt, w.n_steps, z, checkpoint_every=10)
    ref = adjoint.backward_rk4(p, mT_ref, wT, w.dt, w.n_steps, z, checkpoints=ck, with_hnodal=True)
    mesh = gpu_mesh(w, td)
    gz = gpu_zeeman(w, td, h_static=hs)
    gT = dev(wT, td)
    out = drivers.adjoint_gradient(mesh, dev(m0, td), lambda mm: gT, w.dt, w.n_steps, gz, checkpoint_every=10,
                                   with_hnodal=True)
    assert rel_l2(host(out[1]), ref[1]) <= TOL[prec]
    assert rel_l2(wl.from_abi(out[2].cpu().double().numpy()), ref[2]) <= TOL[prec]
    assert_parity(host(out[3]), ref[3], TOL[prec], "u_hn(0)")
