"""GPU parity of the further local terms (NM_TERM_DMI, NM_TERM_CUBIC, NM_TERM_RKKY, SURVEY.md
8(f) row 3) against oracle/more_terms.py through the C-ABI: term by term, together with every other term on
ragged grids with cell-wise materials and a vacuum block, on each node path (column-marching, separable,
27-point), over Runge-Kutta steps, and (DMI, RKKY) in the adjoint right-hand side.  Wall time: ~8 s."""
import numpy as np
import pytest
import torch

from _sides import assert_parity, dev, host, rel_l2
from paper_2411_11725_b200 import binding as nm
from paper_2411_11725_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-11, "f32": 1e-5}
TD = {"f64": torch.float64, "f32": torch.float32}
ND = {"f64": np.float64, "f32": np.float32}

AXES = np.linalg.qr(np.random.default_rng(77).standard_normal((3, 3)))[0]      # a rotated cubic frame


def _case(n, prec, terms, kind="bulk", normal=2, uniform=False, vacuum=True, seed=0, rkky=None):
    """Seeded inputs (rounded to the build precision), the oracle Problem and the GPU mesh."""
    from oracle import llg
    nd, td = ND[prec], TD[prec]
    rng = np.random.default_rng(1000 + seed + sum(n))
    n = tuple(n)
    dx = (2e-9, 3e-9, 2.5e-9)
    r = lambda a: wl.round_to(a, nd)
    if uniform:
        Ms, A, Ku, D, Kc = 8e5, 1.3e-11, 4e4, 2.5e-3, 3e4
        cells = lambda v: np.full(n, float(np.float64(nd(v)))) if np.isscalar(v) else v
    else:
        Ms = r(rng.uniform(2e5, 8e5, n))
        if vacuum and n[0] >= 4:
            Ms[: n[0] // 3, : max(1, n[1] // 2), :] = 0.0
        A, Ku = r(rng.uniform(0.5e-11, 2e-11, n)), r(rng.uniform(1e4, 5e4, n))
        D, Kc = r(rng.uniform(1e-3, 3e-3, n)), r(rng.uniform(1e4, 5e4, n))
        cells = lambda v: v
    rk_J, rk_planes = rkky if rkky else (0.0, (0, 0))
    if rkky and n[2] > 1:                         # vacuum spacer: the cell layers between the coupled node planes
        Ms = cells(Ms).copy()
        Ms[:, :, rk_planes[0]:rk_planes[1]] = 0.0
    m = wl.box_filter3(wl.random_unit_field(tuple(k + 1 for k in n), 50 + seed))
    m = r(m / np.sqrt((m ** 2).sum(axis=0)))
    axes = AXES                                   # fp64 on both sides (the library casts it to the build precision)
    kax = np.array([1.0, 2.0, 2.0]) / 3.0
    p = llg.Problem(n, dx, cells(Ms), cells(A), cells(Ku), tuple(kax), 2.211e5, 0.05, terms, D=cells(D), dmi_kind=kind,
                    dmi_normal=normal, Kc=cells(Kc), cubic_axes=axes, rkky_J=rk_J, rkky_planes=rk_planes)
    g = lambda v: float(np.float64(nd(v))) if np.isscalar(v) else dev(v, td)
    mesh = nm.Mesh(n, dx, dtype=td, terms=terms, gamma=2.211e5, alpha=0.05, ku_axis=kax, Ms=g(Ms), A=g(A), Ku=g(Ku),
                   D=g(D), Kc=g(Kc), dmi_kind=nm.NM_DMI_BULK if kind == "bulk" else nm.NM_DMI_INTERFACIAL,
                   dmi_normal=normal, cubic_axes=axes, rkky_J=rk_J, rkky_planes=rk_planes)
    return p, mesh, m


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("kind,normal", [("bulk", 2), ("interfacial", 2), ("interfacial", 0)])
def test_dmi_field_alone(kind, normal, prec):
    from oracle import llg
    p, mesh, m = _case((7, 5, 4), prec, nm.NM_TERM_DMI, kind, normal)
    H = host(mesh.nm_heff(0.0, dev(m, TD[prec])))
    assert_parity(H, llg.effective_field(p, m), TOL[prec], "H_dmi %s" % kind)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cubic_field_alone(prec):
    from oracle import llg
    p, mesh, m = _case((6, 5, 3), prec, nm.NM_TERM_CUBIC)
    H = host(mesh.nm_heff(0.0, dev(m, TD[prec])))
    ref = llg.effective_field(p, m)
    assert_parity(H, ref, TOL[prec], "H_cubic")
    vac = np.asarray(p.L) == 0
    assert vac.any() and np.all(H[:, vac] == 0)                # reading C3(iii)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [(9, 6, 5), (1, 1, 1), (12, 1, 3), (5, 35, 6)])
def test_all_terms_ragged_cellwise(n, prec):
    """Exchange + demag + uniaxial + Zeeman + DMI + cubic with cell-wise materials (27-point node kernel)."""
    from oracle import llg
    terms = 63
    p, mesh, m = _case(n, prec, terms, "interfacial", 2, seed=3)
    hu = (1e4, -2e4, 3e4)
    z = nm.Zeeman(h_uniform=hu)
    H = host(mesh.nm_heff(0.0, dev(m, TD[prec]), z))
    assert_parity(H, llg.effective_field(p, m, np.array(hu)), TOL[prec], "H all terms")
    f = host(mesh.nm_llg_rhs(0.0, dev(m, TD[prec]), z))
    assert_parity(f, llg.llg_rhs(p, 0.0, m, lambda t: np.array(hu)), TOL[prec], "f all terms")


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,path", [((128, 6, 5), None), ((24, 10, 7), None), ((24, 10, 7), "generic")])
def test_uniform_materials_each_node_path(n, path, prec, monkeypatch):
    """Uniform A, Ku: the field of the new terms is added by the column-marching kernel (n1 >= 96), the
    separable kernel and the 27-point kernel alike; with a nodal Zeeman array on top (smoothed field +
    new terms share the added array)."""
    from oracle import llg
    if path:
        monkeypatch.setenv("NM_NODE_PATH", path)
    terms = 1 | 2 | 8 | 16 | 32
    p, mesh, m = _case(n, prec, terms, "bulk", uniform=True, seed=5)
    rng = np.random.default_rng(9)
    hs = wl.round_to(rng.standard_normal(m.shape) * 2e4, ND[prec])
    z = nm.Zeeman(h_uniform=(0.0, 1e4, 0.0), h_static=dev(hs, TD[prec]))
    href = hs + np.array([0.0, 1e4, 0.0]).reshape(3, 1, 1, 1)
    H = host(mesh.nm_heff(0.0, dev(m, TD[prec]), z))
    assert_parity(H, llg.effective_field(p, m, href), TOL[prec], "H uniform materials")
    H2 = host(mesh.nm_heff(0.0, dev(m, TD[prec]), nm.Zeeman(h_uniform=(0.0, 1e4, 0.0))))
    assert_parity(H2, llg.effective_field(p, m, np.array([0.0, 1e4, 0.0])), TOL[prec], "H uniform Zeeman")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_runge_kutta_steps_with_the_new_terms(prec):
    """Five RK4 steps and one Dormand-Prince step with DMI + cubic on (graph replay included: the extra
    kernel is part of the captured sequence)."""
    from oracle import llg
    terms = 1 | 2 | 16 | 32
    p, mesh, m = _case((10, 6, 4), prec, terms, "interfacial", 2, seed=7)
    y, ref = dev(m, TD[prec]), m.copy()
    dt = 2e-14
    for s in range(5):
        mesh.nm_rk_step(nm.NM_RK4, s * dt, dt, y)
        ref = llg.rk4_step(p, s * dt, dt, ref)
    assert_parity(host(y), ref, TOL[prec], "RK4 trajectory")
    y2 = dev(m, TD[prec])
    err = mesh.nm_rk_step(nm.NM_DOPRI5, 0.0, 5e-14, y2, rtol=1e-5, atol=1e-5, want_err=True)
    ref2, err_ref, _ = llg.dopri5_step(p, 0.0, 5e-14, m, rtol=1e-5, atol=1e-5)
    assert rel_l2(host(y2), ref2) <= TOL[prec]
    assert abs(err - err_ref) <= (2e-2 if prec == "f32" else 1e-8) * err_ref + (1e-4 if prec == "f32" else 0.0)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,kind,uniform", [((9, 6, 5), "interfacial", False), ((128, 6, 5), "bulk", True), ((24, 10, 7), "bulk", True)])
def test_adjoint_rhs_and_backward_step_with_dmi(n, kind, uniform, prec):
    """The DMI term in the adjoint right-hand side (linear in m: it rides in H and in Hlin^T b) on the 27-point,
    the column-marching and the separable node kernels: (f, -(df/dm)^T a, -(df/dMs)^T a) against the oracle,
    then three backward RK4 steps of (m, a, u)."""
    from oracle import adjoint, llg
    terms = 1 | 2 | 4 | 16
    p, mesh, m = _case(n, prec, terms, kind, 2, uniform=uniform, seed=11)
    a = wl.round_to(np.random.default_rng(12).standard_normal(m.shape), ND[prec])
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, TD[prec]), dev(a, TD[prec]))
    assert_parity(host(f), f_ref, TOL[prec], "f")
    assert_parity(host(da), da_ref, TOL[prec], "da/dt")
    assert rel_l2(wl.from_abi(du.cpu().double().numpy()), du_ref) <= TOL[prec]
    dt = 2e-14
    mT = m.copy()
    for s in range(3):
        mT = llg.rk4_step(p, s * dt, dt, mT)
    ref = adjoint.backward_rk4(p, mT, a, dt, 3)
    mm, aa = dev(mT, TD[prec]), dev(a, TD[prec])
    uu = torch.zeros(mesh.cell_shape_abi, dtype=TD[prec], device=mm.device)
    for s in range(3, 0, -1):
        mesh.nm_adjoint_rk4_step(s * dt, dt, mm, aa, uu)
    assert rel_l2(host(aa), ref[1]) <= TOL[prec]
    assert rel_l2(wl.from_abi(uu.cpu().double().numpy()), ref[2]) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,uniform,terms", [((9, 6, 5), False, 1 | 2 | 4 | 16 | 32), ((128, 6, 5), True, 1 | 2 | 32),
                                             ((7, 5, 4), False, 32)])
def test_adjoint_rhs_and_backward_step_with_cubic_anisotropy(n, uniform, terms, prec):
    """The cubic term is not linear in m: pass 2 of the adjoint right-hand side applies the Hessian of its energy at
    m to q = b / (S Ms) (oracle more_terms.hessvec_cubic).  (f, -(df/dm)^T a, -(df/dMs)^T a) against the oracle,
    then three backward RK4 steps of (m, a, u)."""
    from oracle import adjoint, llg
    p, mesh, m = _case(n, prec, terms, "bulk", uniform=uniform, seed=21)
    a = wl.round_to(np.random.default_rng(22).standard_normal(m.shape), ND[prec])
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, TD[prec]), dev(a, TD[prec]))
    assert_parity(host(f), f_ref, TOL[prec], "f")
    assert_parity(host(da), da_ref, TOL[prec], "da/dt with cubic")
    assert rel_l2(wl.from_abi(du.cpu().double().numpy()), du_ref) <= TOL[prec]
    dt = 2e-14
    mT = m.copy()
    for s in range(3):
        mT = llg.rk4_step(p, s * dt, dt, mT)
    ref = adjoint.backward_rk4(p, mT, a, dt, 3)
    mm, aa = dev(mT, TD[prec]), dev(a, TD[prec])
    uu = torch.zeros(mesh.cell_shape_abi, dtype=TD[prec], device=mm.device)
    for s in range(3, 0, -1):
        mesh.nm_adjoint_rk4_step(s * dt, dt, mm, aa, uu)
    assert rel_l2(host(aa), ref[1]) <= TOL[prec]
    assert rel_l2(wl.from_abi(uu.cpu().double().numpy()), ref[2]) <= TOL[prec]


def test_further_terms_on_a_reduced_basis_and_a_skewed_frame_are_refused():
    with pytest.raises(nm.NmError) as e:
        nm.Mesh((8, 8, 1), (2e-9,) * 3, dtype=torch.float64, terms=1 | 32, Ms=8e5, A=1.3e-11, Kc=1e4, basis=2)
    assert e.value.status == nm.NM_EUNSUPPORTED
    with pytest.raises(nm.NmError) as e:
        nm.Mesh((4, 4, 4), (2e-9,) * 3, dtype=torch.float64, terms=32, Ms=8e5, Kc=1e4, cubic_axes=(1, 0, 0, 0, 1, 0, 0, 1, 0))
    assert e.value.status == nm.NM_EINVAL


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,planes,uniform", [((9, 6, 5), (2, 3), False), ((128, 6, 5), (1, 4), True), ((5, 4, 1), (0, 1), False)])
def test_rkky_interlayer_coupling(n, planes, uniform, prec):
    """NM_TERM_RKKY against oracle variation_rkky: two layers across a vacuum spacer (the cell layers
    between the coupled node planes have Ms = 0; the one-layer film couples its two faces), alone and with
    exchange + demag + DMI, then the adjoint right-hand side (the term is linear in m: it rides in H and in
    Hlin^T b)."""
    from oracle import adjoint, llg
    J = -1.2e-3                                           # antiferromagnetic coupling
    for terms in (64, 1 | 2 | 16 | 64):
        p, mesh, m = _case(n, prec, terms, "bulk", uniform=uniform, vacuum=False, seed=13, rkky=(J, planes))
        H = host(mesh.nm_heff(0.0, dev(m, TD[prec])))
        ref = llg.effective_field(p, m)
        assert_parity(H, ref, TOL[prec], "H with RKKY, terms %d" % terms)
        if terms == 64:
            other = [k for k in range(n[2] + 1) if k not in planes]
            assert np.all(H[:, :, :, other] == 0) and np.abs(H).max() > 0
    a = wl.round_to(np.random.default_rng(14).standard_normal(m.shape), ND[prec])
    f_ref, da_ref, du_ref = adjoint.adjoint_rhs(p, 0.0, m, a)
    f, da, du = mesh.nm_llg_adjoint_rhs(0.0, dev(m, TD[prec]), dev(a, TD[prec]))
    assert_parity(host(da), da_ref, TOL[prec], "da/dt with RKKY")
    assert rel_l2(wl.from_abi(du.cpu().double().numpy()), du_ref) <= TOL[prec]
