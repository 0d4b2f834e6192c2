"""Pins for oracle/adjoint.py (C7, C8 of SURVEY.md §8(c); Eqs. 27-30)."""
import numpy as np
import pytest

from oracle import adjoint, llg, mesh
import dataclasses

from oracle.llg import Problem, TERM_EXCHANGE, TERM_DEMAG, TERM_ANISO, TERM_ZEEMAN, TERM_DMI, TERM_CUBIC, TERM_RKKY

ALL = TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO | TERM_ZEEMAN


def rand_unit(shape, seed):
    v = np.random.default_rng(seed).standard_normal((3,) + tuple(shape))
    return v / np.sqrt(np.sum(v * v, axis=0))


def make(n=(3, 2, 2), alpha=0.1, terms=ALL, seed=0):
    rng = np.random.default_rng(seed)
    dx = (3e-9, 2.5e-9, 3.5e-9)
    p = Problem(n, dx, rng.uniform(4e5, 8e5, n), rng.uniform(0.8e-11, 1.3e-11, n),
                rng.uniform(1e5, 5e5, n), ku_axis=(0.0, 0.6, 0.8), alpha=alpha, terms=terms)
    hext = rng.standard_normal((3,) + p.node_shape) * 3e4
    if terms & TERM_DMI:        # cell-wise DMI constant; the interfacial kind when the demag term is off
        p = dataclasses.replace(p, D=rng.uniform(1e-3, 3e-3, n), dmi_kind="bulk" if terms & TERM_DEMAG else "interfacial",
                                dmi_normal=1)
    if terms & TERM_RKKY:
        p = dataclasses.replace(p, rkky_J=2e-3, rkky_planes=(0, n[2]))
    if terms & TERM_CUBIC:
        p = dataclasses.replace(p, Kc=rng.uniform(1e4, 5e4, n), cubic_axes=np.linalg.qr(rng.standard_normal((3, 3)))[0])
    return p, (lambda t: hext)


def with_Ms(p, Ms):
    return dataclasses.replace(p, Ms=Ms)


@pytest.mark.parametrize("terms", [ALL, TERM_EXCHANGE | TERM_DEMAG, TERM_DEMAG, TERM_EXCHANGE | TERM_ANISO | TERM_ZEEMAN,
                                   ALL | TERM_DMI, TERM_EXCHANGE | TERM_DMI, TERM_DMI, ALL | TERM_RKKY, TERM_RKKY | TERM_DMI, ALL | TERM_CUBIC, TERM_CUBIC])
def test_dense_jacobians_by_finite_differences(terms):
    """Explicit dense Jacobians of the oracle's own forward RHS by central differences on a
    3x2x2-cell mesh; both vector-Jacobian products must equal a^T J."""
    p, zee = make(terms=terms)
    p.Nt  # build tensor once
    rng = np.random.default_rng(1)
    m = rand_unit(p.node_shape, 2) * (1 + 0.05 * rng.standard_normal(p.node_shape))   # |m| != 1 on purpose
    a = rng.standard_normal(m.shape)
    f, dadt, dudt = adjoint.adjoint_rhs(p, 0.0, m, a, zee)
    assert np.allclose(f, llg.llg_rhs(p, 0.0, m, zee), rtol=1e-14)
    # J_m
    Jm_T_a = np.zeros(m.size)
    fl = m.ravel()
    for k in range(m.size):
        h = 1e-6
        mp_, mm_ = fl.copy(), fl.copy()
        mp_[k] += h
        mm_[k] -= h
        col = (llg.llg_rhs(p, 0.0, mp_.reshape(m.shape), zee) - llg.llg_rhs(p, 0.0, mm_.reshape(m.shape), zee)) / (2 * h)
        Jm_T_a[k] = np.sum(a * col)
    assert np.allclose(-dadt.ravel(), Jm_T_a, rtol=1e-7, atol=1e-8 * np.abs(Jm_T_a).max())
    # J_Ms
    JMs_T_a = np.zeros(p.Ms.size)
    for k in range(p.Ms.size):
        h = 1e-4 * p.Ms.ravel()[k]
        Mp, Mm = p.Ms.ravel().copy(), p.Ms.ravel().copy()
        Mp[k] += h
        Mm[k] -= h
        col = (llg.llg_rhs(with_Ms(p, Mp.reshape(p.n_cells)), 0.0, m, zee)
               - llg.llg_rhs(with_Ms(p, Mm.reshape(p.n_cells)), 0.0, m, zee)) / (2 * h)
        JMs_T_a[k] = np.sum(a * col)
    assert np.allclose(-dudt.ravel(), JMs_T_a, rtol=1e-6, atol=1e-7 * np.abs(JMs_T_a).max())


def test_dense_jacobian_with_a_vacuum_corner():
    """Reading C7 carries no adjoint at nodes with (S Ms)_n = 0.  With every material constant 0 in the vacuum cells
    (the vacuum is empty) that is the exact transposed Jacobian, vacuum nodes included: a node of a magnetic cell
    always has (S Ms) > 0, so m at a vacuum node enters no field.  3x3x2 cells with a 2x2x2 vacuum corner, every term
    on (DMI and the cubic term included), a^T J by central differences of the forward RHS."""
    terms = ALL | TERM_DMI | TERM_CUBIC
    p, zee = make(n=(3, 3, 2), terms=terms, seed=7)
    vac = np.zeros(p.n_cells, dtype=bool)
    vac[:2, :2, :] = True
    p = dataclasses.replace(p, **{k: np.where(vac, 0.0, getattr(p, k)) for k in ("Ms", "A", "Ku", "D", "Kc")})
    assert np.any(p.L == 0) and np.any(p.L > 0)
    rng = np.random.default_rng(8)
    m = rand_unit(p.node_shape, 9) * (1 + 0.05 * rng.standard_normal(p.node_shape))
    a = rng.standard_normal(m.shape)
    _, dadt, _ = adjoint.adjoint_rhs(p, 0.0, m, a, zee)
    fl, Jm_T_a = m.ravel(), np.zeros(m.size)
    for k in range(m.size):
        h = 1e-6
        mp_, mm_ = fl.copy(), fl.copy()
        mp_[k] += h
        mm_[k] -= h
        col = (llg.llg_rhs(p, 0.0, mp_.reshape(m.shape), zee) - llg.llg_rhs(p, 0.0, mm_.reshape(m.shape), zee)) / (2 * h)
        Jm_T_a[k] = np.sum(a * col)
    assert np.allclose(-dadt.ravel(), Jm_T_a, rtol=1e-7, atol=1e-8 * np.abs(Jm_T_a).max())
    assert np.all(dadt[:, p.L == 0] == 0)


def test_dot_product_test_larger_mesh():
    """<a, J v> = <J^T a, v> with J v by central differences (6x5x3 cells, all terms)."""
    p, zee = make(n=(6, 5, 3), seed=3)
    rng = np.random.default_rng(4)
    m = rand_unit(p.node_shape, 5)
    a = rng.standard_normal(m.shape)
    v = rng.standard_normal(m.shape)
    w = rng.standard_normal(p.n_cells) * 1e5
    _, dadt, dudt = adjoint.adjoint_rhs(p, 0.0, m, a, zee)
    h = 1e-6
    Jv = (llg.llg_rhs(p, 0.0, m + h * v, zee) - llg.llg_rhs(p, 0.0, m - h * v, zee)) / (2 * h)
    lhs, rhs = np.sum(a * Jv), np.sum(-dadt * v)
    assert abs(lhs - rhs) < 1e-8 * abs(lhs)
    h = 1e-5
    Jw = (llg.llg_rhs(with_Ms(p, p.Ms + h * w), 0.0, m, zee) - llg.llg_rhs(with_Ms(p, p.Ms - h * w), 0.0, m, zee)) / (2 * h)
    lhs, rhs = np.sum(a * Jw), np.sum(-dudt * w)
    assert abs(lhs - rhs) < 1e-6 * abs(lhs)


def test_transpose_field_operator_is_L_H_Linv():
    """H^T b = L o H(b/L) equals the explicit transpose of the dense field matrix."""
    p, _ = make(terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO)
    nn = int(np.prod((3,) + p.node_shape))
    Hmat = np.zeros((nn, nn))
    for k in range(nn):
        e = np.zeros(nn)
        e[k] = 1.0
        Hmat[:, k] = llg.effective_field(p, e.reshape((3,) + p.node_shape)).ravel()
    b = np.random.default_rng(6).standard_normal((3,) + p.node_shape)
    L = p.L
    got = L * llg.effective_field(p, b / L)
    assert np.allclose(got.ravel(), Hmat.T @ b.ravel(), rtol=1e-12, atol=1e-12 * np.abs(got).max())


def objective_and_grad(p, m0, zee, dt, nst, w, ckpt_every):
    mT, ck = adjoint.forward_rk4(p, m0, dt, nst, zee, checkpoint_every=ckpt_every)
    J = float(np.sum(w * mT))
    _, _, u0 = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck if ckpt_every else None)
    return J, u0, mT


def test_adjoint_state_gradient_against_finite_differences():
    """C8 on an 8x3x1 film, 300 RK4 steps: dJ/dMs from Eq. (29)-(30) vs central differences."""
    rng = np.random.default_rng(7)
    n, dx = (8, 3, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), np.full(n, 3.65e-12), np.zeros(n), alpha=1e-2,
                terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ZEEMAN)
    p.Nt
    zee = lambda t: np.array([0.0, 2e3, 0.0])
    m0 = 0.1 * rng.standard_normal((3,) + p.node_shape)
    m0[0] += 1
    m0 /= np.sqrt(np.sum(m0 * m0, axis=0))
    w = np.zeros_like(m0)
    w[1, -3:] = 1.0 / w[1, -3:].size
    dt, nst = 5e-14, 300
    J, u0, _ = objective_and_grad(p, m0, zee, dt, nst, w, 50)
    _, u0_nock, _ = objective_and_grad(p, m0, zee, dt, nst, w, 0)
    cells = [(0, 0, 0), (3, 1, 0), (7, 2, 0), (5, 0, 0)]
    for c in cells:
        h = 1e-4 * p.Ms[c]
        Mp, Mm = p.Ms.copy(), p.Ms.copy()
        Mp[c] += h
        Mm[c] -= h
        Jp = float(np.sum(w * adjoint.forward_rk4(with_Ms(p, Mp), m0, dt, nst, zee)[0]))
        Jm = float(np.sum(w * adjoint.forward_rk4(with_Ms(p, Mm), m0, dt, nst, zee)[0]))
        fd = (Jp - Jm) / (2 * h)
        assert abs(u0[c] - fd) < 1e-3 * abs(fd), (c, u0[c], fd)
        assert abs(u0_nock[c] - fd) < 1e-3 * abs(fd)
    # invariance under the checkpoint interval (same tolerance)
    _, u0_b, _ = objective_and_grad(p, m0, zee, dt, nst, w, 100)
    assert np.abs(u0_b - u0).max() < 1e-3 * np.abs(u0).max()


def test_objectives_at_several_times_against_finite_differences():
    """PAPER.md:228 on a 6x2x1 film: L = w1 . m(T1) + w2 . m(T2) + wT . m(T), T1 < T2 < T; the
    adjoint variable jumps by grad L_i at T_i.  dL/dMs against central differences, and additivity:
    the gradient equals the sum of the single-time gradients over [0, T1], [0, T2], [0, T]."""
    rng = np.random.default_rng(17)
    n, dx = (6, 2, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), np.full(n, 3.65e-12), np.zeros(n), alpha=1e-2,
                terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ZEEMAN)
    p.Nt
    zee = lambda t: np.array([0.0, 2e3, 0.0])
    m0 = 0.1 * rng.standard_normal((3,) + p.node_shape)
    m0[0] += 1
    m0 /= np.sqrt(np.sum(m0 * m0, axis=0))
    dt, nst, s1, s2 = 5e-14, 72, 24, 54
    w1, w2, wT = (rng.standard_normal(m0.shape) for _ in range(3))

    def traj(prob):
        out, m = {}, m0.copy()
        for s in range(nst):
            if s in (s1, s2):
                out[s] = m.copy()
            m = llg.rk4_step(prob, s * dt, dt, m, zee)
        return out[s1], out[s2], m

    def L(prob):
        a, b, c = traj(prob)
        return float(np.sum(w1 * a) + np.sum(w2 * b) + np.sum(wT * c))

    mT, ck = adjoint.forward_rk4(p, m0, dt, nst, zee, checkpoint_every=18)
    _, _, u0 = adjoint.backward_rk4(p, mT, wT, dt, nst, zee, checkpoints=ck, a_jumps={s1: w1, s2: w2})
    for c in [(0, 0, 0), (3, 1, 0), (5, 0, 0)]:
        h = 1e-4 * p.Ms[c]
        Mp, Mm = p.Ms.copy(), p.Ms.copy()
        Mp[c] += h
        Mm[c] -= h
        fd = (L(with_Ms(p, Mp)) - L(with_Ms(p, Mm))) / (2 * h)
        assert abs(u0[c] - fd) < 1e-3 * abs(fd), (c, u0[c], fd)
    # additivity over the objectives (the adjoint system is linear in a): three single-time runs;
    # equal up to the backward reconstruction of m between checkpoints (a run that ends at T_i
    # starts from the exact m(T_i), the joint run arrives there by inverse integration)
    total = np.zeros_like(u0)
    for steps, w in ((s1, w1), (s2, w2), (nst, wT)):
        mS, ckS = adjoint.forward_rk4(p, m0, dt, steps, zee, checkpoint_every=18)
        total += adjoint.backward_rk4(p, mS, w, dt, steps, zee, checkpoints=ckS)[2]
    assert np.abs(total - u0).max() < 1e-6 * np.abs(u0).max()
    # a jump of zero is no jump
    _, _, u_plain = adjoint.backward_rk4(p, mT, wT, dt, nst, zee, checkpoints=ck)
    _, _, u_zero = adjoint.backward_rk4(p, mT, wT, dt, nst, zee, checkpoints=ck, a_jumps={s1: 0.0 * w1})
    assert np.array_equal(u_plain, u_zero)


def test_hext_vjp_against_finite_differences():
    """adjoint_rhs_hext: a . (df/dh) e_j by central differences of the forward RHS in a uniform field
    h added to a nodal H_ext, on a mesh with a vacuum corner (nodes with L = 0 see no field)."""
    p, zee = make((3, 2, 2), seed=3)
    Ms = p.Ms.copy()
    Ms[0, 0, :] = 0.0
    Ms[0, 1, 0] = 0.0
    p = with_Ms(p, Ms)
    assert np.any(p.L == 0) and np.any(p.L > 0)
    m = rand_unit(p.node_shape, 4)
    a = np.random.default_rng(5).standard_normal(m.shape)
    base = zee(0.0)
    got = adjoint.adjoint_rhs_hext(p, 0.0, m, a)
    for j in range(3):
        e = np.zeros((3, 1, 1, 1))
        e[j] = 1.0
        eps = 10.0
        fp = llg.llg_rhs(p, 0.0, m, lambda t: base + eps * e)
        fm = llg.llg_rhs(p, 0.0, m, lambda t: base - eps * e)
        fd = -np.sum(a * (fp - fm)) / (2 * eps)
        assert abs(got[j] - fd) <= 1e-9 * np.abs(got).max(), (j, got[j], fd)
    # no Zeeman term: no dependence on h
    p0 = Problem(p.n_cells, p.dx, p.Ms, p.A, p.Ku, p.ku_axis, p.gamma, p.alpha, TERM_EXCHANGE | TERM_DEMAG, p._Nt)
    assert np.all(adjoint.adjoint_rhs_hext(p0, 0.0, m, a) == 0.0)


def test_hext_gradient_of_a_trajectory_against_finite_differences():
    """dL/dh of L = w . m(T) for a uniform external field h (the design variable behind the field
    angles of Eqs. 31-33): u_h(0) of the backward pass vs central differences of the forward solve."""
    rng = np.random.default_rng(27)
    n, dx = (6, 2, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), np.full(n, 3.65e-12), np.full(n, 2e4), ku_axis=(0.0, 0.6, 0.8),
                alpha=0.05, terms=ALL)
    p.Nt
    h0 = np.array([1e3, 2e3, -1.5e3])
    m0 = 0.1 * rng.standard_normal((3,) + p.node_shape)
    m0[0] += 1
    m0 /= np.sqrt(np.sum(m0 * m0, axis=0))
    w = rng.standard_normal(m0.shape)
    dt, nst = 5e-14, 80
    zee = lambda t: h0
    mT, ck = adjoint.forward_rk4(p, m0, dt, nst, zee, checkpoint_every=40)
    _, _, u0, uh = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck, with_hext=True)
    _, _, u0_plain = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck)
    assert np.array_equal(u0, u0_plain)
    for j in range(3):
        e = np.zeros(3)
        e[j] = 20.0
        Jp = float(np.sum(w * adjoint.forward_rk4(p, m0, dt, nst, lambda t: h0 + e)[0]))
        Jm = float(np.sum(w * adjoint.forward_rk4(p, m0, dt, nst, lambda t: h0 - e)[0]))
        fd = (Jp - Jm) / 40.0
        assert abs(uh[j] - fd) < 1e-3 * np.abs(uh).max(), (j, uh[j], fd)


def with_A_Ku(p, A, Ku):
    return Problem(p.n_cells, p.dx, p.Ms, A, Ku, p.ku_axis, p.gamma, p.alpha, p.terms, p._Nt)


def test_materials_vjp_against_finite_differences():
    """adjoint_rhs_materials: a . (df/dA_c), a . (df/dKu_c) for every cell of a 3x2x2 mesh with a
    vacuum corner by central differences of the forward RHS (f is linear in A and Ku)."""
    p, zee = make((3, 2, 2), seed=13)
    Ms = p.Ms.copy()
    Ms[0, 0, :] = 0.0
    p = with_Ms(p, Ms)
    m = rand_unit(p.node_shape, 14)
    a = np.random.default_rng(15).standard_normal(m.shape)
    gA, gKu = adjoint.adjoint_rhs_materials(p, 0.0, m, a)
    for c in np.ndindex(*p.n_cells):
        for which, got in (("A", gA), ("Ku", gKu)):
            base = p.A if which == "A" else p.Ku
            h = 0.1 * base[c]
            up, dn = base.copy(), base.copy()
            up[c] += h
            dn[c] -= h
            pp = with_A_Ku(p, up, p.Ku) if which == "A" else with_A_Ku(p, p.A, up)
            pm = with_A_Ku(p, dn, p.Ku) if which == "A" else with_A_Ku(p, p.A, dn)
            fd = -np.sum(a * (llg.llg_rhs(pp, 0.0, m, zee) - llg.llg_rhs(pm, 0.0, m, zee))) / (2 * h)
            assert abs(got[c] - fd) <= 1e-9 * np.abs(got).max(), (which, c, got[c], fd)
    assert np.abs(gA).max() > 0 and np.abs(gKu).max() > 0
    # terms that are off do not depend on their coefficient
    p0 = Problem(p.n_cells, p.dx, p.Ms, p.A, p.Ku, p.ku_axis, p.gamma, p.alpha, TERM_DEMAG | TERM_ZEEMAN, p._Nt)
    g0 = adjoint.adjoint_rhs_materials(p0, 0.0, m, a)
    assert np.all(g0[0] == 0.0) and np.all(g0[1] == 0.0)


def test_materials_gradient_of_a_trajectory_against_finite_differences():
    """dL/dA_c and dL/dKu_c of L = w . m(T): (u_A, u_Ku)(0) of the backward pass vs central
    differences of the forward solve on three cells."""
    rng = np.random.default_rng(37)
    n, dx = (6, 2, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), rng.uniform(3e-12, 4e-12, n), rng.uniform(1e4, 3e4, n),
                ku_axis=(0.0, 0.6, 0.8), alpha=0.05, terms=ALL)
    p.Nt
    zee = lambda t: np.array([1e3, 2e3, -1.5e3])
    m0 = 0.3 * rng.standard_normal((3,) + p.node_shape)
    m0[0] += 1
    m0 /= np.sqrt(np.sum(m0 * m0, axis=0))
    w = rng.standard_normal(m0.shape)
    dt, nst = 5e-14, 50
    mT, ck = adjoint.forward_rk4(p, m0, dt, nst, zee, checkpoint_every=25)
    out = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck, with_hext=True, with_materials=True)
    assert len(out) == 6
    uA, uKu = out[4], out[5]
    plain = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck)
    assert np.array_equal(out[2], plain[2]) and np.array_equal(out[1], plain[1])
    J = lambda prob: float(np.sum(w * adjoint.forward_rk4(prob, m0, dt, nst, zee)[0]))
    for c in [(0, 0, 0), (3, 1, 0), (5, 0, 0)]:
        for which, got, base in (("A", uA, p.A), ("Ku", uKu, p.Ku)):
            h = 1e-3 * base[c]
            up, dn = base.copy(), base.copy()
            up[c] += h
            dn[c] -= h
            pp = with_A_Ku(p, up, p.Ku) if which == "A" else with_A_Ku(p, p.A, up)
            pm = with_A_Ku(p, dn, p.Ku) if which == "A" else with_A_Ku(p, p.A, dn)
            fd = (J(pp) - J(pm)) / (2 * h)
            assert abs(got[c] - fd) < 2e-3 * np.abs(got).max(), (which, c, got[c], fd)


def test_adjoint_driver_zero_and_linearity():
    rng = np.random.default_rng(8)
    n, dx = (4, 2, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), np.full(n, 3.65e-12), np.zeros(n), alpha=1e-2,
                terms=TERM_EXCHANGE | TERM_DEMAG)
    m0 = rand_unit(p.node_shape, 9)
    mT, ck = adjoint.forward_rk4(p, m0, 5e-14, 20, checkpoint_every=10)
    a1 = rng.standard_normal(m0.shape)
    a2 = rng.standard_normal(m0.shape)
    run = lambda a: adjoint.backward_rk4(p, mT, a, 5e-14, 20, checkpoints=ck)[2]
    assert np.all(run(np.zeros_like(a1)) == 0.0)
    u1, u2, u12 = run(a1), run(a2), run(2.0 * a1 - 0.5 * a2)
    assert np.allclose(u12, 2.0 * u1 - 0.5 * u2, rtol=1e-10, atol=1e-12 * np.abs(u1).max())
    # checkpoints put m back exactly on the forward trajectory
    mb = adjoint.backward_rk4(p, mT, a1, 5e-14, 20, checkpoints=ck)[0]
    assert np.array_equal(mb, m0)


def test_hnodal_vjp_against_finite_differences_entry_by_entry():
    """adjoint_rhs_hnodal: a . (df/dh_{n,j}) for EVERY nodal entry of a nodal external field, by central
    differences of the forward RHS, on a mesh with a vacuum corner and cell-wise Ms; its sum over the
    nodes is the uniform-field gradient adjoint_rhs_hext."""
    p, zee = make((3, 2, 2), seed=3)
    Ms = p.Ms.copy()
    Ms[0, 0, :] = 0.0
    Ms[0, 1, 0] = 0.0
    p = with_Ms(p, Ms)
    m = rand_unit(p.node_shape, 4)
    a = np.random.default_rng(5).standard_normal(m.shape)
    base = zee(0.0)
    got = adjoint.adjoint_rhs_hnodal(p, 0.0, m, a)
    assert got.shape == m.shape
    eps = 10.0
    for idx in np.ndindex(*m.shape):
        d = np.zeros_like(m)
        d[idx] = eps
        fp = llg.llg_rhs(p, 0.0, m, lambda t: base + d)
        fm = llg.llg_rhs(p, 0.0, m, lambda t: base - d)
        fd = -np.sum(a * (fp - fm)) / (2 * eps)
        assert abs(got[idx] - fd) <= 1e-9 * np.abs(got).max(), (idx, got[idx], fd)
    assert np.allclose(got.sum(axis=(1, 2, 3)), adjoint.adjoint_rhs_hext(p, 0.0, m, a), rtol=1e-12)
    p0 = Problem(p.n_cells, p.dx, p.Ms, p.A, p.Ku, p.ku_axis, p.gamma, p.alpha, TERM_EXCHANGE | TERM_DEMAG, p._Nt)
    assert np.all(adjoint.adjoint_rhs_hnodal(p0, 0.0, m, a) == 0.0)


def test_hnodal_gradient_of_a_trajectory_against_finite_differences():
    """dL/dh_{n,j} of L = w . m(T) for a time-constant nodal external field: u_hn(0) of the backward pass
    vs central differences of the forward solve at seeded entries; summed over nodes it is dL/dh of the
    uniform field."""
    rng = np.random.default_rng(27)
    n, dx = (6, 2, 1), (4e-9, 4e-9, 5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 1.5e5, n), np.full(n, 3.65e-12), np.full(n, 2e4), ku_axis=(0.0, 0.6, 0.8),
                alpha=0.05, terms=ALL)
    p.Nt
    hn = 2e3 * rng.standard_normal((3,) + p.node_shape)
    m0 = 0.1 * rng.standard_normal((3,) + p.node_shape)
    m0[0] += 1
    m0 /= np.sqrt(np.sum(m0 * m0, axis=0))
    w = rng.standard_normal(m0.shape)
    dt, nst = 5e-14, 80
    zee = lambda t: hn
    mT, ck = adjoint.forward_rk4(p, m0, dt, nst, zee, checkpoint_every=40)
    out = adjoint.backward_rk4(p, mT, w, dt, nst, zee, checkpoints=ck, with_hext=True, with_hnodal=True)
    uh, uhn = out[3], out[4]
    assert np.allclose(uhn.sum(axis=(1, 2, 3)), uh, rtol=1e-10)
    scale = np.abs(uhn).max()
    for _ in range(6):
        idx = tuple(int(rng.integers(0, k)) for k in hn.shape)
        d = np.zeros_like(hn)
        d[idx] = 50.0
        Lp = np.sum(w * adjoint.forward_rk4(p, m0, dt, nst, lambda t: hn + d)[0])
        Lm = np.sum(w * adjoint.forward_rk4(p, m0, dt, nst, lambda t: hn - d)[0])
        fd = (Lp - Lm) / 100.0
        assert abs(uhn[idx] - fd) <= 1e-3 * scale, (idx, uhn[idx], fd)


def test_cubic_hessian_vector_product_is_the_derivative_of_the_variation():
    """hessvec_cubic(m, v) against a central difference of variation_cubic along v; symmetric: u . H v = v . H u."""
    from oracle import more_terms as mt
    rng = np.random.default_rng(4)
    n, dx = (3, 2, 2), np.array([1.0, 1.2, 0.8])
    Kc = rng.uniform(0.5, 2.0, n)
    axes = np.linalg.qr(rng.standard_normal((3, 3)))[0]
    nn = tuple(k + 1 for k in n)
    m, v, u = (rng.standard_normal((3,) + nn) for _ in range(3))
    hv = mt.hessvec_cubic(m, v, Kc, axes, dx)
    eps = 1e-6
    fd = (mt.variation_cubic(m + eps * v, Kc, axes, dx) - mt.variation_cubic(m - eps * v, Kc, axes, dx)) / (2 * eps)
    assert np.allclose(hv, fd, rtol=1e-8, atol=1e-9 * np.abs(fd).max())
    assert np.isclose(np.sum(u * hv), np.sum(v * mt.hessvec_cubic(m, u, Kc, axes, dx)), rtol=1e-12)


@pytest.mark.parametrize("D,n", [(2, (3, 2, 1)), (1, (4, 1, 1))])
def test_reduced_basis_vjps_against_finite_differences(D, n):
    """The adjoint right-hand side on the reduced bases of Eqs. (23)-(24) (Problem.basis = 2, 1): every
    vector-Jacobian product against central differences of the forward RHS of the same basis (itself pinned in
    tests/test_oracle_lowdim.py), all four base terms on, one vacuum cell: a^T df/dm and a^T df/dMs densely,
    a^T df/dh for a uniform and for a nodal external field, a^T df/dA_c and a^T df/dKu_c for every cell."""
    rng = np.random.default_rng(40 + D)
    dx = (3e-9, 2.5e-9, 3.5e-9)
    Ms = rng.uniform(4e5, 8e5, n)
    Ms[0, 0, 0] = 0.0
    p = Problem(n, dx, Ms, rng.uniform(0.8e-11, 1.3e-11, n), rng.uniform(1e5, 5e5, n), ku_axis=(0.0, 0.6, 0.8),
                alpha=0.1, terms=ALL, basis=D)
    p.Nt
    assert np.any(p.L == 0)
    hext = rng.standard_normal((3,) + p.node_shape) * 3e4
    zee = lambda t: hext
    m = rand_unit(p.node_shape, 2) * (1 + 0.05 * rng.standard_normal(p.node_shape))
    a = rng.standard_normal(m.shape)
    rhs = lambda prob, mm, hh=hext: llg.llg_rhs(prob, 0.0, mm, lambda t: hh)
    f, dadt, dudt = adjoint.adjoint_rhs(p, 0.0, m, a, zee)
    assert np.allclose(f, rhs(p, m), rtol=1e-14)
    live = np.broadcast_to(p.L > 0, m.shape).ravel()
    got = -dadt.ravel()
    for k in range(m.size):
        e = np.zeros(m.size)
        e[k] = 1e-6
        fd = np.sum(a * (rhs(p, m + e.reshape(m.shape)) - rhs(p, m - e.reshape(m.shape)))) / 2e-6
        if live[k]:
            assert abs(got[k] - fd) <= 1e-7 * np.abs(got).max(), (k, got[k], fd)
        else:
            assert got[k] == 0.0          # reading C7: no adjoint at vacuum nodes
    for c in np.ndindex(*n):
        if p.Ms[c] == 0:
            continue
        h = 1e-4 * p.Ms[c]
        up, dn = p.Ms.copy(), p.Ms.copy()
        up[c] += h
        dn[c] -= h
        fd = np.sum(a * (rhs(dataclasses.replace(p, Ms=up), m) - rhs(dataclasses.replace(p, Ms=dn), m))) / (2 * h)
        assert abs(-dudt[c] - fd) <= 1e-6 * np.abs(dudt).max(), (c, dudt[c], fd)
    # external field: uniform and nodal
    gu = adjoint.adjoint_rhs_hext(p, 0.0, m, a)
    gn = adjoint.adjoint_rhs_hnodal(p, 0.0, m, a)
    assert np.allclose(gn.reshape(3, -1).sum(axis=1), gu, rtol=1e-12)
    eps = 10.0
    for k in range(0, m.size, 3):
        e = np.zeros(m.size)
        e[k] = eps
        e = e.reshape(m.shape)
        fd = -np.sum(a * (rhs(p, m, hext + e) - rhs(p, m, hext - e))) / (2 * eps)
        assert abs(gn.ravel()[k] - fd) <= 1e-9 * np.abs(gn).max(), (k, gn.ravel()[k], fd)
    gA, gKu = adjoint.adjoint_rhs_materials(p, 0.0, m, a)
    for c in np.ndindex(*n):
        for name, g in (("A", gA), ("Ku", gKu)):
            base = getattr(p, name)
            h = 0.1 * base[c]
            up, dn = base.copy(), base.copy()
            up[c] += h
            dn[c] -= h
            fd = -np.sum(a * (rhs(dataclasses.replace(p, **{name: up}), m) - rhs(dataclasses.replace(p, **{name: dn}), m))) / (2 * h)
            assert abs(g[c] - fd) <= 1e-9 * np.abs(g).max(), (name, c, g[c], fd)
