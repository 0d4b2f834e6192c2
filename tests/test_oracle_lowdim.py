"""Pins for oracle/lowdim.py: the reduced 2-D / 1-D nodal bases of PAPER.md:183-195 (Eqs. 23-24).

What fixes them other than the code itself: numerical quadrature of the products of Eqs. (23)-(24)
over the 3-D cell; a brute-force global assembly of the weak form (17) with global hat functions that
are constant along the reduced axes; closed forms (helix, the textbook 1-D difference Laplacian,
uniform states); the identity behind Sec. III C -- a reduced basis function is the sum of the 3-D ones
along the reduced axes, so the reduced scheme must reproduce the (separately pinned) 3-D oracle on
states that are uniform along those axes, term by term and for the demag averaging; and the L-weighted
symmetry the adjoint would rely on.
"""
import itertools

import numpy as np
import pytest

from oracle import llg, local_fields as lf, lowdim as ld, mesh
from oracle.llg import Problem, TERM_ANISO, TERM_DEMAG, TERM_EXCHANGE, TERM_ZEEMAN

MU0 = 4e-7 * np.pi
ALL = TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO | TERM_ZEEMAN


def _cells(D, n1=6, n2=4):
    return (n1, n2, 1) if D == 2 else (n1, 1, 1)


@pytest.mark.parametrize("D", [2, 1])
def test_basis_is_nodal_constant_along_reduced_axes_and_sums_to_one(D):
    rng = np.random.default_rng(0)
    x = rng.uniform(0, 1, (50, 3))
    tot = 0.0
    for i in ld.local(D):
        corner = np.array(list(i) + [0.3] * (3 - D), dtype=float)
        for ip in ld.local(D):
            other = np.array(list(ip) + [0.9] * (3 - D), dtype=float)
            assert ld.phi_ref(i, other, D) == (1.0 if ip == i else 0.0)
        assert ld.phi_ref(i, corner, D) == 1.0
        # constant along the reduced axes
        y = x.copy()
        y[:, D:] = rng.uniform(0, 1, (50, 3 - D))
        assert np.array_equal(ld.phi_ref(i, x, D), ld.phi_ref(i, y, D))
        # gradient against a central difference, zero along the reduced axes
        g = ld.grad_phi_ref(i, x, D)
        for d in range(3):
            e = np.zeros(3)
            e[d] = 1e-6
            fd = (ld.phi_ref(i, x + e, D) - ld.phi_ref(i, x - e, D)) / 2e-6
            assert np.allclose(g[:, d], fd, atol=1e-9)
        assert np.all(g[:, D:] == 0)
        tot = tot + ld.phi_ref(i, x, D)
    assert np.allclose(tot, 1.0)
    # the reduced function is the sum of the 3-D ones along the reduced axes
    for i in ld.local(D):
        s = sum(mesh.phi_ref(tuple(i) + r, x) for r in itertools.product((0, 1), repeat=3 - D))
        assert np.allclose(s, ld.phi_ref(i, x, D))


@pytest.mark.parametrize("D", [2, 1])
def test_element_matrices_equal_gauss_quadrature_over_the_3d_cell(D):
    dx = np.array([2e-9, 3e-9, 5e-9])
    K, M = ld.element_matrices(dx, D)
    g = 0.5 + 0.5 * np.array([-np.sqrt(3 / 5), 0.0, np.sqrt(3 / 5)])
    gw = 0.5 * np.array([5 / 9, 8 / 9, 5 / 9])
    pts = np.array(list(itertools.product(g, repeat=3)))
    wts = np.array([a * b * c for a, b, c in itertools.product(gw, repeat=3)]) * dx.prod()
    for i in ld.local(D):
        for ip in ld.local(D):
            mq = np.sum(wts * ld.phi_ref(i, pts, D) * ld.phi_ref(ip, pts, D))
            kq = np.sum(wts * np.sum(ld.grad_phi_ref(i, pts, D) / dx * ld.grad_phi_ref(ip, pts, D) / dx, axis=1))
            assert np.isclose(M[i + ip], mq, rtol=1e-13)
            assert np.isclose(K[i + ip], kq, rtol=1e-13, atol=1e-13 * np.abs(K).max())
    n = 2 ** D
    Km, Mm = K.reshape(n, n), M.reshape(n, n)
    assert np.allclose(Km, Km.T) and np.allclose(Mm, Mm.T)
    assert np.allclose(Km.sum(axis=1), 0, atol=1e-12 * np.abs(Km).max())
    assert np.allclose(Mm.sum(axis=1), dx.prod() / n)
    assert np.linalg.eigvalsh(Km).min() > -1e-12 * np.abs(Km).max()


@pytest.mark.parametrize("D", [2, 1])
def test_scatter_gather_are_transposes_and_lumped_mass_sums_to_the_volume_integral(D):
    rng = np.random.default_rng(1)
    n = _cells(D)
    dx = (2e-9, 3e-9, 5e-9)
    b = rng.standard_normal(n)
    a = rng.standard_normal(ld.node_shape(n, D))
    assert np.isclose(np.sum(ld.scatter_cells_to_nodes(b, D) * a), np.sum(b * ld.gather_nodes_to_cells(a, D)))
    cnt = ld.scatter_cells_to_nodes(np.ones(n), D)
    assert cnt.min() == 1 and cnt.max() == 2 ** D
    Ms = rng.uniform(1e5, 8e5, n)
    assert np.isclose(ld.lumped_mass(Ms, dx, D).sum(), MU0 * Ms.sum() * np.prod(dx), rtol=1e-14)
    with pytest.raises(ValueError):
        ld.node_shape((4, 4, 2), 2)
    with pytest.raises(ValueError):
        ld.node_shape((4, 2, 1), 1)


@pytest.mark.parametrize("D", [2, 1])
def test_reduced_scheme_equals_the_3d_scheme_on_states_uniform_along_the_reduced_axes(D):
    """Sec. III C in one identity: with random cell-wise Ms, A, Ku, a tilted axis, a nodal external
    field and a vacuum cell, every term of the reduced oracle equals the 3-D oracle's field (at every
    copy of the node along the reduced axes) on the expanded state."""
    rng = np.random.default_rng(2)
    n = _cells(D, 7, 5)
    dx = (2e-9, 3e-9, 4e-9)
    Ms = rng.uniform(1e5, 8e5, n)
    Ms[0, 0, 0] = 0.0
    A = rng.uniform(0.5e-11, 2e-11, n)
    Ku = rng.uniform(1e4, 5e5, n)
    kax = (0.36, 0.48, 0.8)
    pr = Problem(n, dx, Ms, A, Ku, kax, 2.211e5, 0.1, ALL, basis=D)
    p3 = Problem(n, dx, Ms, A, Ku, kax, 2.211e5, 0.1, ALL, pr.Nt)
    m = rng.standard_normal((3,) + pr.node_shape)
    h = 1e4 * rng.standard_normal((3,) + pr.node_shape)
    got = llg.effective_field(pr, m, h, parts=True)
    ref = llg.effective_field(p3, ld.expand_to_3d(m, D), ld.expand_to_3d(h, D), parts=True)
    assert set(got) == {"exchange", "aniso", "zeeman", "demag"}
    for name in got:
        scale = np.abs(ref[name]).max()
        for r in itertools.product((0, 1), repeat=3 - D):
            sl = (slice(None), slice(None)) + tuple(slice(None) if d < D else slice(r[d - D], r[d - D] + 1)
                                                     for d in range(1, 3))
            assert np.abs(ref[name][sl] - got[name]).max() <= 1e-13 * scale, name
    # the vacuum corner node has L = 0 and H = 0
    assert np.all(llg.effective_field(pr, m, h)[:, 0, 0, 0] == 0)
    # and so do the right-hand side and a Runge-Kutta step
    z = lambda t: h
    z3 = lambda t: ld.expand_to_3d(h, D)
    mu = m / np.where(np.sum(m * m, axis=0) > 0, np.sqrt(np.sum(m * m, axis=0)), 1.0)
    y = llg.rk4_step(pr, 0.0, 2e-14, mu, z)
    y3 = llg.rk4_step(p3, 0.0, 2e-14, ld.expand_to_3d(mu, D), z3)
    assert np.abs(ld.expand_to_3d(y, D) - y3).max() <= 1e-13


def test_helix_closed_form_on_a_film():
    """m = (cos kx, sin kx, 0) on the film nodes, uniform A: E = A V_total 4 sin^2(k dx/2)/dx^2 and
    H = -(2A/mu0 Ms) 4 sin^2(k dx/2)/dx^2 m at the nodes interior in x (the y mass row sums to 1)."""
    n, dx = (16, 3, 1), (2e-9, 3e-9, 5e-9)
    A, Ms = 1.3e-11, 8e5
    kx = 2 * np.pi / (10.5 * dx[0])
    X = (np.arange(n[0] + 1) * dx[0])[:, None, None] * np.ones(ld.node_shape(n, 2))
    m = np.stack([np.cos(kx * X), np.sin(kx * X), np.zeros_like(X)])
    lam = 4 * np.sin(kx * dx[0] / 2) ** 2 / dx[0] ** 2
    E = ld.energy_exchange(m, np.full(n, A), dx, 2)
    assert np.isclose(E, A * np.prod(n) * np.prod(dx) * lam, rtol=1e-13)
    H = lf.field_from_variation(ld.variation_exchange(m, np.full(n, A), dx, 2), ld.lumped_mass(np.full(n, Ms), dx, 2))
    expect = -(2 * A / (MU0 * Ms)) * lam * m
    assert np.allclose(H[:, 1:-1], expect[:, 1:-1], rtol=1e-12, atol=1e-6)
    # energy identity E = -1/2 sum L m . H
    L = ld.lumped_mass(np.full(n, Ms), dx, 2)
    assert np.isclose(E, -0.5 * np.sum(L * np.sum(m * H, axis=0)), rtol=1e-13)


def test_rod_basis_gives_the_textbook_difference_laplacian():
    """D = 1: H_i = (2A/mu0 Ms) (m_{i+1} - 2 m_i + m_{i-1}) / dx^2 at interior nodes, the one-sided
    difference (natural boundary condition) at the ends."""
    rng = np.random.default_rng(3)
    n, dx = (9, 1, 1), (1.5e-9, 4e-9, 6e-9)
    A, Ms = 1e-11, 5e5
    m = rng.standard_normal((3, 10, 1, 1))
    H = lf.field_from_variation(ld.variation_exchange(m, np.full(n, A), dx, 1), ld.lumped_mass(np.full(n, Ms), dx, 1))
    c = 2 * A / (MU0 * Ms) / dx[0] ** 2
    assert np.allclose(H[:, 1:-1], c * (m[:, 2:] - 2 * m[:, 1:-1] + m[:, :-2]), rtol=1e-12)
    assert np.allclose(H[:, 0], 2 * c * (m[:, 1] - m[:, 0]), rtol=1e-12)        # L is halved at the ends
    assert np.allclose(H[:, -1], 2 * c * (m[:, -2] - m[:, -1]), rtol=1e-12)


@pytest.mark.parametrize("D", [2, 1])
def test_uniform_states(D):
    rng = np.random.default_rng(4)
    n, dx = _cells(D), (2e-9, 2e-9, 5e-9)
    Ms = rng.uniform(1e5, 8e5, n)
    A = rng.uniform(1e-12, 2e-11, n)
    ns = ld.node_shape(n, D)
    L = ld.lumped_mass(Ms, dx, D)
    m = np.broadcast_to(np.array([0.6, 0.0, 0.8])[:, None, None, None], (3,) + ns).copy()
    H = lf.field_from_variation(ld.variation_exchange(m, A, dx, D), L)
    assert np.abs(H).max() <= 1e-14 * 2 * A.max() / (MU0 * Ms.min() * min(dx) ** 2)
    h = np.broadcast_to(np.array([1e3, -2e4, 5e4])[:, None, None, None], (3,) + ns)
    assert np.allclose(lf.field_from_variation(ld.variation_zeeman(h, Ms, dx, D), L), h, rtol=1e-14, atol=0)
    k = np.array([0.0, 0.6, 0.8])
    mk = np.broadcast_to(k[:, None, None, None], (3,) + ns).copy()
    Hk = lf.field_from_variation(ld.variation_uniaxial(mk, np.full(n, 5e5), k, dx, D),
                                 ld.lumped_mass(np.full(n, 8e5), dx, D))
    assert np.allclose(Hk, (2 * 5e5 / (MU0 * 8e5) * k)[:, None, None, None], rtol=1e-13)
    # node <-> cell averaging of a constant
    Hc = np.broadcast_to(np.array([1.0, 2.0, 3.0])[:, None, None, None], (3,) + n)
    assert np.allclose(ld.demag_field_nodes(Hc, Ms, D), np.array([1.0, 2.0, 3.0])[:, None, None, None])
    assert np.allclose(ld.cell_magnetization(m, Ms, D), Ms * np.array([0.6, 0.0, 0.8])[:, None, None, None])


def _hat(s):
    return np.maximum(0.0, 1.0 - np.abs(s))


def _dhat(s):
    return np.where(np.abs(s) < 1, -np.sign(s), 0.0)


@pytest.mark.parametrize("D,n", [(2, (4, 3, 1)), (1, (5, 1, 1))])
def test_brute_force_global_assembly_by_quadrature(D, n):
    """Eq. (17) assembled with global functions phi_n(x) = prod_{d<D} hat(x_d/dx_d - n_d), constant along
    the reduced axes, by 3-point Gauss quadrature over every 3-D cell; all three local terms and L."""
    rng = np.random.default_rng(5)
    dx = np.array([2e-9, 3e-9, 5e-9])
    ns = ld.node_shape(n, D)
    A = rng.uniform(0.5, 2.0, n) * 1e-11
    Ms = rng.uniform(1e5, 8e5, n)
    Ku = rng.uniform(1e4, 5e5, n)
    kax = np.array([0.36, 0.48, 0.8])
    m = rng.standard_normal((3,) + ns)
    hext = rng.standard_normal((3,) + ns) * 1e4
    g = 0.5 + 0.5 * np.array([-np.sqrt(3 / 5), 0.0, np.sqrt(3 / 5)])
    gw = 0.5 * np.array([5 / 9, 8 / 9, 5 / 9])
    nodes = list(itertools.product(*[range(k) for k in ns]))
    dE_ex, dE_an, dE_ze = (np.zeros((3,) + ns) for _ in range(3))
    lump = np.zeros(ns)
    for c in itertools.product(*[range(k) for k in n]):
        V = dx.prod()
        for (a, wa), (b, wb), (cc, wc) in itertools.product(zip(g, gw), repeat=3):
            w = wa * wb * wc * V
            s = np.array(c) + np.array([a, b, cc])
            phi, gphi = {}, {}
            for nd in nodes:
                h = [_hat(s[d] - nd[d]) for d in range(D)]
                if np.prod(h) == 0:
                    continue
                phi[nd] = np.prod(h)
                gr = np.zeros(3)
                for d in range(D):
                    gr[d] = _dhat(s[d] - nd[d]) / dx[d] * np.prod([h[e] for e in range(D) if e != d])
                gphi[nd] = gr
            mh = sum(m[(slice(None),) + nd] * v for nd, v in phi.items())
            hh = sum(hext[(slice(None),) + nd] * v for nd, v in phi.items())
            gm = sum(np.outer(m[(slice(None),) + nd], v) for nd, v in gphi.items())
            for nd in phi:
                idx = (slice(None),) + nd
                dE_ex[idx] += w * 2 * A[c] * gm @ gphi[nd]
                dE_an[idx] += w * (-2 * Ku[c]) * (mh @ kax) * kax * phi[nd]
                dE_ze[idx] += w * (-MU0 * Ms[c]) * hh * phi[nd]
                lump[nd] += w * MU0 * Ms[c] * phi[nd]
    assert np.allclose(lump, ld.lumped_mass(Ms, dx, D), rtol=1e-13)
    for got, ref in ((ld.variation_exchange(m, A, dx, D), dE_ex),
                     (ld.variation_uniaxial(m, Ku, kax, dx, D), dE_an),
                     (ld.variation_zeeman(hext, Ms, dx, D), dE_ze)):
        assert np.allclose(got, ref, rtol=1e-12, atol=1e-13 * np.abs(ref).max())


@pytest.mark.parametrize("D", [2, 1])
def test_field_operator_is_self_adjoint_in_the_lumped_mass(D):
    """<L u, H v> = <L v, H u> for exchange + anisotropy + demag with random cell-wise materials."""
    rng = np.random.default_rng(6)
    n, dx = _cells(D, 6, 5), (2e-9, 3e-9, 4e-9)
    p = Problem(n, dx, rng.uniform(1e5, 8e5, n), rng.uniform(0.5e-11, 2e-11, n), rng.uniform(1e4, 5e5, n),
                (0.36, 0.48, 0.8), 2.211e5, 0.1, TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO, basis=D)
    u, v = (rng.standard_normal((3,) + p.node_shape) for _ in range(2))
    L = p.L
    a = np.sum(L * np.sum(u * llg.effective_field(p, v), axis=0))
    b = np.sum(L * np.sum(v * llg.effective_field(p, u), axis=0))
    assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))
    # demag energy of any state is non-negative
    pd = Problem(n, dx, p.Ms, p.A, p.Ku, p.ku_axis, p.gamma, p.alpha, TERM_DEMAG, p.Nt, basis=D)
    assert -0.5 * np.sum(L * np.sum(u * llg.effective_field(pd, u), axis=0)) > 0


def test_demag_through_the_direct_sum_on_a_film():
    rng = np.random.default_rng(7)
    n, dx = (5, 4, 1), (2e-9, 3e-9, 4e-9)
    p = Problem(n, dx, rng.uniform(1e5, 8e5, n), np.zeros(n), np.zeros(n), terms=TERM_DEMAG, basis=2)
    m = rng.standard_normal((3,) + p.node_shape)
    assert np.allclose(llg.effective_field(p, m), llg.effective_field(p, m, demag_direct=True), rtol=1e-12, atol=1e-6)
