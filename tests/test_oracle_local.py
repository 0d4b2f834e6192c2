"""Pins for oracle/local_fields.py (C3 of SURVEY.md §8(c))."""
import itertools

import numpy as np
import pytest

from oracle import local_fields as lf
from oracle import mesh
from oracle.llg import Problem, effective_field, TERM_EXCHANGE, TERM_ANISO, TERM_ZEEMAN

MU0 = 4e-7 * np.pi


def node_coords(n_cells, dx):
    ax = [np.arange(n + 1) * d for n, d in zip(n_cells, dx)]
    return np.meshgrid(*ax, indexing="ij")


def test_uniform_m_has_zero_exchange_field():
    rng = np.random.default_rng(0)
    n, dx = (5, 4, 3), (1e-9, 2e-9, 1.5e-9)
    A = rng.uniform(1e-12, 2e-11, n)
    Ms = rng.uniform(1e5, 8e5, n)
    m = np.broadcast_to(np.array([0.6, 0.0, 0.8])[:, None, None, None], (3,) + mesh.n_nodes(n)).copy()
    H = lf.field_from_variation(lf.variation_exchange(m, A, dx), mesh.lumped_mass(Ms, dx))
    scale = 2 * A.max() / (MU0 * Ms.min() * min(dx) ** 2)
    assert np.abs(H).max() <= 1e-14 * scale


def test_uniform_external_field_is_returned_exactly_at_every_node():
    rng = np.random.default_rng(1)
    n, dx = (4, 3, 2), (2e-9, 2e-9, 5e-9)
    Ms = rng.uniform(1e5, 8e5, n)
    h = np.array([1e3, -2e4, 5e4])
    hn = np.broadcast_to(h[:, None, None, None], (3,) + mesh.n_nodes(n))
    H = lf.field_from_variation(lf.variation_zeeman(hn, Ms, dx), mesh.lumped_mass(Ms, dx))
    assert np.allclose(H, hn, rtol=1e-14, atol=0)


def test_uniform_m_parallel_to_axis_gives_textbook_anisotropy_field():
    n, dx = (3, 3, 2), (2e-9, 2e-9, 2e-9)
    Ms, Ku = 8e5, 5e5
    k = np.array([0.0, 0.6, 0.8])
    m = np.broadcast_to(k[:, None, None, None], (3,) + mesh.n_nodes(n)).copy()
    H = lf.field_from_variation(lf.variation_uniaxial(m, np.full(n, Ku), k, dx),
                                mesh.lumped_mass(np.full(n, Ms), dx))
    expect = 2 * Ku / (MU0 * Ms) * k
    assert np.allclose(H, expect[:, None, None, None], rtol=1e-13)
    # m perpendicular to k: zero field
    mp = np.broadcast_to(np.array([1.0, 0, 0])[:, None, None, None], m.shape).copy()
    H = lf.field_from_variation(lf.variation_uniaxial(mp, np.full(n, Ku), k, dx),
                                mesh.lumped_mass(np.full(n, Ms), dx))
    assert np.abs(H).max() < 1e-9


def test_helix_closed_form_energy_and_field():
    # m = (cos kx, sin kx, 0) sampled on nodes, uniform A:
    #   E_h = A V_total 4 sin^2(k dx/2)/dx^2,  interior H = -(2A/mu0 Ms) 4 sin^2(k dx/2)/dx^2 m
    n, dx = (16, 3, 2), (2e-9, 3e-9, 1e-9)
    A, Ms = 1.3e-11, 8e5
    kx = 2 * np.pi / (10.5 * dx[0])
    X, _, _ = node_coords(n, dx)
    m = np.stack([np.cos(kx * X), np.sin(kx * X), np.zeros_like(X)])
    lam = 4 * np.sin(kx * dx[0] / 2) ** 2 / dx[0] ** 2
    Vtot = np.prod(n) * np.prod(dx)
    E = lf.energy_exchange(m, np.full(n, A), dx)
    assert np.isclose(E, A * Vtot * lam, rtol=1e-13)
    assert np.isclose(lam, kx ** 2, rtol=0.05)             # -> A k^2 V, second order
    H = lf.field_from_variation(lf.variation_exchange(m, np.full(n, A), dx),
                                mesh.lumped_mass(np.full(n, Ms), dx))
    expect = -(2 * A / (MU0 * Ms)) * lam * m
    # nodes interior in x; y/z boundaries are fine because m does not vary there
    assert np.allclose(H[:, 1:-1], expect[:, 1:-1], rtol=1e-12, atol=1e-6)


def test_energy_identity():
    # sum_c A_c tr(m_loc^T K m_loc) = -1/2 sum_n L_n m_n . H^ex_n
    rng = np.random.default_rng(2)
    n, dx = (4, 3, 3), (1e-9, 2e-9, 3e-9)
    A = rng.uniform(1e-12, 2e-11, n)
    Ms = rng.uniform(1e5, 8e5, n)
    m = rng.standard_normal((3,) + mesh.n_nodes(n))
    L = mesh.lumped_mass(Ms, dx)
    H = lf.field_from_variation(lf.variation_exchange(m, A, dx), L)
    assert np.isclose(lf.energy_exchange(m, A, dx), -0.5 * np.sum(L * np.sum(m * H, axis=0)), rtol=1e-13)


def test_one_dimensional_reduction():
    # m varying along one axis only -> (m_{i+1} - 2 m_i + m_{i-1})/dx^2 at interior nodes
    rng = np.random.default_rng(3)
    for axis in range(3):
        n = [3, 3, 3]
        n[axis] = 9
        dx = (1.5e-9, 2e-9, 2.5e-9)
        A, Ms = 1e-11, 5e5
        prof = rng.standard_normal((3, n[axis] + 1))
        shape = [1, 1, 1]
        shape[axis] = n[axis] + 1
        m = np.broadcast_to(prof.reshape([3] + shape), (3,) + mesh.n_nodes(n)).copy()
        H = lf.field_from_variation(lf.variation_exchange(m, np.full(n, A), dx),
                                    mesh.lumped_mass(np.full(n, Ms), dx))
        lap = (prof[:, 2:] - 2 * prof[:, 1:-1] + prof[:, :-2]) / dx[axis] ** 2
        Hline = np.moveaxis(H, axis + 1, 1)[:, 1:-1, 1, 1]
        assert np.allclose(Hline, 2 * A / (MU0 * Ms) * lap, rtol=1e-12)
        # also identical on the boundary faces of the other two axes (natural BC)
        Hface = np.moveaxis(H, axis + 1, 1)[:, 1:-1, 0, 0]
        assert np.allclose(Hface, 2 * A / (MU0 * Ms) * lap, rtol=1e-12)


def test_plane_wave_symbol():
    n, dx = (8, 7, 6), (2e-9, 3e-9, 2.5e-9)
    A, Ms = 1.3e-11, 8e5
    k = np.array([0.9e9, -0.4e9, 0.7e9])
    X, Y, Z = node_coords(n, dx)
    ph = k[0] * X + k[1] * Y + k[2] * Z
    m = np.stack([np.cos(ph), np.sin(ph), 0.3 * np.cos(ph + 0.4)])
    H = lf.field_from_variation(lf.variation_exchange(m, np.full(n, A), dx),
                                mesh.lumped_mass(np.full(n, Ms), dx))
    sym = 0.0
    for d in range(3):
        t = -4 * np.sin(k[d] * dx[d] / 2) ** 2 / dx[d] ** 2
        for e in range(3):
            if e != d:
                t *= (2 + np.cos(k[e] * dx[e])) / 3
        sym += t
    inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))
    assert np.allclose(H[inner], 2 * A / (MU0 * Ms) * sym * m[inner], rtol=1e-11, atol=1e-4)


def _hat(s):
    return np.maximum(0.0, 1.0 - np.abs(s))


def _dhat(s):
    return np.where(np.abs(s) < 1, -np.sign(s), 0.0)


@pytest.mark.parametrize("n,dx", [((4, 3, 2), (1.0, 1.5, 0.5)), ((2, 2, 1), (2e-9, 3e-9, 5e-9))])
def test_brute_force_global_assembly_by_quadrature(n, dx):
    """Assemble Eq. (17) with global hat functions phi_n(x) = prod_d hat(x_d/dx_d - n_d) (Eq. 11)
    and 3-point Gauss quadrature cell by cell; compare all three local terms."""
    rng = np.random.default_rng(4)
    dx = np.array(dx)
    nn = mesh.n_nodes(n)
    A = rng.uniform(0.5, 2.0, n) * 1e-11
    Ms = rng.uniform(1e5, 8e5, n)
    Ku = rng.uniform(1e4, 5e5, n)
    kax = np.array([0.36, 0.48, 0.8])
    m = rng.standard_normal((3,) + nn)
    hext = rng.standard_normal((3,) + nn) * 1e4
    g = 0.5 + 0.5 * np.array([-np.sqrt(3 / 5), 0.0, np.sqrt(3 / 5)])
    gw = 0.5 * np.array([5 / 9, 8 / 9, 5 / 9])
    nodes = list(itertools.product(*[range(k) for k in nn]))
    dE_ex = np.zeros((3,) + nn)
    dE_an = np.zeros((3,) + nn)
    dE_ze = np.zeros((3,) + nn)
    lump = np.zeros(nn)
    for c in itertools.product(*[range(k) for k in n]):
        V = dx.prod()
        for (a, wa), (b, wb), (cc, wc) in itertools.product(zip(g, gw), repeat=3):
            w = wa * wb * wc * V
            s = np.array(c) + np.array([a, b, cc])          # x / dx at the quadrature point
            # values and gradients of all global basis functions at the point
            phi = {}
            gphi = {}
            for nd in nodes:
                h = [_hat(s[d] - nd[d]) for d in range(3)]
                if h[0] * h[1] * h[2] == 0:
                    continue
                phi[nd] = h[0] * h[1] * h[2]
                gphi[nd] = np.array([_dhat(s[d] - nd[d]) / dx[d] * h[(d + 1) % 3] * h[(d + 2) % 3]
                                     for d in range(3)])
            mh = sum(m[(slice(None),) + nd] * v for nd, v in phi.items())
            hh = sum(hext[(slice(None),) + nd] * v for nd, v in phi.items())
            gm = sum(np.outer(m[(slice(None),) + nd], v) for nd, v in gphi.items())  # [j, d]
            for nd in phi:
                idx = (slice(None),) + nd
                dE_ex[idx] += w * 2 * A[c] * gm @ gphi[nd]
                dE_an[idx] += w * (-2 * Ku[c]) * (mh @ kax) * kax * phi[nd]
                dE_ze[idx] += w * (-MU0 * Ms[c]) * hh * phi[nd]
                lump[nd] += w * MU0 * Ms[c] * phi[nd]
    assert np.allclose(lump, mesh.lumped_mass(Ms, dx), rtol=1e-13)
    for got, ref in ((lf.variation_exchange(m, A, dx), dE_ex),
                     (lf.variation_uniaxial(m, Ku, kax, dx), dE_an),
                     (lf.variation_zeeman(hext, Ms, dx), dE_ze)):
        assert np.allclose(got, ref, rtol=1e-12, atol=1e-13 * np.abs(ref).max())


def test_vacuum_nodes_get_zero_field():
    n, dx = (3, 2, 2), (1e-9, 1e-9, 1e-9)
    Ms = np.full(n, 8e5)
    Ms[0] = 0.0       # first slab of cells is vacuum -> nodes n1 = 0 have L = 0
    p = Problem(n, dx, Ms, np.full(n, 1e-11), np.full(n, 1e5), terms=TERM_EXCHANGE | TERM_ANISO | TERM_ZEEMAN)
    m = np.random.default_rng(5).standard_normal((3,) + mesh.n_nodes(n))
    H = effective_field(p, m, np.array([0.0, 0.0, 1e4]))
    assert np.all(np.isfinite(H)) and np.all(H[:, 0] == 0.0) and np.any(H[:, 1] != 0.0)


def test_exchange_jump_condition_two_phase():
    """Eq. (6): in the static 1-D two-phase solution of A m'' = 0 the discrete
    field vanishes at the interface node iff A1 m1' = A2 m2' (piecewise-linear profile)."""
    n, dx = (8, 1, 1), (1e-9, 1e-9, 1e-9)
    A = np.full(n, 1e-11)
    A[4:] = 3e-11
    s1 = 0.03
    s2 = s1 * A[0, 0, 0] / A[7, 0, 0]
    x = np.arange(9.0)
    th = np.where(x <= 4, s1 * (x - 4), s2 * (x - 4))        # small-angle profile, exact for linear comps
    m = np.zeros((3, 9, 2, 2))
    m[0] = 1.0
    m[1] = th[:, None, None]
    H = lf.field_from_variation(lf.variation_exchange(m, A, dx), mesh.lumped_mass(np.full(n, 8e5), dx))
    assert np.abs(H[1, 1:-1]).max() < 1e-9 * 2 * 3e-11 / (MU0 * 8e5 * 1e-18)
    # violating the jump condition leaves a field at the interface node only
    th_bad = s1 * (x - 4)
    m[1] = th_bad[:, None, None]
    H = lf.field_from_variation(lf.variation_exchange(m, A, dx), mesh.lumped_mass(np.full(n, 8e5), dx))
    assert np.abs(H[1, 4]).min() > 1.0 and np.abs(H[1, [1, 2, 3, 5, 6, 7]]).max() < 1e-6
