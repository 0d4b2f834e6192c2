"""Pins of oracle/more_terms.py (DMI, cubic anisotropy and RKKY interlayer coupling through the weak form,
PAPER.md:79, 171):
quadrature of Eq. 12's products, closed forms, invariants, and a brute-force global assembly that
shares nothing with the element loop (global hat functions, energy by 4-point Gauss quadrature,
gradient by central differences of that energy)."""
import itertools

import numpy as np
import pytest

from oracle import mesh
from oracle import more_terms as mt
from oracle.llg import Problem, effective_field, TERM_CUBIC, TERM_DMI, TERM_EXCHANGE
from oracle.mesh import MU0


def _gauss(npts):
    x, w = np.polynomial.legendre.leggauss(npts)
    return 0.5 + 0.5 * x, 0.5 * w


def test_gradient_matrices_equal_quadrature_of_eq12():
    """G^d[i,i'] = int_cell phi_i d_d phi_i' dx by a 3-point tensor Gauss rule on Eq. (12)."""
    dx = np.array([2.0, 3.0, 0.5])
    G = mt.gradient_matrices(dx)
    g, gw = _gauss(3)
    pts = np.array(list(itertools.product(g, repeat=3)))
    wts = np.array([a * b * c for a, b, c in itertools.product(gw, repeat=3)]) * dx.prod()
    for d in range(3):
        for i in mesh.LOCAL:
            for ip in mesh.LOCAL:
                ref = np.sum(wts * mesh.phi_ref(i, pts) * mesh.grad_phi_ref(ip, pts)[:, d] / dx[d])
                assert abs(G[d][i + ip] - ref) < 1e-14 * dx.prod()
    # sum over i' of G^d[i,i'] = int phi_i d_d(1) = 0; sum over i = int d_d phi_i' = +-V/(4 dx_d) by face
    for d in range(3):
        assert np.allclose(G[d].reshape(8, 8).sum(axis=1), 0.0, atol=1e-15)


def test_dmi_tensors():
    T = mt.dmi_tensor("bulk")
    a, b = np.array([0.3, -1.2, 0.7]), np.array([1.1, 0.4, -0.5])
    assert np.allclose(np.einsum("adb,a,b->d", T, a, b), -np.cross(a, b))      # sum_ab e_adb a_a b_b = (b x a)_d
    Ti = mt.dmi_tensor("interfacial", normal=2)
    assert Ti[2, 0, 0] == 1 and Ti[2, 1, 1] == 1 and Ti[0, 0, 2] == -1 and Ti[1, 1, 2] == -1
    assert np.count_nonzero(Ti) == 4
    for Tq in (T, Ti):                         # antisymmetric in the two magnetisation slots
        assert np.allclose(Tq, -np.transpose(Tq, (2, 1, 0)))


def _helix(n, dx, k, axis=0):
    """Bloch helix turning about `axis` and propagating along it, sampled on the nodes."""
    nn = mesh.n_nodes(n)
    x = np.arange(nn[axis]) * dx[axis]
    shape = [1, 1, 1]
    shape[axis] = nn[axis]
    ph = (k * x).reshape(shape) * np.ones(nn)
    m = np.zeros((3,) + nn)
    m[(axis + 1) % 3] = np.cos(ph)
    m[(axis + 2) % 3] = np.sin(ph)
    return m


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_bulk_dmi_helix_closed_form(axis):
    """m . curl m = -k for the Bloch helix; with nodal (linear) interpolation along the propagation
    axis the cell integral is -sin(k dx)/dx exactly, so E = -D V_total sin(k dx)/dx, and at interior
    nodes H = (2D/(mu0 Ms)) sin(k dx)/dx m."""
    n, dx = (6, 5, 4), np.array([2e-9, 3e-9, 2.5e-9])
    k, D, Ms = 2 * np.pi / 40e-9, 3e-3, 8e5
    m = _helix(n, dx, k, axis)
    Dc = np.full(n, D)
    E = mt.energy_dmi(m, Dc, dx, "bulk")
    Vtot = np.prod(np.array(n) * dx)
    s = np.sin(k * dx[axis]) / dx[axis]
    assert np.isclose(E, -D * Vtot * s, rtol=1e-12)
    p = Problem.uniform(n, dx, Ms, 0.0, terms=TERM_DMI, D=Dc)
    H = effective_field(p, m)
    inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))      # boundary nodes carry the natural boundary term
    assert np.allclose(H[inner], 2 * D / (MU0 * Ms) * s * m[inner], rtol=1e-11, atol=1e-6)


def test_interfacial_dmi_neel_cycloid_closed_form():
    """Neel cycloid m = (sin kx, 0, cos kx) in a film with normal z: m_z div m - (m.grad) m_z =
    cos(kx) k cos(kx) + sin(kx) k sin(kx) = k; with linear interpolation per cell sin(k dx)/dx."""
    n, dx = (8, 3, 2), np.array([2e-9, 2e-9, 1e-9])
    k, D = 2 * np.pi / 50e-9, 2e-3
    nn = mesh.n_nodes(n)
    x = (np.arange(nn[0]) * dx[0]).reshape(-1, 1, 1) * np.ones(nn)
    m = np.stack([np.sin(k * x), np.zeros(nn), np.cos(k * x)])
    E = mt.energy_dmi(m, np.full(n, D), dx, "interfacial", normal=2)
    assert np.isclose(E, D * np.prod(np.array(n) * dx) * np.sin(k * dx[0]) / dx[0], rtol=1e-12)


@pytest.mark.parametrize("kind", ["bulk", "interfacial"])
def test_dmi_energy_identity_and_uniform_state(kind):
    """The energy is bilinear: E = (1/2) sum m . dE; a uniform m has zero energy and zero variation
    at interior nodes (only the natural boundary term survives)."""
    rng = np.random.default_rng(11)
    n, dx = (4, 3, 3), np.array([1.0, 1.5, 0.7])
    D = rng.uniform(0.5, 2.0, n)
    m = rng.standard_normal((3,) + mesh.n_nodes(n))
    dE = mt.variation_dmi(m, D, dx, kind)
    assert np.isclose(mt.energy_dmi(m, D, dx, kind), 0.5 * np.sum(m * dE), rtol=1e-12)
    mu = np.broadcast_to(np.array([0.3, -0.5, 0.8]).reshape(3, 1, 1, 1), m.shape)
    Du = np.full(n, 1.3)
    assert abs(mt.energy_dmi(mu, Du, dx, kind)) < 1e-13
    dEu = mt.variation_dmi(mu, Du, dx, kind)
    assert np.allclose(dEu[:, 1:-1, 1:-1, 1:-1], 0.0, atol=1e-14)
    assert np.abs(dEu).max() > 1e-3            # boundary term of the Lifshitz invariant


def test_cubic_uniform_state_closed_form():
    """Uniform unit m: the weak form returns the pointwise field H = -(2Kc/(mu0 Ms)) sum_q a_q (1 - a_q^2) c_q
    at every node including corners (partition of unity), with a rotated frame."""
    n, dx = (3, 2, 2), (2e-9, 2e-9, 3e-9)
    Kc, Ms = 4.5e4, 4.8e5
    c1 = np.array([1.0, 1.0, 0.0]) / np.sqrt(2)
    c2 = np.array([-1.0, 1.0, 1.0]) / np.sqrt(3)
    c3 = np.cross(c1, c2)
    axes = np.stack([c1, c2, c3])
    mv = np.array([0.48, -0.6, 0.64])
    m = np.broadcast_to(mv.reshape(3, 1, 1, 1), (3,) + mesh.n_nodes(n)).copy()
    p = Problem.uniform(n, dx, Ms, 0.0, terms=TERM_CUBIC, Kc=np.full(n, Kc), cubic_axes=axes)
    H = effective_field(p, m)
    al = axes @ mv
    ref = -(2 * Kc / (MU0 * Ms)) * sum(al[q] * (1 - al[q] ** 2) * axes[q] for q in range(3))
    assert np.allclose(H, ref.reshape(3, 1, 1, 1), rtol=1e-12)
    # energy density of a uniform state: Kc (a1^2 a2^2 + a2^2 a3^2 + a3^2 a1^2); Kc/3 along <111>, 0 along an axis
    V = np.prod(np.array(n) * np.array(dx))
    e = al[0] ** 2 * al[1] ** 2 + al[1] ** 2 * al[2] ** 2 + al[2] ** 2 * al[0] ** 2
    assert np.isclose(mt.energy_cubic(m, np.full(n, Kc), axes, dx), Kc * V * e, rtol=1e-12)
    m111 = np.broadcast_to(((c1 + c2 + c3) / np.sqrt(3)).reshape(3, 1, 1, 1), m.shape)
    assert np.isclose(mt.energy_cubic(m111, np.full(n, Kc), axes, dx), Kc * V / 3, rtol=1e-12)
    max_ = np.broadcast_to(c2.reshape(3, 1, 1, 1), m.shape)
    assert abs(mt.energy_cubic(max_, np.full(n, Kc), axes, dx)) < 1e-30
    assert np.abs(mt.variation_cubic(max_, np.full(n, Kc), axes, dx)).max() < 1e-25


def test_cubic_quadrature_is_exact_and_frame_permutation_invariant():
    """The 3-point rule integrates the quartic density exactly: a 6-point rule gives the same energy;
    relabelling the frame axes changes nothing."""
    rng = np.random.default_rng(5)
    n, dx = (3, 2, 2), np.array([1.0, 0.8, 1.3])
    Kc = rng.uniform(0.5, 2.0, n)
    m = rng.standard_normal((3,) + mesh.n_nodes(n))
    axes = np.linalg.qr(rng.standard_normal((3, 3)))[0]
    E3 = mt.energy_cubic(m, Kc, axes, dx)
    g, gw = _gauss(6)
    E6 = 0.0
    for (a, wa), (b, wb), (c, wc) in itertools.product(zip(g, gw), repeat=3):
        x = np.array([a, b, c])
        mq = sum(mesh.phi_ref(i, x) * mesh.node_view(m, i) for i in mesh.LOCAL)
        al = np.einsum("qj,j...->q...", axes, mq)
        e = al[0] ** 2 * al[1] ** 2 + al[1] ** 2 * al[2] ** 2 + al[2] ** 2 * al[0] ** 2
        E6 += wa * wb * wc * dx.prod() * np.sum(Kc * e)
    assert np.isclose(E3, E6, rtol=1e-13)
    assert np.isclose(E3, mt.energy_cubic(m, Kc, axes[[2, 0, 1]], dx), rtol=1e-13)
    assert np.allclose(mt.variation_cubic(m, Kc, axes, dx), mt.variation_cubic(m, Kc, axes[[1, 2, 0]], dx), rtol=1e-12)


def _hat(s):
    return np.maximum(0.0, 1.0 - np.abs(s))


def _dhat(s):
    return np.where(np.abs(s) < 1, -np.sign(s), 0.0)


def _brute_energy(m, n, dx, D, T, Kc, axes):
    """E(m) of DMI + cubic anisotropy with global hat functions (Eq. 11) and a 4-point Gauss rule per
    cell and axis; nothing from oracle/more_terms.py except the constant tensor T."""
    nn = mesh.n_nodes(n)
    g, gw = _gauss(4)
    E = 0.0
    for c in itertools.product(*[range(k) for k in n]):
        lo = [slice(c[d], c[d] + 2) for d in range(3)]
        mloc = m[(slice(None),) + tuple(lo)]                                   # the 8 vertices of the cell
        for (a, wa), (b, wb), (cc, wc) in itertools.product(zip(g, gw), repeat=3):
            s = np.array([a, b, cc])
            h = [np.array([_hat(s[d]), _hat(s[d] - 1)]) for d in range(3)]          # values of the two hats per axis
            dh = [np.array([_dhat(s[d]), _dhat(s[d] - 1)]) / dx[d] for d in range(3)]
            phi = np.einsum("i,j,k->ijk", h[0], h[1], h[2])
            gphi = [np.einsum("i,j,k->ijk", dh[0], h[1], h[2]), np.einsum("i,j,k->ijk", h[0], dh[1], h[2]),
                    np.einsum("i,j,k->ijk", h[0], h[1], dh[2])]
            mh = np.einsum("aijk,ijk->a", mloc, phi)
            gm = np.array([[np.sum(mloc[b_] * gphi[d]) for b_ in range(3)] for d in range(3)])   # [d, b] = d_d m_b
            w = wa * wb * wc * np.prod(dx)
            E += w * D[c] * np.einsum("adb,a,db->", T, mh, gm)
            al = axes @ mh
            E += w * Kc[c] * (al[0] ** 2 * al[1] ** 2 + al[1] ** 2 * al[2] ** 2 + al[2] ** 2 * al[0] ** 2)
    return E


@pytest.mark.parametrize("kind", ["bulk", "interfacial"])
def test_variations_equal_finite_differences_of_a_brute_force_energy(kind):
    """dE_{n,j} of both terms against central differences, node by node, of an energy assembled with
    global hat functions and a different quadrature rule (random cell-wise D, Kc; rotated frame)."""
    rng = np.random.default_rng(21)
    n, dx = (2, 2, 1), np.array([1.0, 1.4, 0.6])
    nn = mesh.n_nodes(n)
    D = rng.uniform(0.5, 2.0, n)
    Kc = rng.uniform(0.5, 2.0, n)
    axes = np.linalg.qr(rng.standard_normal((3, 3)))[0]
    T = mt.dmi_tensor(kind, normal=2)
    m = rng.standard_normal((3,) + nn)
    got = mt.variation_dmi(m, D, dx, kind) + mt.variation_cubic(m, Kc, axes, dx)
    ref = np.zeros_like(m)
    eps = 1e-5
    for idx in itertools.product(range(3), *[range(k) for k in nn]):
        mp, mm = m.copy(), m.copy()
        mp[idx] += eps
        mm[idx] -= eps
        ref[idx] = (_brute_energy(mp, n, dx, D, T, Kc, axes) - _brute_energy(mm, n, dx, D, T, Kc, axes)) / (2 * eps)
    assert np.allclose(got, ref, rtol=1e-7, atol=1e-8 * np.abs(ref).max())


def test_dmi_operator_is_self_adjoint_in_the_lumped_inner_product():
    """<L u, H_dmi(v)> = <L v, H_dmi(u)>: the DMI field is minus the gradient of a quadratic form."""
    rng = np.random.default_rng(3)
    n, dx = (3, 3, 2), (1e-9, 2e-9, 1.5e-9)
    Ms = rng.uniform(2e5, 8e5, n)
    D = rng.uniform(1e-3, 3e-3, n)
    p = Problem(n, dx, Ms, np.zeros(n), np.zeros(n), terms=TERM_DMI, D=D, dmi_kind="interfacial")
    u = rng.standard_normal((3,) + mesh.n_nodes(n))
    v = rng.standard_normal((3,) + mesh.n_nodes(n))
    L = p.L
    a = np.sum(L * u * effective_field(p, v))
    b = np.sum(L * v * effective_field(p, u))
    assert np.isclose(a, b, rtol=1e-12)


def test_terms_add_in_effective_field():
    rng = np.random.default_rng(8)
    n, dx = (3, 2, 2), (2e-9, 2e-9, 2e-9)
    m = rng.standard_normal((3,) + mesh.n_nodes(n))
    m /= np.sqrt((m ** 2).sum(axis=0))
    kw = dict(D=np.full(n, 2e-3), Kc=np.full(n, 3e4))
    p = Problem.uniform(n, dx, 8e5, 1.3e-11, terms=TERM_EXCHANGE | TERM_DMI | TERM_CUBIC, **kw)
    parts = effective_field(p, m, parts=True)
    assert set(parts) == {"exchange", "dmi", "cubic"}
    assert np.allclose(effective_field(p, m), parts["exchange"] + parts["dmi"] + parts["cubic"])


def _two_layers(n=(4, 3, 5), spacer=(2, 3)):
    """Two magnetic layers separated by one vacuum cell layer (cells c3 = 2): node planes 2 and 3 face each other."""
    Ms = np.full(n, 8e5)
    Ms[:, :, spacer[0]:spacer[1]] = 0.0
    return Ms


def test_rkky_uniform_layers_closed_form():
    """Uniform m_a on plane z_a and m_b on plane z_b: E = -J A (m_a . m_b) exactly; the variation on plane a
    sums to -J A m_b; a corner node carries a quarter of an interior node's share."""
    from oracle.llg import TERM_RKKY
    n, dx = (4, 3, 5), np.array([2e-9, 3e-9, 1e-9])
    J, planes = 1.5e-3, (2, 3)
    nn = mesh.n_nodes(n)
    ma, mb = np.array([0.6, 0.0, 0.8]), np.array([0.0, 1.0, 0.0]) * 0.5 + np.array([0.0, 0.0, 0.5])
    m = np.zeros((3,) + nn)
    m[:, :, :, :3] = ma.reshape(3, 1, 1, 1)
    m[:, :, :, 3:] = mb.reshape(3, 1, 1, 1)
    A = n[0] * dx[0] * n[1] * dx[1]
    assert np.isclose(mt.energy_rkky(m, J, planes, dx), -J * A * (ma @ mb), rtol=1e-13)
    dE = mt.variation_rkky(m, J, planes, dx)
    assert np.allclose(dE[:, :, :, 2].sum(axis=(1, 2)), -J * A * mb, rtol=1e-13)
    assert np.allclose(dE[:, :, :, 3].sum(axis=(1, 2)), -J * A * ma, rtol=1e-13)
    assert np.all(dE[:, :, :, [0, 1, 4, 5]] == 0)
    assert np.allclose(dE[:, 1, 1, 2], -J * dx[0] * dx[1] * mb) and np.allclose(dE[:, 0, 0, 2], -J * dx[0] * dx[1] * mb / 4)
    # field on an interior interface node: H = J m_b / (mu0 Ms t), t = the half cell of magnetic material below it
    p = Problem(n, tuple(dx), _two_layers(n), np.zeros(n), np.zeros(n), terms=TERM_RKKY, rkky_J=J, rkky_planes=planes)
    H = effective_field(p, m)
    assert np.allclose(H[:, 1, 1, 2], J * mb / (MU0 * 8e5 * dx[2] / 2), rtol=1e-12)


def test_rkky_bilinear_identity_symmetry_and_brute_force():
    """E = (1/2) sum m . dE; <u, dE(v)> = <v, dE(u)>; dE against central differences of the face integral
    evaluated with 2-D hat functions and a 3-point Gauss rule per face."""
    rng = np.random.default_rng(6)
    n, dx = (3, 2, 4), np.array([1.0, 1.3, 0.7])
    J, planes = 0.9, (1, 3)
    nn = mesh.n_nodes(n)
    m, u = rng.standard_normal((3,) + nn), rng.standard_normal((3,) + nn)
    dE = mt.variation_rkky(m, J, planes, dx)
    assert np.isclose(mt.energy_rkky(m, J, planes, dx), 0.5 * np.sum(m * dE), rtol=1e-12)
    assert np.isclose(np.sum(u * dE), np.sum(m * mt.variation_rkky(u, J, planes, dx)), rtol=1e-12)
    g, gw = _gauss(3)

    def brute(mm):
        E = 0.0
        for f1 in range(n[0]):
            for f2 in range(n[1]):
                for (a, wa), (b, wb) in itertools.product(zip(g, gw), repeat=2):
                    ph = np.outer([1 - a, a], [1 - b, b])
                    va = np.einsum("jxy,xy->j", mm[:, f1:f1 + 2, f2:f2 + 2, planes[0]], ph)
                    vb = np.einsum("jxy,xy->j", mm[:, f1:f1 + 2, f2:f2 + 2, planes[1]], ph)
                    E += -J * wa * wb * dx[0] * dx[1] * (va @ vb)
        return E
    assert np.isclose(brute(m), mt.energy_rkky(m, J, planes, dx), rtol=1e-12)
    ref = np.zeros_like(m)
    for idx in itertools.product(range(3), range(nn[0]), range(nn[1]), planes):
        mp, mm_ = m.copy(), m.copy()
        mp[idx] += 1e-5
        mm_[idx] -= 1e-5
        ref[idx] = (brute(mp) - brute(mm_)) / 2e-5
    assert np.allclose(dE, ref, rtol=1e-7, atol=1e-9)
