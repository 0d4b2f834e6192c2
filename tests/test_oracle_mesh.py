"""Pins for oracle/mesh.py (C1-C3 of SURVEY.md §8(c))."""
import itertools

import numpy as np
import pytest

from oracle import mesh

GL3_X = 0.5 + 0.5 * np.array([-np.sqrt(3 / 5), 0.0, np.sqrt(3 / 5)])
GL3_W = 0.5 * np.array([5 / 9, 8 / 9, 5 / 9])


def test_reference_basis_is_nodal_and_partition_of_unity():
    # Eq. (12): phi_i(vertex i') = delta_ii', sum_i phi_i = 1
    verts = np.array(mesh.LOCAL, dtype=float)
    for a, i in enumerate(mesh.LOCAL):
        vals = mesh.phi_ref(i, verts)
        expect = np.zeros(8)
        expect[a] = 1.0
        assert np.allclose(vals, expect, atol=0)
    x = np.random.default_rng(0).random((50, 3))
    assert np.allclose(sum(mesh.phi_ref(i, x) for i in mesh.LOCAL), 1.0, atol=1e-15)
    # trilinear: value at the cell centre is 1/8
    assert np.allclose([mesh.phi_ref(i, np.array([0.5, 0.5, 0.5])) for i in mesh.LOCAL], 0.125)


def test_gradient_matches_finite_difference():
    x = np.random.default_rng(1).random((20, 3)) * 0.8 + 0.1
    h = 1e-6
    for i in mesh.LOCAL:
        g = mesh.grad_phi_ref(i, x)
        for d in range(3):
            e = np.zeros(3)
            e[d] = h
            fd = (mesh.phi_ref(i, x + e) - mesh.phi_ref(i, x - e)) / (2 * h)
            assert np.allclose(g[:, d], fd, atol=1e-9)


@pytest.mark.parametrize("dx", [(1.0, 1.0, 1.0), (2e-9, 3e-9, 5e-9), (3.125, 3.125, 3.0)])
def test_element_matrices_equal_numerical_quadrature(dx):
    # brute-force 3-point Gauss quadrature of Eq. (12) over the cell (exact for these integrands)
    dx = np.array(dx)
    V = dx.prod()
    K, M = mesh.element_matrices(dx)
    pts = np.array(list(itertools.product(GL3_X, repeat=3)))
    wts = np.array([a * b * c for a, b, c in itertools.product(GL3_W, repeat=3)])
    for i in mesh.LOCAL:
        for ip in mesh.LOCAL:
            Mq = V * np.sum(wts * mesh.phi_ref(i, pts) * mesh.phi_ref(ip, pts))
            gi = mesh.grad_phi_ref(i, pts) / dx      # physical gradient
            gp = mesh.grad_phi_ref(ip, pts) / dx
            Kq = V * np.sum(wts * np.sum(gi * gp, axis=1))
            assert abs(M[i + ip] - Mq) <= 1e-14 * V
            assert abs(K[i + ip] - Kq) <= 1e-13 * V / dx.min() ** 2


def test_element_matrix_invariants():
    dx = np.array([2.0, 3.0, 0.5])
    V = dx.prod()
    K, M = mesh.element_matrices(dx)
    K8 = K.reshape(8, 8)
    M8 = M.reshape(8, 8)
    assert np.allclose(K8.sum(axis=1), 0.0, atol=1e-14)       # constants have no gradient
    assert np.allclose(M8.sum(axis=1), V / 8.0)               # int phi_i = V/8
    assert np.allclose(K8, K8.T) and np.allclose(M8, M8.T)
    assert np.isclose(M8.sum(), V)
    ev = np.linalg.eigvalsh(K8)
    assert ev[0] > -1e-14 and np.sum(np.abs(ev) < 1e-12) == 1  # semi-definite, rank 7
    # one-point quadrature would leave K rank-deficient (reading C2): rank must be 7
    # x-coordinate function: int |grad x|^2 = V
    xs = np.array([i[0] * dx[0] for i in mesh.LOCAL])
    assert np.isclose(xs @ K8 @ xs, V)


def test_scatter_gather_are_transposes_and_counts():
    rng = np.random.default_rng(2)
    n = (4, 3, 2)
    b = rng.standard_normal(n)
    a = rng.standard_normal(mesh.n_nodes(n))
    assert np.isclose(np.sum(mesh.scatter_cells_to_nodes(b) * a),
                      np.sum(b * mesh.gather_nodes_to_cells(a)))
    cnt = mesh.scatter_cells_to_nodes(np.ones(n))
    assert cnt[0, 0, 0] == 1 and cnt[1, 0, 0] == 2 and cnt[1, 1, 0] == 4 and cnt[1, 1, 1] == 8
    assert cnt.sum() == 8 * np.prod(n)


def test_lumped_mass_total():
    # sum_n L_n = mu0 int Ms dx
    rng = np.random.default_rng(3)
    n = (3, 2, 2)
    dx = (1e-9, 2e-9, 3e-9)
    Ms = rng.uniform(1e5, 8e5, n)
    L = mesh.lumped_mass(Ms, dx)
    assert np.isclose(L.sum(), mesh.MU0 * Ms.sum() * np.prod(dx), rtol=1e-14)
    assert mesh.MU0 == 4e-7 * np.pi
