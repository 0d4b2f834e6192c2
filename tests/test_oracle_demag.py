"""Pins for oracle/demag.py and oracle/newell_quad.c (C4, C5 of SURVEY.md §8(c))."""
import itertools

import mpmath as mp
import numpy as np
import pytest

from oracle import demag, mesh
from oracle.llg import Problem, effective_field, TERM_EXCHANGE, TERM_ANISO, TERM_DEMAG


def dipole_tensor(r, V):
    """Point-dipole limit: H = -N M with N_ij = V/(4 pi) (delta_ij/R^3 - 3 r_i r_j/R^5)."""
    r = np.asarray(r, dtype=float)
    R = np.linalg.norm(r)
    return V / (4 * np.pi) * (np.eye(3) / R ** 3 - 3 * np.outer(r, r) / R ** 5)


def full_matrix(Nt, p):
    N = np.zeros((3, 3))
    for a, (r, s) in enumerate(demag.COMPONENTS):
        N[r, s] = N[s, r] = demag.tensor_at(Nt, a, p)
    return N


def test_self_term_cube_and_trace():
    Nt = demag.demag_tensor((4, 4, 4), (2e-9, 2e-9, 2e-9))
    assert np.allclose(Nt[:3, 0, 0, 0], 1 / 3, atol=1e-15)
    assert np.allclose(Nt[3:, 0, 0, 0], 0, atol=1e-15)
    Nt = demag.demag_tensor((4, 3, 5), (1.0, 2.0, 0.5))
    tr = Nt[0] + Nt[1] + Nt[2]
    assert abs(tr[0, 0, 0] - 1.0) < 1e-15
    tr[0, 0, 0] = 0
    assert np.abs(tr).max() < 1e-15          # tr N(r != 0) = 0 (Laplace)
    # flat cell: N_zz largest; elongated along x: N_xx smallest
    assert Nt[2, 0, 0, 0] > Nt[0, 0, 0, 0] > Nt[1, 0, 0, 0]


def test_symmetries():
    Nt = demag.demag_tensor((4, 4, 4), (1.0, 1.0, 1.0))
    # cubic cells: N_xx(p1,p2,p3) = N_yy(p2,p1,p3) = N_zz(p3,p2,p1); N_xy(p1,p2,p3) = N_xz(p1,p3,p2)
    assert np.allclose(Nt[0], Nt[1].transpose(1, 0, 2), atol=1e-16)
    assert np.allclose(Nt[0], Nt[2].transpose(2, 1, 0), atol=1e-16)
    assert np.allclose(Nt[3], Nt[4].transpose(0, 2, 1), atol=1e-16)
    assert np.allclose(Nt[5], Nt[3].transpose(2, 0, 1), atol=1e-16)   # N_yz(p1,p2,p3) = N_xy(p2,p3,p1)
    # off-diagonals vanish on their symmetry planes
    assert np.abs(Nt[3][0]).max() < 1e-16 and np.abs(Nt[3][:, 0]).max() < 1e-16
    assert np.abs(Nt[4][0]).max() < 1e-16 and np.abs(Nt[4][:, :, 0]).max() < 1e-16
    assert np.abs(Nt[5][:, 0]).max() < 1e-16 and np.abs(Nt[5][:, :, 0]).max() < 1e-16
    # N(r) = N(-r) and N = N^T through tensor_at
    for p in [(1, 2, 3), (3, 1, 0), (2, 2, 1)]:
        A = full_matrix(Nt, p)
        B = full_matrix(Nt, tuple(-v for v in p))
        assert np.array_equal(A, B) and np.array_equal(A, A.T)
    # sign pattern of off-diagonals equals the dipole's
    D = dipole_tensor((1, -2, 3), 1.0)
    A = full_matrix(Nt, (1, -2, 3))
    assert np.all(np.sign(A) == np.sign(D))


@pytest.mark.parametrize("dx,order", [((1.0, 1.0, 1.0), 4), ((1.0, 1.4, 0.6), 2)])
def test_far_field_is_the_dipole_tensor(dx, order):
    n = (24, 24, 24)
    Nt = demag.demag_tensor(n, dx)
    V = np.prod(dx)
    prev = None
    for p in [(6, 4, 5), (12, 8, 10), (23, 16, 20)]:
        r = np.array(p) * np.array(dx)
        D = dipole_tensor(r, V)
        A = full_matrix(Nt, p)
        rel = np.abs(A - D).max() / np.abs(D).max()
        if prev is not None:
            assert rel < prev / 2 ** order * 1.6      # O((dx/R)^order) relative
        prev = rel
    assert rel < (2e-5 if order == 4 else 3e-3)


def _kernel(i, j, rho):
    R = np.sqrt(np.sum(rho * rho, axis=-1))
    return (float(i == j) / R ** 3 - 3 * rho[..., i] * rho[..., j] / R ** 5) / (4 * np.pi)


@pytest.mark.parametrize("p", [(2, 0, 0), (2, 1, 0), (1, 2, 2)])
def test_six_fold_numerical_integration(p):
    """N_ij(R) = 1/V int_cell int_cell' K_ij(R + r - r') d3r d3r' with the dipole kernel
    K_ij = (delta_ij/rho^3 - 3 rho_i rho_j/rho^5)/(4 pi): direct Gauss-Legendre quadrature,
    10 points per coordinate after reducing r - r' to one variable with the triangle weight."""
    dx = np.array([1.0, 0.8, 1.3])
    Nt = demag.demag_tensor((3, 3, 3), dx)
    V = dx.prod()
    x, w = np.polynomial.legendre.leggauss(10)
    # int_0^d int_0^d phi(r - r') dr dr' = int_{-d}^{d} (d - |u|) phi(u) du, split at u = 0
    pts, wts = [], []
    for d in range(3):
        u = np.concatenate([-dx[d] / 2 + dx[d] / 2 * x, dx[d] / 2 + dx[d] / 2 * x])
        ww = np.concatenate([dx[d] / 2 * w, dx[d] / 2 * w]) * (dx[d] - np.abs(u))
        pts.append(u)
        wts.append(ww)
    U = np.stack(np.meshgrid(*pts, indexing="ij"), axis=-1)
    W = wts[0][:, None, None] * wts[1][None, :, None] * wts[2][None, None, :]
    rho = U + np.array(p) * dx
    for a, (i, j) in enumerate(demag.COMPONENTS):
        val = np.sum(W * _kernel(i, j, rho)) / V
        assert abs(val - demag.tensor_at(Nt, a, p)) < 2e-10, (a, val, demag.tensor_at(Nt, a, p))


def _f_mp(x, y, z):
    x2, y2, z2 = x * x, y * y, z * z
    R = mp.sqrt(x2 + y2 + z2)
    if R == 0:
        return mp.mpf(0)
    r = mp.mpf(0)
    if x2 + z2 > 0:
        r += y / 2 * (z2 - x2) * mp.asinh(y / mp.sqrt(x2 + z2))
    if x2 + y2 > 0:
        r += z / 2 * (y2 - x2) * mp.asinh(z / mp.sqrt(x2 + y2))
    if x != 0:
        r -= x * y * z * mp.atan(y * z / (x * R))
    return r + (2 * x2 - y2 - z2) * R / 6


def _g_mp(x, y, z):
    x2, y2, z2 = x * x, y * y, z * z
    R = mp.sqrt(x2 + y2 + z2)
    if R == 0:
        return mp.mpf(0)
    r = mp.mpf(0)
    if x2 + y2 > 0:
        r += x * y * z * mp.asinh(z / mp.sqrt(x2 + y2))
    if y2 + z2 > 0:
        r += y / 6 * (3 * z2 - y2) * mp.asinh(x / mp.sqrt(y2 + z2))
    if x2 + z2 > 0:
        r += x / 6 * (3 * z2 - x2) * mp.asinh(y / mp.sqrt(x2 + z2))
    if z != 0:
        r -= z * z2 / 6 * mp.atan(x * y / (z * R))
    if y != 0:
        r -= z * y2 / 2 * mp.atan(x * z / (y * R))
    if x != 0:
        r -= z * x2 / 2 * mp.atan(y * z / (x * R))
    return r - x * y * R / 3


def _tensor_mp(a, p, dx):
    """60-digit evaluation of the same closed form at one offset (precision check of the C code)."""
    fn = [lambda X, Y, Z: _f_mp(X, Y, Z), lambda X, Y, Z: _f_mp(Y, X, Z), lambda X, Y, Z: _f_mp(Z, Y, X),
          lambda X, Y, Z: _g_mp(X, Y, Z), lambda X, Y, Z: _g_mp(X, Z, Y), lambda X, Y, Z: _g_mp(Y, Z, X)][a]
    d = [mp.mpf(v) for v in dx]
    s = mp.mpf(0)
    for i, j, k in itertools.product((-1, 0, 1), repeat=3):
        w = (-2 if i == 0 else 1) * (-2 if j == 0 else 1) * (-2 if k == 0 else 1)
        s += w * fn((p[0] + i) * d[0], (p[1] + j) * d[1], (p[2] + k) * d[2])
    return -s / (4 * mp.pi * d[0] * d[1] * d[2])


def test_quad_precision_is_sufficient_far_away():
    """fp64 would lose every digit here; the __float128 code must agree with a
    60-digit evaluation to 1e-15 relative at R ~ 440 cells."""
    mp.mp.dps = 60
    n, dx = (260, 2, 260), (2e-9, 2e-9, 2e-9)
    Nt = demag.demag_tensor(n, dx)
    for p in [(255, 1, 255), (100, 0, 3), (259, 1, 0), (17, 1, 200)]:
        for a in range(6):
            ref = _tensor_mp(a, p, dx)
            got = Nt[(a,) + p]
            assert abs(got - float(ref)) <= 1e-15 * abs(float(ref)) + 1e-30, (p, a, got, float(ref))
    # film cells (config 3 shape), non-cubic
    Nt = demag.demag_tensor((40, 40, 1), (2e-9, 2e-9, 5e-9))
    for p in [(0, 0, 0), (1, 0, 0), (39, 38, 0), (5, 20, 0)]:
        for a in range(6):
            ref = float(_tensor_mp(a, p, (2e-9, 2e-9, 5e-9)))
            assert abs(Nt[(a,) + p] - ref) <= 1e-15 * abs(ref) + 1e-30


@pytest.mark.parametrize("n,dx", [((3, 3, 3), (1.0, 1.0, 1.0)), ((4, 3, 2), (1.0, 1.5, 0.7)),
                                  ((6, 5, 1), (2.0, 2.0, 5.0)), ((5, 1, 1), (1.0, 2.0, 3.0))])
def test_fft_convolution_equals_direct_sum(n, dx):
    rng = np.random.default_rng(0)
    Nt = demag.demag_tensor(n, dx)
    M = rng.standard_normal((3,) + n)
    Hd = demag.demag_field_cells_direct(M, Nt)
    Hf = demag.demag_field_cells_fft(M, Nt)
    assert np.abs(Hd - Hf).max() < 1e-13 * np.abs(Hd).max() * 10


def test_direct_sum_matches_explicit_pair_loop():
    """The vectorised direct sum against the literal double loop H_c = -sum_c' N(c-c') M_c'."""
    rng = np.random.default_rng(1)
    n, dx = (3, 2, 2), (1.0, 1.2, 0.9)
    Nt = demag.demag_tensor(n, dx)
    M = rng.standard_normal((3,) + n)
    H = np.zeros_like(M)
    cells = list(itertools.product(*[range(k) for k in n]))
    for c in cells:
        for cp in cells:
            N = full_matrix(Nt, tuple(a - b for a, b in zip(c, cp)))
            H[(slice(None),) + c] -= N @ M[(slice(None),) + cp]
    assert np.allclose(H, demag.demag_field_cells_direct(M, Nt), rtol=1e-13, atol=1e-15)


def test_point_dipole_sum_for_well_separated_cells():
    """Two magnetised cells 9 cells apart in an otherwise empty 10x1x1 row: the field at one
    from the other is the point-dipole field to the far-field error O((dx/R)^4)."""
    n, dx = (10, 1, 1), (1.0, 1.0, 1.0)
    Nt = demag.demag_tensor(n, dx)
    M = np.zeros((3,) + n)
    M[:, 0, 0, 0] = [0.3, -0.5, 0.8]
    H = demag.demag_field_cells_fft(M, Nt)
    r = np.array([9.0, 0, 0])
    mom = M[:, 0, 0, 0]
    Hdip = (3 * r * (mom @ r) / 9.0 ** 5 - mom / 9.0 ** 3) / (4 * np.pi)
    assert np.allclose(H[:, 9, 0, 0], Hdip, rtol=5e-4)


def test_uniform_cube_magnetometric_factor():
    # mean cell field of a uniformly magnetised cube is exactly -M/3 in each direction
    n, dx = (3, 3, 3), (2e-9, 2e-9, 2e-9)
    Nt = demag.demag_tensor(n, dx)
    for j in range(3):
        M = np.zeros((3,) + n)
        M[j] = 8e5
        H = demag.demag_field_cells_fft(M, Nt)
        assert abs(H[j].mean() / 8e5 + 1 / 3) < 1e-15
        # L-weighted nodal mean of the nodal field is the same number
        p = Problem.uniform(n, dx, 8e5, 1e-11, terms=TERM_DEMAG)
        m = np.zeros((3,) + mesh.n_nodes(n))
        m[j] = 1.0
        Hn = effective_field(p, m)
        L = p.L
        assert abs(np.sum(L * Hn[j]) / L.sum() / 8e5 + 1 / 3) < 1e-15


def test_node_cell_averaging():
    rng = np.random.default_rng(2)
    n = (3, 2, 2)
    Ms = rng.uniform(1e5, 8e5, n)
    # cell mean of a trilinear function is the mean of its 8 vertex values: check on x*y*z
    X, Y, Z = np.meshgrid(*[np.arange(k + 1.0) for k in n], indexing="ij")
    fld = np.stack([X * Y * Z, X + Y, np.ones_like(X)])
    Mc = demag.cell_magnetization(fld, Ms)
    cx, cy, cz = np.meshgrid(*[np.arange(k) + 0.5 for k in n], indexing="ij")
    assert np.allclose(Mc[0], Ms * cx * cy * cz) and np.allclose(Mc[1], Ms * (cx + cy)) and np.allclose(Mc[2], Ms)
    # uniform cell field is returned unchanged at every node, whatever Ms is
    Hc = np.broadcast_to(np.array([1.0, -2.0, 3.0])[:, None, None, None], (3,) + n)
    Hn = demag.demag_field_nodes(Hc, Ms)
    assert np.allclose(Hn, np.array([1.0, -2.0, 3.0])[:, None, None, None], rtol=1e-14)
    # uniform Ms: plain mean over the existing cells
    Hc = rng.standard_normal((3,) + n)
    Hn = demag.demag_field_nodes(Hc, np.full(n, 5e5))
    assert np.isclose(Hn[0, 0, 0, 0], Hc[0, 0, 0, 0])
    assert np.isclose(Hn[1, 1, 1, 1], Hc[1, :2, :2, :2].mean())
    assert np.isclose(Hn[2, 1, 0, 0], Hc[2, :2, 0, 0].mean())


def test_L_weighted_self_adjointness_and_positive_energy():
    """<L u, H v> = <L v, H u> for H = exchange + anisotropy + demag with random cell-wise
    Ms, A, Ku (C5: the reading of the cell->node average that keeps L o H symmetric)."""
    rng = np.random.default_rng(3)
    n, dx = (4, 3, 2), (2e-9, 3e-9, 2.5e-9)
    p = Problem(n, dx, rng.uniform(1e5, 8e5, n), rng.uniform(1e-12, 2e-11, n), rng.uniform(1e4, 5e5, n),
                ku_axis=(0.6, 0.0, 0.8), terms=TERM_EXCHANGE | TERM_ANISO | TERM_DEMAG)
    u = rng.standard_normal((3,) + mesh.n_nodes(n))
    v = rng.standard_normal((3,) + mesh.n_nodes(n))
    L = p.L
    a = np.sum(L * np.sum(u * effective_field(p, v), axis=0))
    b = np.sum(L * np.sum(v * effective_field(p, u), axis=0))
    assert abs(a - b) < 1e-14 * max(abs(a), abs(b)) * 10
    pd = Problem(n, dx, p.Ms, p.A, p.Ku, terms=TERM_DEMAG)
    a = np.sum(L * np.sum(u * effective_field(pd, v), axis=0))
    b = np.sum(L * np.sum(v * effective_field(pd, u), axis=0))
    assert abs(a - b) < 1e-13 * max(abs(a), abs(b))
    assert -0.5 * np.sum(L * np.sum(u * effective_field(pd, u), axis=0)) > 0   # demag energy >= 0


def test_tensor_at_listed_offsets_matches_table_and_dipole_limit():
    """demag_tensor_at (offset-by-offset evaluation used by the full-size sampled GPU checks)
    equals the table with the parity rules of tensor_at, and at a separation far outside any
    table it tends to the point-dipole tensor (independent of the table code path)."""
    dx = (2.0, 3.0, 2.5)
    Nt = demag.demag_tensor((6, 5, 7), dx)
    offs = [(0, 0, 0), (1, 0, 0), (-1, 2, -3), (5, -4, 6), (-5, -4, -6), (0, 3, -2)]
    T = demag.demag_tensor_at(offs, dx)
    for k, p in enumerate(offs):
        for a in range(6):
            assert abs(T[k, a] - demag.tensor_at(Nt, a, p)) <= 1e-16   # summation order only
    p = (300, -170, 410)
    T = demag.demag_tensor_at([p], dx)[0]
    D = dipole_tensor(np.array(p) * np.array(dx), np.prod(dx))
    A = np.zeros((3, 3))
    for a, (r, s) in enumerate(demag.COMPONENTS):
        A[r, s] = A[s, r] = T[a]
    assert np.abs(A - D).max() <= 1e-4 * np.abs(D).max()
    assert abs(np.trace(A)) <= 1e-9 * np.abs(D).max()


def test_tensor_table_of_a_smaller_grid_is_a_sub_block():
    """N(p) depends on the offset and the cell size only (tests/_sides.py slices the table of the
    largest config-4 grid for the smaller ones)."""
    dx = (2e-9, 3e-9, 2.5e-9)
    big = demag.demag_tensor((8, 7, 6), dx)
    small = demag.demag_tensor((5, 4, 3), dx)
    assert np.array_equal(big[:, :5, :4, :3], small)
