"""Mesh, basis and element matrices of the nodal finite-difference scheme (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

C1  PAPER.md:92-125 (Eqs. 8-14): cells c, nodes n = c + i, local vertex i in {0,1}^3,
    trilinear reference functions  phi_i(x) = prod_d [1 - i_d + (2 i_d - 1) x_d]  on [0,1]^3.
C2  Element matrices of the two bilinear forms that occur (exact integration; reading C2):
      stiffness  K[i,i'] = int_cell grad(phi_i) . grad(phi_i') dx
      mass       M[i,i'] = int_cell phi_i phi_i' dx
    Both factor over the three axes into the 1-D matrices of the linear "hat" functions
      K1 = [[1,-1],[-1,1]]       (int_0^1 phi_a' phi_b' dx)
      M1 = [[1/3,1/6],[1/6,1/3]] (int_0^1 phi_a  phi_b  dx)
C3  Lumped mass  L_n = int mu0 Ms^h phi_n dx = mu0 (V/8) sum_{c containing n} Ms_c
    (Eq. 22; Ms cell-wise, Eq. 15).
"""
import itertools

import numpy as np

# Reading C3(iv): mu0 = 4 pi 1e-7 exactly (pre-2019 SI value), the same literal on both sides.
MU0 = 4.0e-7 * np.pi

K1 = np.array([[1.0, -1.0], [-1.0, 1.0]])
M1 = np.array([[1.0 / 3.0, 1.0 / 6.0], [1.0 / 6.0, 1.0 / 3.0]])

# the 8 local vertices i = (i1, i2, i3) of Fig. 2(b), PAPER.md:98 (Eq. 10)
LOCAL = list(itertools.product((0, 1), repeat=3))


def n_nodes(n_cells):
    return tuple(int(n) + 1 for n in n_cells)


def phi_ref(i, x):
    """Reference basis function of Eq. (12), at points x[..., 3] in [0,1]^3."""
    x = np.asarray(x, dtype=np.float64)
    out = np.ones(x.shape[:-1])
    for d in range(3):
        out = out * (1 - i[d] + (2 * i[d] * x[..., d] - x[..., d]))
    return out


def grad_phi_ref(i, x):
    """Gradient of Eq. (12) with respect to the reference coordinates, shape x.shape."""
    x = np.asarray(x, dtype=np.float64)
    fac = [(1 - i[d] + (2 * i[d] * x[..., d] - x[..., d])) for d in range(3)]
    g = np.empty(x.shape)
    for d in range(3):
        v = (2 * i[d] - 1) * np.ones(x.shape[:-1])
        for e in range(3):
            if e != d:
                v = v * fac[e]
        g[..., d] = v
    return g


def element_matrices(dx):
    """K[i,i'], M[i,i'] as arrays indexed [i1,i2,i3,i1',i2',i3'] for a cell of size dx.

    K = V sum_d dx_d^-2 K1[i_d,i'_d] prod_{e != d} M1[i_e,i'_e],  M = V prod_d M1[i_d,i'_d].
    """
    dx = np.asarray(dx, dtype=np.float64)
    V = dx[0] * dx[1] * dx[2]
    K = np.zeros((2, 2, 2, 2, 2, 2))
    M = np.zeros((2, 2, 2, 2, 2, 2))
    for i in LOCAL:
        for ip in LOCAL:
            M[i + ip] = V * M1[i[0], ip[0]] * M1[i[1], ip[1]] * M1[i[2], ip[2]]
            s = 0.0
            for d in range(3):
                t = K1[i[d], ip[d]] / dx[d] ** 2
                for e in range(3):
                    if e != d:
                        t *= M1[i[e], ip[e]]
                s += t
            K[i + ip] = V * s
    return K, M


def node_view(a, i):
    """View of a nodal array (..., N1+1, N2+1, N3+1) at the nodes n = c + i for every cell c.

    This is the paper's "tensor slicing" of the relative index (removing the
    first [1:] or the last [:-1] value in a dimension).
    """
    sl = tuple(slice(1, None) if i[d] else slice(0, -1) for d in range(3))
    return a[(Ellipsis,) + sl]


def scatter_cells_to_nodes(b):
    """(S b)_n = sum over the 1..8 cells c that contain node n of b_c (Eq. 20 for scalars)."""
    b = np.asarray(b, dtype=np.float64)
    out = np.zeros(b.shape[:-3] + n_nodes(b.shape[-3:]))
    for i in LOCAL:
        node_view(out, i)[...] += b
    return out


def gather_nodes_to_cells(a):
    """(S^T a)_c = sum over the 8 vertices i of cell c of a_{c+i}."""
    a = np.asarray(a, dtype=np.float64)
    out = np.zeros(a.shape[:-3] + tuple(n - 1 for n in a.shape[-3:]))
    for i in LOCAL:
        out += node_view(a, i)
    return out


def lumped_mass(Ms, dx):
    """L_n = mu0 (V/8) (S Ms)_n, Eq. (22), PAPER.md:166 (int of phi_n over one cell is V/8)."""
    V = float(dx[0]) * float(dx[1]) * float(dx[2])
    return MU0 * (V / 8.0) * scatter_cells_to_nodes(Ms)
