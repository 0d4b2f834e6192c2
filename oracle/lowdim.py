"""Reduced 2-D / 1-D nodal bases for thin films and rods (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

PAPER.md:183-195 (Sec. III C, Eqs. 23-24, Fig. 4): a film meshed with one layer of cells
(N1 x N2 x 1) is described by basis functions that are constant along the third dimension,

    phi_i(x) = 1_ref(x) [1 - i_1 + (2 i_1 x_1 - x_1)] [1 - i_2 + (2 i_2 x_2 - x_2)],  i in {0,1}^2   (23)

and a rod (N1 x 1 x 1) by functions constant along the second and third dimensions,

    phi_i(x) = 1_ref(x) [1 - i + (2 i x_1 - x_1)],                                      i in {0,1}     (24)

"while maintaining full 3D integration in the weak form (17)".  D = 2 or 1 below is the number of
dimensions the basis varies in.  The degrees of freedom are the (N1+1)(N2+1) nodes of the film's
mid-plane (the paper says "N1 x N2 x 1"; a nodal basis has one more node than cells per varying axis,
PAPER.md:185) or the N1+1 nodes of the rod's axis; arrays keep three spatial axes, the reduced ones of
extent 1:

    nodal vector field   m[j, n1, n2, 0]   shape (3, N1+1, N2+1, 1)   (D = 2)
                         m[j, n1, 0, 0]    shape (3, N1+1, 1, 1)      (D = 1)
    cell fields as in 3-D: (N1, N2, 1) or (N1, 1, 1).

Everything of Sec. III A carries over with the D-dimensional multi-index (Eqs. 17-22):
  element matrices (integration over the whole 3-D cell; the integrand does not depend on the reduced
  coordinates, whose cell lengths therefore sit in V)
      K[i,i'] = V sum_{d<D} dx_d^-2 K1[i_d,i'_d] prod_{e<D, e!=d} M1[i_e,i'_e]     (no derivative along
      M[i,i'] = V prod_{d<D} M1[i_d,i'_d]                                            a reduced axis)
  lumped mass  L_n = int mu0 Ms phi_n = mu0 (V / 2^D) sum_{c containing n} Ms_c
  demag (reading C5): M_c = Ms_c 2^-D sum_i m_{c+i} (the cell mean of m^h), the same
  cell convolution, H^d_n = S(Ms o H^cell)_n / (S Ms)_n with the D-dimensional S.
"""
import itertools

import numpy as np

from . import demag as _demag
from .mesh import K1, M1, MU0


def local(D):
    """The 2^D local vertices i of Eqs. (23)-(24)."""
    return list(itertools.product((0, 1), repeat=D))


def check(n_cells, D):
    n = tuple(int(v) for v in n_cells)
    if D not in (1, 2) or any(v != 1 for v in n[D:]):
        raise ValueError("a %d-D basis needs one cell along the reduced axes, got %r" % (D, n))
    return n


def node_shape(n_cells, D):
    n = check(n_cells, D)
    return tuple(n[d] + 1 if d < D else 1 for d in range(3))


def phi_ref(i, x, D):
    """Eq. (23) / (24) at points x[..., 3] of the reference cell [0,1]^3."""
    x = np.asarray(x, dtype=np.float64)
    out = np.ones(x.shape[:-1])
    for d in range(D):
        out = out * (1 - i[d] + (2 * i[d] * x[..., d] - x[..., d]))
    return out


def grad_phi_ref(i, x, D):
    """Gradient of Eq. (23) / (24) with respect to the three reference coordinates (the components
    along the reduced axes are zero)."""
    x = np.asarray(x, dtype=np.float64)
    fac = [(1 - i[d] + (2 * i[d] * x[..., d] - x[..., d])) for d in range(D)]
    g = np.zeros(x.shape)
    for d in range(D):
        v = (2 * i[d] - 1) * np.ones(x.shape[:-1])
        for e in range(D):
            if e != d:
                v = v * fac[e]
        g[..., d] = v
    return g


def element_matrices(dx, D):
    """K[i + i'], M[i + i'] (arrays with 2 D axes of extent 2) for a cell of size dx."""
    dx = np.asarray(dx, dtype=np.float64)
    V = dx[0] * dx[1] * dx[2]
    K = np.zeros((2,) * (2 * D))
    M = np.zeros((2,) * (2 * D))
    for i in local(D):
        for ip in local(D):
            mm = V
            for d in range(D):
                mm *= M1[i[d], ip[d]]
            M[i + ip] = mm
            s = 0.0
            for d in range(D):
                t = K1[i[d], ip[d]] / dx[d] ** 2
                for e in range(D):
                    if e != d:
                        t *= M1[i[e], ip[e]]
                s += t
            K[i + ip] = V * s
    return K, M


def node_view(a, i, D):
    """Nodal array (..., N1+1, N2+1 or 1, 1) at the nodes n = c + i for every cell c."""
    sl = tuple((slice(1, None) if i[d] else slice(0, -1)) if d < D else slice(None) for d in range(3))
    return a[(Ellipsis,) + sl]


def scatter_cells_to_nodes(b, D):
    """(S b)_n = sum over the 1..2^D cells that contain node n."""
    b = np.asarray(b, dtype=np.float64)
    out = np.zeros(b.shape[:-3] + node_shape(b.shape[-3:], D))
    for i in local(D):
        node_view(out, i, D)[...] += b
    return out


def gather_nodes_to_cells(a, D):
    """(S^T a)_c = sum over the 2^D vertices of cell c."""
    a = np.asarray(a, dtype=np.float64)
    out = 0.0
    for i in local(D):
        out = out + node_view(a, i, D)
    return np.array(out)


def lumped_mass(Ms, dx, D):
    """L_n = mu0 (V / 2^D) (S Ms)_n: the integral of phi_n over one 3-D cell is V / 2^D."""
    V = float(dx[0]) * float(dx[1]) * float(dx[2])
    return MU0 * (V / 2 ** D) * scatter_cells_to_nodes(Ms, D)


def variation_exchange(m, A, dx, D):
    K, _ = element_matrices(dx, D)
    dE = np.zeros_like(m, dtype=np.float64)
    for i in local(D):
        for ip in local(D):
            node_view(dE, i, D)[...] += 2.0 * A * K[i + ip] * node_view(m, ip, D)
    return dE


def variation_uniaxial(m, Ku, axis, dx, D):
    _, M = element_matrices(dx, D)
    k = np.asarray(axis, dtype=np.float64)
    mk = k[0] * m[0] + k[1] * m[1] + k[2] * m[2]
    s = np.zeros_like(mk)
    for i in local(D):
        for ip in local(D):
            node_view(s, i, D)[...] += -2.0 * Ku * M[i + ip] * node_view(mk, ip, D)
    return k[:, None, None, None] * s[None]


def variation_zeeman(h_ext, Ms, dx, D):
    _, M = element_matrices(dx, D)
    dE = np.zeros_like(h_ext, dtype=np.float64)
    for i in local(D):
        for ip in local(D):
            node_view(dE, i, D)[...] += -MU0 * Ms * M[i + ip] * node_view(h_ext, ip, D)
    return dE


def energy_exchange(m, A, dx, D):
    K, _ = element_matrices(dx, D)
    E = 0.0
    for i in local(D):
        for ip in local(D):
            E += np.sum(A * K[i + ip] * np.sum(node_view(m, i, D) * node_view(m, ip, D), axis=0))
    return float(E)


def cell_magnetization(m, Ms, D):
    """M_c = Ms_c 2^-D sum_i m_{c+i}: the mean of m^h over the cell."""
    return Ms * gather_nodes_to_cells(m, D) / 2 ** D


def demag_field_nodes(Hc, Ms, D):
    num = scatter_cells_to_nodes(Ms * Hc, D)
    den = scatter_cells_to_nodes(Ms, D)
    out = np.zeros_like(num)
    ok = den > 0
    out[:, ok] = num[:, ok] / den[ok]
    return out


def demag_field(m, Ms, Nt, D, direct=False):
    M = cell_magnetization(m, Ms, D)
    Hc = _demag.demag_field_cells_direct(M, Nt) if direct else _demag.demag_field_cells_fft(M, Nt)
    return demag_field_nodes(Hc, Ms, D)


def expand_to_3d(m, D):
    """The same function m^h written in the full 3-D nodal basis of the mesh (the reduced basis
    functions are sums of the 3-D ones along the reduced axes): repeat the values along them."""
    reps = [1, 1, 1, 1]
    for d in range(D, 3):
        reps[d + 1] = 2
    return np.tile(m, reps)
