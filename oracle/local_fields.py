"""Local effective-field terms through the mass-lumped weak form (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

PAPER.md:136-169, Eqs. (17)-(22): for every cell c the variation of the energy with respect
to the 8x3 nodal values of that cell is a linear map F_{i,j} (the element matrix), the
cell contributions are summed into the nodes n = c + i (Eqs. 19-20), and the field is
H_{n,j} = -dE_{n,j} / L_n with the lumped mass L_n (Eq. 22).  The loops below run over the
local indices i, i' exactly as Eqs. (19)-(20) are written; the cell index c is the array axis
("parallel evaluation over the cell index c").

Energies:
  exchange    E = int A (grad m)^2                      (Eq. 3)
              dE_{c+i}  += 2 A_c sum_i' K[i,i'] m_{c+i'}
  uniaxial    E = -int Ku (m.k)^2   (reading C3(i); the paper names the term only)
              dE_{c+i}  += -2 Ku_c sum_i' M[i,i'] (m_{c+i'}.k) k
  Zeeman      E = -int mu0 Ms m.H_ext, H_ext nodal (Eq. 21 lists nodal fields as arguments)
              dE_{c+i}  += -mu0 Ms_c sum_i' M[i,i'] H_ext_{c+i'}
"""
import numpy as np

from .mesh import LOCAL, MU0, element_matrices, node_view


def variation_exchange(m, A, dx):
    """dE_{n,j} for the exchange energy; A is cell-wise (N1,N2,N3)."""
    K, _ = element_matrices(dx)
    dE = np.zeros_like(m, dtype=np.float64)
    for i in LOCAL:
        for ip in LOCAL:
            node_view(dE, i)[...] += 2.0 * A * K[i + ip] * node_view(m, ip)
    return dE


def variation_uniaxial(m, Ku, axis, dx):
    """dE_{n,j} for E = -int Ku (m.k)^2 with one global unit vector k = axis."""
    _, M = element_matrices(dx)
    k = np.asarray(axis, dtype=np.float64)
    mk = k[0] * m[0] + k[1] * m[1] + k[2] * m[2]
    s = np.zeros_like(mk)
    for i in LOCAL:
        for ip in LOCAL:
            node_view(s, i)[...] += -2.0 * Ku * M[i + ip] * node_view(mk, ip)
    return k[:, None, None, None] * s[None]


def variation_zeeman(h_ext, Ms, dx):
    """dE_{n,j} for E = -int mu0 Ms m.H_ext with nodal H_ext (3, nodes)."""
    _, M = element_matrices(dx)
    dE = np.zeros_like(h_ext, dtype=np.float64)
    for i in LOCAL:
        for ip in LOCAL:
            node_view(dE, i)[...] += -MU0 * Ms * M[i + ip] * node_view(h_ext, ip)
    return dE


def field_from_variation(dE, L):
    """Eq. (22): H = -dE / L.  Reading C3(iii): nodes with L_n = 0 (vacuum all round) get H = 0."""
    H = np.zeros_like(dE)
    ok = L > 0
    H[:, ok] = -dE[:, ok] / L[ok]
    return H


def energy_exchange(m, A, dx):
    """E = sum_c A_c sum_j m_loc_j^T K m_loc_j  (the discrete Eq. 3)."""
    K, _ = element_matrices(dx)
    E = 0.0
    for i in LOCAL:
        for ip in LOCAL:
            E += np.sum(A * K[i + ip] * np.sum(node_view(m, i) * node_view(m, ip), axis=0))
    return float(E)
