"""Further local energy terms through the same mass-lumped weak form (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

PAPER.md:171: "The proposed method is applicable to any energy contribution whose density depends
solely on the magnetization and its first-order spatial derivatives, such as Zeeman energy,
crystalline anisotropies, and both symmetric and antisymmetric exchange interactions."  The paper
writes out the symmetric exchange only (Eq. 3); this file adds, through Eqs. (17)-(22) unchanged
(element contributions summed into the nodes, H = -dE / L):

  antisymmetric exchange (DMI)    E = int D  sum_{a,d,b} T[a,d,b] m_a d_d m_b  dx
      bulk          T = Levi-Civita symbol              (density D m . curl m)
      interfacial   T[n,d,d] = +1, T[d,d,n] = -1 for the two in-plane axes d, n = film normal
                    (density D [m_n div m - (m . grad) m_n])
      dE_{c+i,a} += D_c sum_{i'} sum_{d,b} (T[a,d,b] G^d[i,i'] + T[b,d,a] G^d[i',i]) m_{c+i',b}
      with the element matrices G^d[i,i'] = int_cell phi_i d_d phi_i' dx (exact for Eq. 12).
  cubic anisotropy                E = int Kc (a1^2 a2^2 + a2^2 a3^2 + a3^2 a1^2) dx,  a_q = m . c_q
      (c_1, c_2, c_3 one global orthonormal frame), quartic in the trilinear m^h; integrated by the
      3-point Gauss rule per axis, which is exact for it (degree 4 per coordinate; reading C2: "Gauss
      quadrature", read as exact integration):
      dE_{c+i,j} += Kc_c sum_q w_q phi_i(x_q) de/dm_j (m^h(x_q))

  interlayer (RKKY) coupling      E = -J int_Gamma m(x, y, z_a) . m(x, y, z_b) dGamma  across a spacer between the node
      planes z_a and z_b ("interfacial energy contributions such as the RKKY coupling between two
      ferromagnetic layers"), Gamma = the whole x-y cross-section; m^h restricted to a node plane is bilinear on
      the faces, so with the 2-D element mass matrix M2[i,i'] = dx dy M1[i_x,i'_x] M1[i_y,i'_y]
      dE_{(f+i, z_a)} += -J sum_{i'} M2[i,i'] m_{(f+i', z_b)}   and the same with a and b exchanged.

Readings (rows F3): the paper names these terms without formulas; the densities above
are the standard ones; D and Kc are cell-wise like every other material parameter (Eq. 15).
"""
import numpy as np

from .mesh import LOCAL, M1, grad_phi_ref, node_view, phi_ref

# int_0^1 phi_a(x) phi_b'(x) dx for the 1-D hat functions phi_0 = 1 - x, phi_1 = x
C1 = np.array([[-0.5, 0.5], [-0.5, 0.5]])

LEVI = np.zeros((3, 3, 3))
LEVI[0, 1, 2] = LEVI[1, 2, 0] = LEVI[2, 0, 1] = 1.0
LEVI[0, 2, 1] = LEVI[2, 1, 0] = LEVI[1, 0, 2] = -1.0


def dmi_tensor(kind, normal=2):
    """T[a,d,b] of the density D sum T[a,d,b] m_a d_d m_b; kind = 'bulk' or 'interfacial'."""
    if kind == "bulk":
        return LEVI.copy()
    if kind == "interfacial":
        T = np.zeros((3, 3, 3))
        for d in range(3):
            if d != normal:
                T[normal, d, d] = 1.0       # m_n d_d m_d
                T[d, d, normal] = -1.0      # -m_d d_d m_n
        return T
    raise ValueError(kind)


def gradient_matrices(dx):
    """G[d][i1,i2,i3,i1',i2',i3'] = int_cell phi_i d_d phi_i' dx = (V/dx_d) C1[i_d,i'_d] prod_{e != d} M1[i_e,i'_e]."""
    dx = np.asarray(dx, dtype=np.float64)
    V = dx[0] * dx[1] * dx[2]
    G = np.zeros((3, 2, 2, 2, 2, 2, 2))
    for d in range(3):
        for i in LOCAL:
            for ip in LOCAL:
                t = C1[i[d], ip[d]] / dx[d]
                for e in range(3):
                    if e != d:
                        t *= M1[i[e], ip[e]]
                G[d][i + ip] = V * t
    return G


def variation_dmi(m, D, dx, kind, normal=2):
    """dE_{n,a} of the DMI energy; D cell-wise (N1,N2,N3)."""
    G = gradient_matrices(dx)
    T = dmi_tensor(kind, normal)
    dE = np.zeros_like(m, dtype=np.float64)
    for i in LOCAL:
        for ip in LOCAL:
            for a in range(3):
                for d in range(3):
                    for b in range(3):
                        w = T[a, d, b] * G[d][i + ip] + T[b, d, a] * G[d][ip + i]
                        if w != 0.0:
                            node_view(dE[a], i)[...] += D * w * node_view(m[b], ip)
    return dE


def energy_dmi(m, D, dx, kind, normal=2):
    """E = sum_c D_c sum_{i,i'} sum_{a,d,b} T[a,d,b] m_{c+i,a} G^d[i,i'] m_{c+i',b}."""
    G = gradient_matrices(dx)
    T = dmi_tensor(kind, normal)
    E = 0.0
    for i in LOCAL:
        for ip in LOCAL:
            for a in range(3):
                for d in range(3):
                    for b in range(3):
                        if T[a, d, b] != 0.0:
                            E += np.sum(D * T[a, d, b] * G[d][i + ip] * node_view(m[a], i) * node_view(m[b], ip))
    return float(E)


# 3-point Gauss-Legendre rule on [0,1]
_GX = 0.5 + 0.5 * np.array([-np.sqrt(0.6), 0.0, np.sqrt(0.6)])
_GW = 0.5 * np.array([5.0 / 9.0, 8.0 / 9.0, 5.0 / 9.0])


def _cubic_density_and_gradient(mq, axes):
    """e / Kc and d(e / Kc)/dm at field values mq (3, ...) for the orthonormal frame axes[q]."""
    c = np.asarray(axes, dtype=np.float64)
    al = [c[q, 0] * mq[0] + c[q, 1] * mq[1] + c[q, 2] * mq[2] for q in range(3)]
    e = al[0] ** 2 * al[1] ** 2 + al[1] ** 2 * al[2] ** 2 + al[2] ** 2 * al[0] ** 2
    g = np.zeros_like(mq)
    for q in range(3):
        others = sum(al[r] ** 2 for r in range(3) if r != q)
        for j in range(3):
            g[j] = g[j] + 2.0 * al[q] * others * c[q, j]
    return e, g


def _interpolate(m, x):
    """m^h at the reference point x of every cell: sum_i phi_i(x) m_{c+i}  (Eq. 14)."""
    out = 0.0
    for i in LOCAL:
        out = out + phi_ref(i, x) * node_view(m, i)
    return out


def variation_cubic(m, Kc, axes, dx):
    """dE_{n,j} of the cubic anisotropy energy; Kc cell-wise, axes = three orthonormal rows."""
    V = float(dx[0]) * float(dx[1]) * float(dx[2])
    dE = np.zeros_like(m, dtype=np.float64)
    for q1 in range(3):
        for q2 in range(3):
            for q3 in range(3):
                x = np.array([_GX[q1], _GX[q2], _GX[q3]])
                w = V * _GW[q1] * _GW[q2] * _GW[q3]
                _, g = _cubic_density_and_gradient(_interpolate(m, x), axes)
                for i in LOCAL:
                    node_view(dE, i)[...] += Kc * w * phi_ref(i, x) * g
    return dE


def hessvec_cubic(m, v, Kc, axes, dx):
    """(d^2 E / dm^2)(m) v for the cubic anisotropy energy: the derivative of variation_cubic at m in the nodal
    direction v (used by the adjoint: (dH/dm)^T b = -Hess (b / L), the Hessian being symmetric).  In the frame,
    d^2 e / da_q da_r = 2 (|a|^2 - a_q^2) delta_qr + 4 a_q a_r (1 - delta_qr)."""
    c = np.asarray(axes, dtype=np.float64)
    V = float(dx[0]) * float(dx[1]) * float(dx[2])
    out = np.zeros_like(m, dtype=np.float64)
    for q1 in range(3):
        for q2 in range(3):
            for q3 in range(3):
                x = np.array([_GX[q1], _GX[q2], _GX[q3]])
                w = V * _GW[q1] * _GW[q2] * _GW[q3]
                mq, vq = _interpolate(m, x), _interpolate(v, x)
                al = [c[q, 0] * mq[0] + c[q, 1] * mq[1] + c[q, 2] * mq[2] for q in range(3)]
                be = [c[q, 0] * vq[0] + c[q, 1] * vq[1] + c[q, 2] * vq[2] for q in range(3)]
                S = al[0] ** 2 + al[1] ** 2 + al[2] ** 2
                ab = al[0] * be[0] + al[1] * be[1] + al[2] * be[2]
                h = np.zeros_like(mq)
                for q in range(3):
                    hq = 2.0 * (S - al[q] ** 2) * be[q] + 4.0 * al[q] * (ab - al[q] * be[q])
                    for j in range(3):
                        h[j] = h[j] + hq * c[q, j]
                for i in LOCAL:
                    node_view(out, i)[...] += Kc * w * phi_ref(i, x) * h
    return out


def energy_cubic(m, Kc, axes, dx):
    V = float(dx[0]) * float(dx[1]) * float(dx[2])
    E = 0.0
    for q1 in range(3):
        for q2 in range(3):
            for q3 in range(3):
                x = np.array([_GX[q1], _GX[q2], _GX[q3]])
                w = V * _GW[q1] * _GW[q2] * _GW[q3]
                e, _ = _cubic_density_and_gradient(_interpolate(m, x), axes)
                E += np.sum(Kc * w * e)
    return float(E)


def variation_rkky(m, J, planes, dx):
    """dE_{n,j} of E = -J int m(., z_a) . m(., z_b) dGamma; planes = (z_a, z_b) node-plane indices along axis 3."""
    za, zb = int(planes[0]), int(planes[1])
    dE = np.zeros_like(m, dtype=np.float64)
    area = float(dx[0]) * float(dx[1])
    for src, dst in ((zb, za), (za, zb)):
        ms = m[:, :, :, src]                      # (3, n1, n2) on the source plane
        out = dE[:, :, :, dst]
        for i in ((0, 0), (0, 1), (1, 0), (1, 1)):
            for ip in ((0, 0), (0, 1), (1, 0), (1, 1)):
                w = -J * area * M1[i[0], ip[0]] * M1[i[1], ip[1]]
                si = tuple(slice(1, None) if i[d] else slice(0, -1) for d in range(2))
                sp = tuple(slice(1, None) if ip[d] else slice(0, -1) for d in range(2))
                out[(slice(None),) + si] += w * ms[(slice(None),) + sp]
    return dE


def energy_rkky(m, J, planes, dx):
    """E = -J sum_faces sum_{i,i'} M2[i,i'] m_{(f+i, z_a)} . m_{(f+i', z_b)}."""
    za, zb = int(planes[0]), int(planes[1])
    area = float(dx[0]) * float(dx[1])
    a, b = m[:, :, :, za], m[:, :, :, zb]
    E = 0.0
    for i in ((0, 0), (0, 1), (1, 0), (1, 1)):
        for ip in ((0, 0), (0, 1), (1, 0), (1, 1)):
            si = tuple(slice(1, None) if i[d] else slice(0, -1) for d in range(2))
            sp = tuple(slice(1, None) if ip[d] else slice(0, -1) for d in range(2))
            E += -J * area * M1[i[0], ip[0]] * M1[i[1], ip[1]] * np.sum(a[(slice(None),) + si] * b[(slice(None),) + sp])
    return float(E)


__all__ = ["variation_rkky", "energy_rkky", "hessvec_cubic", "dmi_tensor", "gradient_matrices", "variation_dmi", "energy_dmi", "variation_cubic", "energy_cubic",
           "grad_phi_ref"]
