"""Effective field, LLG right-hand side and explicit Runge-Kutta steps (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

C6  PAPER.md:32-37, Eq. (1):
      dm/dt = -gamma/(1+alpha^2) m x H - alpha gamma/(1+alpha^2) m x (m x H)
    H = H_ex + H_an + H_zeeman + H_demag (Eq. 2 term by term).
    Integrators named at PAPER.md:286: RK4 (classical tableau) and Dormand-Prince 5(4).
    Readings (the paper is silent): m is renormalised once per accepted step, stages see the
    un-normalised intermediate states; Dormand-Prince error norm and controller as in C6.
"""
from dataclasses import dataclass, field

import numpy as np

from . import demag as _demag
from . import local_fields as _lf
from . import lowdim as _ld
from . import more_terms as _mt
from .mesh import lumped_mass, n_nodes

TERM_EXCHANGE, TERM_DEMAG, TERM_ANISO, TERM_ZEEMAN = 1, 2, 4, 8
TERM_DMI, TERM_CUBIC, TERM_RKKY = 16, 32, 64      # further local terms of PAPER.md:79, 171 (oracle/more_terms.py)


@dataclass
class Problem:
    """Static description of one simulation: mesh, cell-wise materials, scalar LLG constants."""
    n_cells: tuple
    dx: tuple
    Ms: np.ndarray            # (N1,N2,N3) A/m
    A: np.ndarray             # (N1,N2,N3) J/m
    Ku: np.ndarray            # (N1,N2,N3) J/m^3
    ku_axis: tuple = (0.0, 0.0, 1.0)
    gamma: float = 2.211e5
    alpha: float = 0.0
    terms: int = TERM_EXCHANGE | TERM_DEMAG
    _Nt: np.ndarray = field(default=None, repr=False)
    basis: int = 3            # dimensions the nodal basis varies in: 3, or 2 / 1 (Eqs. 23-24, oracle/lowdim.py)
    D: np.ndarray = None      # (N1,N2,N3) J/m^2, DMI constant (TERM_DMI)
    dmi_kind: str = "bulk"    # "bulk" or "interfacial"
    dmi_normal: int = 2       # film normal of the interfacial form
    Kc: np.ndarray = None     # (N1,N2,N3) J/m^3, cubic anisotropy constant (TERM_CUBIC)
    cubic_axes: tuple = ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0))
    rkky_J: float = 0.0       # J/m^2, interlayer coupling between the node planes rkky_planes (TERM_RKKY)
    rkky_planes: tuple = (0, 0)

    @staticmethod
    def uniform(n_cells, dx, Ms, A, Ku=0.0, **kw):
        n_cells = tuple(int(v) for v in n_cells)
        f = lambda v: np.full(n_cells, float(v)) if np.isscalar(v) else np.asarray(v, dtype=np.float64)
        return Problem(n_cells, tuple(float(v) for v in dx), f(Ms), f(A), f(Ku), **kw)

    @property
    def node_shape(self):
        return n_nodes(self.n_cells) if self.basis == 3 else _ld.node_shape(self.n_cells, self.basis)

    @property
    def L(self):
        return lumped_mass(self.Ms, self.dx) if self.basis == 3 else _ld.lumped_mass(self.Ms, self.dx, self.basis)

    @property
    def Nt(self):
        if self._Nt is None:
            self._Nt = _demag.demag_tensor(self.n_cells, self.dx)
        return self._Nt


def effective_field(p, m, h_ext=None, parts=False, demag_direct=False):
    """H_eff on nodes.  h_ext: nodal external field (3, nodes), a 3-vector, or None."""
    if p.basis != 3:
        return _effective_field_lowdim(p, m, h_ext, parts, demag_direct)
    L = p.L
    out = {}
    if p.terms & TERM_EXCHANGE:
        out["exchange"] = _lf.field_from_variation(_lf.variation_exchange(m, p.A, p.dx), L)
    if p.terms & TERM_ANISO:
        out["aniso"] = _lf.field_from_variation(_lf.variation_uniaxial(m, p.Ku, p.ku_axis, p.dx), L)
    if p.terms & TERM_ZEEMAN and h_ext is not None:
        h = np.asarray(h_ext, dtype=np.float64)
        if h.ndim == 1:
            h = np.broadcast_to(h[:, None, None, None], m.shape)
        out["zeeman"] = _lf.field_from_variation(_lf.variation_zeeman(h, p.Ms, p.dx), L)
    if p.terms & TERM_DEMAG:
        out["demag"] = _demag.demag_field(m, p.Ms, p.Nt, direct=demag_direct)
    if p.terms & TERM_DMI:
        out["dmi"] = _lf.field_from_variation(_mt.variation_dmi(m, p.D, p.dx, p.dmi_kind, p.dmi_normal), L)
    if p.terms & TERM_CUBIC:
        out["cubic"] = _lf.field_from_variation(_mt.variation_cubic(m, p.Kc, p.cubic_axes, p.dx), L)
    if p.terms & TERM_RKKY:
        out["rkky"] = _lf.field_from_variation(_mt.variation_rkky(m, p.rkky_J, p.rkky_planes, p.dx), L)
    if parts:
        return out
    H = np.zeros_like(m, dtype=np.float64)
    for v in out.values():
        H = H + v
    return H


def _effective_field_lowdim(p, m, h_ext, parts, demag_direct):
    """effective_field with the reduced basis of Eqs. (23)-(24): the same terms through oracle/lowdim.py."""
    if p.terms & (TERM_DMI | TERM_CUBIC | TERM_RKKY):
        raise NotImplementedError("DMI / cubic anisotropy / RKKY are written for the 3-D basis only")
    D = p.basis
    L = p.L
    out = {}
    if p.terms & TERM_EXCHANGE:
        out["exchange"] = _lf.field_from_variation(_ld.variation_exchange(m, p.A, p.dx, D), L)
    if p.terms & TERM_ANISO:
        out["aniso"] = _lf.field_from_variation(_ld.variation_uniaxial(m, p.Ku, p.ku_axis, p.dx, D), L)
    if p.terms & TERM_ZEEMAN and h_ext is not None:
        h = np.asarray(h_ext, dtype=np.float64)
        if h.ndim == 1:
            h = np.broadcast_to(h[:, None, None, None], m.shape)
        out["zeeman"] = _lf.field_from_variation(_ld.variation_zeeman(h, p.Ms, p.dx, D), L)
    if p.terms & TERM_DEMAG:
        out["demag"] = _ld.demag_field(m, p.Ms, p.Nt, D, direct=demag_direct)
    if parts:
        return out
    H = np.zeros_like(m, dtype=np.float64)
    for v in out.values():
        H = H + v
    return H


def cross(a, b):
    return np.stack([a[1] * b[2] - a[2] * b[1],
                     a[2] * b[0] - a[0] * b[2],
                     a[0] * b[1] - a[1] * b[0]])


def llg_from_field(p, m, H):
    """Eq. (1)."""
    gp = p.gamma / (1.0 + p.alpha ** 2)
    mxH = cross(m, H)
    return -gp * mxH - p.alpha * gp * cross(m, mxH)


def llg_rhs(p, t, m, zeeman=None):
    """f(t, m); zeeman: callable t -> h_ext (nodal array or 3-vector) or None."""
    h = zeeman(t) if zeeman is not None else None
    return llg_from_field(p, m, effective_field(p, m, h))


def normalise(m):
    """m_n / |m_n|; a zero vector stays zero (vacuum nodes are usually given m = 0; with reading
    C3(iii) they feel H = 0, so they stay at 0 for ever and never enter a cell average as NaN)."""
    nrm = np.sqrt(m[0] ** 2 + m[1] ** 2 + m[2] ** 2)
    return m / np.where(nrm > 0, nrm, 1.0)


def rk4_step(p, t, dt, m, zeeman=None, renormalise=True):
    """Classical RK4."""
    k1 = llg_rhs(p, t, m, zeeman)
    k2 = llg_rhs(p, t + 0.5 * dt, m + 0.5 * dt * k1, zeeman)
    k3 = llg_rhs(p, t + 0.5 * dt, m + 0.5 * dt * k2, zeeman)
    k4 = llg_rhs(p, t + dt, m + dt * k3, zeeman)
    y = m + dt / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
    return normalise(y) if renormalise else y


# Dormand-Prince 5(4) tableau (Dormand & Prince 1980; the "Dormand-Prince method" of PAPER.md:286)
DP_C = (0.0, 1 / 5, 3 / 10, 4 / 5, 8 / 9, 1.0, 1.0)
DP_A = (
    (),
    (1 / 5,),
    (3 / 40, 9 / 40),
    (44 / 45, -56 / 15, 32 / 9),
    (19372 / 6561, -25360 / 2187, 64448 / 6561, -212 / 729),
    (9017 / 3168, -355 / 33, 46732 / 5247, 49 / 176, -5103 / 18656),
    (35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84),
)
DP_B5 = (35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84, 0.0)
DP_B4 = (5179 / 57600, 0.0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40)


def dopri5_step(p, t, dt, m, zeeman=None, renormalise=True, rtol=1e-5, atol=1e-5):
    """One Dormand-Prince 5(4) trial step.  Returns (m_out, err_norm, accepted).

    err = y5 - y4; err_norm = sqrt(mean over all 3*nodes components of
    (err / (atol + rtol*max(|y0|, |y5|)))^2); accepted iff err_norm <= 1; on rejection m_out = m.
    The seventh stage is evaluated at the un-normalised y5 (reading C6).
    """
    k = []
    for s in range(7):
        y = m.copy()
        for j, a in enumerate(DP_A[s]):
            y = y + dt * a * k[j]
        k.append(llg_rhs(p, t + DP_C[s] * dt, y, zeeman))
    y5 = m.copy()
    err = np.zeros_like(m)
    for j in range(7):
        y5 = y5 + dt * DP_B5[j] * k[j]
        err = err + dt * (DP_B5[j] - DP_B4[j]) * k[j]
    sc = atol + rtol * np.maximum(np.abs(m), np.abs(y5))
    err_norm = float(np.sqrt(np.mean((err / sc) ** 2)))
    if err_norm <= 1.0:
        return (normalise(y5) if renormalise else y5), err_norm, True
    return m, err_norm, False


def dopri5_next_dt(dt, err_norm):
    """dt_new = dt * clip(0.9 * err_norm^(-1/5), 0.2, 5) (reading C6)."""
    if not np.isfinite(err_norm):
        return 0.2 * dt          # a non-finite trial state is a rejected step: shrink
    if err_norm == 0.0:
        return 5.0 * dt
    return dt * min(5.0, max(0.2, 0.9 * err_norm ** (-0.2)))


def energy(p, m, h_ext=None):
    """Discrete energy E = -1/2 sum L m.(H_ex + H_an + H_d) - sum L m.H_zeeman (C6 pins)."""
    parts = effective_field(p, m, h_ext, parts=True)
    L = p.L
    E = 0.0
    for name, H in parts.items():
        w = 1.0 if name == "zeeman" else 0.5
        E -= w * float(np.sum(L * np.sum(m * H, axis=0)))
    return E
