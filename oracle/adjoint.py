"""Adjoint (vector-Jacobian) right-hand side and adjoint-state driver (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

PAPER.md:210-228, Eqs. (27)-(30): after the forward solve, the system
    dm/dt = f(t, m),           m(T) = m_output
    da/dt = -(df/dm)^T a,      a(T) = grad_y L
    du/dt = -(df/dtheta)^T a,  u(T) = 0
is integrated backwards in time and u(0) = grad_theta L.  (Eq. 29 prints the products without
the transpose; the adjoint variable multiplies the Jacobian from the left, as in the cited
neural-ODE reference 26.)  The paper delegates both products to framework autodiff
(PAPER.md:288); C7 of SURVEY.md §8(c) writes them out for theta = Ms (cell-wise):

  H = Hlin(m) + H_zeeman,  Hlin = exchange + anisotropy + demag (linear in m),
  f = -g' m x H - alpha g' m x (m x H),  g' = gamma/(1+alpha^2)

  b = (df/dH)^T a       = g' m x a - alpha g' m x (m x a)
  d = (df/dm|_H)^T a    = -g' H x a - alpha g' [(m.H) a + (a.m) H - 2 (a.H) m]
  (df/dm)^T a           = d + Hlin^T b,   Hlin^T b = L o Hlin(b / L)     (L Hlin is symmetric)
  (df/dMs_c)^T a        = - S^T[ b.H / (S Ms) ]_c
                          + sum_i b_{c+i} . mu0 (M Hext_loc)_i / L_{c+i}
                          + (S^T q)_c . Hcell_c + mbar_c . Y_c
     q = b / (S Ms),  mbar = S^T m / 8,  Hcell = -N * (Ms mbar),  Y = -N * (Ms o S^T q)

On the reduced 2-D / 1-D bases of Eqs. (23)-(24) (Problem.basis) the same formulas hold with the operators of
oracle/lowdim.py: S, S^T over the 2^D vertices of a cell, mbar = S^T m / 2^D, the reduced element matrices.
"""
import dataclasses

import numpy as np

from . import demag as _demag
from . import llg as _llg
from . import local_fields as _lf
from . import lowdim as _ld
from . import more_terms as _mt
from .mesh import (LOCAL, MU0, element_matrices, gather_nodes_to_cells, node_view,
                   scatter_cells_to_nodes)


def _basis_ops(p):
    """(local vertices, node_view, S, S^T, mass matrix M, vertices per cell) of the problem's nodal basis:
    the 3-D one (oracle/mesh.py) or the reduced one of Eqs. (23)-(24) (oracle/lowdim.py).  The formulas in
    this file's header hold for both, with 2^D vertices per cell in place of 8."""
    D = p.basis
    if D == 3:
        return LOCAL, node_view, scatter_cells_to_nodes, gather_nodes_to_cells, element_matrices(p.dx)[1], 8
    return (_ld.local(D), lambda a, i: _ld.node_view(a, i, D), lambda b: _ld.scatter_cells_to_nodes(b, D),
            lambda a: _ld.gather_nodes_to_cells(a, D), _ld.element_matrices(p.dx, D)[1], 2 ** D)


def _safe_div(num, den):
    out = np.zeros_like(num)
    ok = den > 0
    out[..., ok] = num[..., ok] / den[ok]
    return out


def adjoint_rhs(p, t, m, a, zeeman=None, pieces=None):
    """Returns (f, dadt, dudt_Ms) = (f(t,m), -(df/dm)^T a, -(df/dMs)^T a).

    pieces: optional dict that receives the summands of (df/dMs)^T a as they are added ("field",
    "zeeman", "demag_H", "demag_Y"), so that a test can state how strongly they cancel."""
    gp = p.gamma / (1.0 + p.alpha ** 2)
    al = p.alpha
    L = p.L
    local, nview, scatter, gather, M, nv = _basis_ops(p)
    SMs = scatter(p.Ms)
    h_ext = zeeman(t) if zeeman is not None else None
    if h_ext is not None:
        h_ext = np.asarray(h_ext, dtype=np.float64)
        if h_ext.ndim == 1:
            h_ext = np.broadcast_to(h_ext[:, None, None, None], m.shape)
    H = _llg.effective_field(p, m, h_ext)
    f = _llg.llg_from_field(p, m, H)

    cross = _llg.cross
    dot = lambda x, y: x[0] * y[0] + x[1] * y[1] + x[2] * y[2]
    mxa = cross(m, a)
    b = gp * mxa - al * gp * cross(m, mxa)
    d = -gp * cross(H, a) - al * gp * (dot(m, H) * a + dot(a, m) * H - 2.0 * dot(a, H) * m)

    # Hlin^T b = L o Hlin(b / L): the same field operators, without the Zeeman term
    # (exchange, anisotropy, demag, DMI and RKKY are linear in m with an L-symmetric operator; the cubic
    # anisotropy is not: H_cub = -L^-1 g(m), so (dH_cub/dm)^T b = -Hess E_cub(m) (b / L), the Hessian being symmetric)
    p_lin = dataclasses.replace(p, terms=p.terms & ~(_llg.TERM_ZEEMAN | _llg.TERM_CUBIC))
    HTb = L * _llg.effective_field(p_lin, _safe_div(b, L), None)
    if p.terms & _llg.TERM_CUBIC:
        # (0 at nodes with L = 0, like L o Hlin(b / L) above: reading C7 carries no adjoint at vacuum nodes)
        HTb = HTb - np.where(L > 0, _mt.hessvec_cubic(m, _safe_div(b, L), p.Kc, p.cubic_axes, p.dx), 0.0)
    dadt = -(d + HTb)

    # -(df/dMs)^T a
    grad = -gather(_safe_div(dot(b, H), SMs))
    if pieces is not None:
        pieces["field"] = grad.copy()
        # the same sum with every product b_j H_j taken in magnitude: b is perpendicular to m, so the
        # m-parallel part of H (most of the exchange field of a smooth m) cancels inside b . H
        pieces["field_abs"] = gather(
            _safe_div(np.abs(b[0] * H[0]) + np.abs(b[1] * H[1]) + np.abs(b[2] * H[2]), SMs))
    if (p.terms & _llg.TERM_ZEEMAN) and h_ext is not None:
        bL = _safe_div(b, L)
        zee = np.zeros_like(grad)
        for i in local:
            for ip in local:
                zee = zee + MU0 * M[i + ip] * np.sum(nview(bL, i) * nview(h_ext, ip), axis=0)
        grad = grad + zee
        if pieces is not None:
            pieces["zeeman"] = zee
    if p.terms & _llg.TERM_DEMAG:
        q = _safe_div(b, SMs)
        STq = gather(q)
        mbar = gather(m) / nv
        Hcell = _demag.demag_field_cells_fft(p.Ms * mbar, p.Nt)
        Y = _demag.demag_field_cells_fft(p.Ms * STq, p.Nt)
        grad = grad + np.sum(STq * Hcell, axis=0) + np.sum(mbar * Y, axis=0)
        if pieces is not None:
            pieces["demag_H"] = np.sum(STq * Hcell, axis=0)
            pieces["demag_Y"] = np.sum(mbar * Y, axis=0)
    return f, dadt, -grad


def adjoint_rhs_hext(p, t, m, a):
    """-(df/dh)^T a for a spatially uniform external field h added to H_ext (the design variable of
    the field-angle problem, Eqs. 31-33).

    A uniform h passes through the weak form of Eq. (21) unchanged at every node with L_n > 0 and
    gives no field at vacuum nodes (reading C3(ii), (iii)), so dH_n/dh = [L_n > 0] I and
        (df/dh)^T a = sum_{n: L_n > 0} b_n,   b = (df/dH)^T a = g' m x a - alpha g' m x (m x a)
    (b depends on m and a only).  Returns the 3-vector -(df/dh)^T a; zero without the Zeeman term."""
    if not (p.terms & _llg.TERM_ZEEMAN):
        return np.zeros(3)
    gp = p.gamma / (1.0 + p.alpha ** 2)
    mxa = _llg.cross(m, a)
    b = gp * mxa - p.alpha * gp * _llg.cross(m, mxa)
    inside = p.L > 0
    return -np.array([np.sum(b[j][inside]) for j in range(3)])


def adjoint_rhs_hnodal(p, t, m, a):
    """-(df/dh)^T a for a *nodal* external field h (3, nodes) added to H_ext through the weak form of
    Eq. (21) (SURVEY.md §8(f) row 2 lists H^ext among the design variables; reading C3(ii)).

    H^z = -L^-1 Z(h) with Z = variation_zeeman, linear in h and symmetric (an assembled mass matrix), so
        (dH^z/dh)^T b = -Z(b / L),   b = (df/dH)^T a = g' m x a - alpha g' m x (m x a),
    and -(df/dh)^T a = Z(b / L), with b / L := 0 where L_n = 0 (reading C3(iii)).  Returns a nodal
    3-vector field; zero without the Zeeman term.  For a uniform h its sum over the nodes is
    adjoint_rhs_hext."""
    if not (p.terms & _llg.TERM_ZEEMAN):
        return np.zeros_like(m)
    gp = p.gamma / (1.0 + p.alpha ** 2)
    mxa = _llg.cross(m, a)
    b = gp * mxa - p.alpha * gp * _llg.cross(m, mxa)
    if p.basis != 3:
        return _ld.variation_zeeman(_safe_div(b, p.L), p.Ms, p.dx, p.basis)
    return _lf.variation_zeeman(_safe_div(b, p.L), p.Ms, p.dx)


def adjoint_rhs_materials(p, t, m, a):
    """(-(df/dA)^T a, -(df/dKu)^T a), cell-wise (design variables A_c, Ku_c).

    A and Ku enter f only through H = -dE/L with L independent of both (Eq. 22), and dE is linear
    in them (Eqs. 19-20; oracle/local_fields.py):
        dE_{c+i} += 2 A_c sum_i' K[i,i'] m_{c+i'}            - 2 Ku_c sum_i' M[i,i'] (m_{c+i'}.k) k
    so with b = (df/dH)^T a = g' m x a - alpha g' m x (m x a) and bL = b / L (0 where L = 0)
        (df/dA_c)^T a  = -2 sum_{i,i'} K[i,i'] bL_{c+i} . m_{c+i'}
        (df/dKu_c)^T a = +2 sum_{i,i'} M[i,i'] (bL_{c+i}.k) (m_{c+i'}.k)
    Terms that are off contribute zero."""
    gp = p.gamma / (1.0 + p.alpha ** 2)
    mxa = _llg.cross(m, a)
    b = gp * mxa - p.alpha * gp * _llg.cross(m, mxa)
    bL = _safe_div(b, p.L)
    local, nview = _basis_ops(p)[:2]
    K, M = element_matrices(p.dx) if p.basis == 3 else _ld.element_matrices(p.dx, p.basis)
    k = np.asarray(p.ku_axis, dtype=np.float64)
    bk = k[0] * bL[0] + k[1] * bL[1] + k[2] * bL[2]
    mk = k[0] * m[0] + k[1] * m[1] + k[2] * m[2]
    gA = np.zeros(p.n_cells)
    gKu = np.zeros(p.n_cells)
    for i in local:
        for ip in local:
            if p.terms & _llg.TERM_EXCHANGE:
                gA += -2.0 * K[i + ip] * np.sum(nview(bL, i) * nview(m, ip), axis=0)
            if p.terms & _llg.TERM_ANISO:
                gKu += 2.0 * M[i + ip] * nview(bk, i) * nview(mk, ip)
    return -gA, -gKu


def forward_rk4(p, m0, dt, n_steps, zeeman=None, checkpoint_every=0, t0=0.0):
    """Fixed-step RK4 with renormalisation; returns (m_T, {step index: m}) (C8)."""
    m = m0.copy()
    ckpt = {}
    for s in range(n_steps):
        if checkpoint_every and s % checkpoint_every == 0:
            ckpt[s] = m.copy()
        m = _llg.rk4_step(p, t0 + s * dt, dt, m, zeeman, renormalise=True)
    return m, ckpt


def backward_rk4(p, mT, aT, dt, n_steps, zeeman=None, checkpoints=None, t0=0.0, a_jumps=None,
                 with_hext=False, with_materials=False, with_hnodal=False):
    """Integrate Eq. (29) from T = t0 + n_steps dt back to t0 with RK4 steps of -dt.

    State (m, a, u); m is renormalised after every step and replaced by the stored forward
    value whenever a checkpoint index is reached (reading C8).  Returns (m0, a0, u0);
    u0 = dJ/dMs per cell (Eq. 30).

    Objectives at several times ("adding appropriate terms depending on m(T_i)"):
    for L = L_T(m(T)) + sum_i L_i(m(T_i)), T_i = t0 + s_i dt, pass aT = grad L_T and
    a_jumps = {s_i: grad_m L_i(m(T_i))}; the adjoint variable takes the jump a += a_jumps[s_i]
    when the backward integration arrives at T_i (the term of L_i enters the adjoint equation as
    a delta function in time).

    with_hext: also integrate du_h/dt = -(df/dh)^T a (adjoint_rhs_hext) with u_h(T) = 0 and return
    (m0, a0, u0, u_h(0)); u_h(0) = dL/dh for a uniform external field h.
    with_materials: also integrate (u_A, u_Ku) with adjoint_rhs_materials and append
    (u_A(0), u_Ku(0)) = (dL/dA, dL/dKu) per cell to the returned tuple.
    with_hnodal: also integrate u_hn with adjoint_rhs_hnodal and append u_hn(0) = dL/dh per node and
    component for a time-constant nodal external field h (last in the returned tuple).
    """
    m, a = mT.copy(), aT.copy()
    u = np.zeros(p.n_cells)
    h = -dt

    uh = np.zeros(3)

    def F(t, m_, a_):
        r = adjoint_rhs(p, t, m_, a_, zeeman)
        return r + (adjoint_rhs_hext(p, t, m_, a_) if with_hext else None,) + \
            (adjoint_rhs_materials(p, t, m_, a_) if with_materials else (None, None))
    uA = np.zeros(p.n_cells)
    uKu = np.zeros(p.n_cells)

    uhn = np.zeros_like(mT)
    G = (lambda t, m_, a_: adjoint_rhs_hnodal(p, t, m_, a_)) if with_hnodal else None

    for s in range(n_steps, 0, -1):
        t = t0 + s * dt
        if with_hnodal:         # the stage states are those of the RK4 step below
            g1 = G(t, m, a)
        k1 = F(t, m, a)
        k2 = F(t + 0.5 * h, m + 0.5 * h * k1[0], a + 0.5 * h * k1[1])
        k3 = F(t + 0.5 * h, m + 0.5 * h * k2[0], a + 0.5 * h * k2[1])
        k4 = F(t + h, m + h * k3[0], a + h * k3[1])
        if with_hnodal:
            g2 = G(t + 0.5 * h, m + 0.5 * h * k1[0], a + 0.5 * h * k1[1])
            g3 = G(t + 0.5 * h, m + 0.5 * h * k2[0], a + 0.5 * h * k2[1])
            g4 = G(t + h, m + h * k3[0], a + h * k3[1])
            uhn = uhn + h / 6.0 * (g1 + 2 * g2 + 2 * g3 + g4)
        m = _llg.normalise(m + h / 6.0 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0]))
        a = a + h / 6.0 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1])
        u = u + h / 6.0 * (k1[2] + 2 * k2[2] + 2 * k3[2] + k4[2])
        if with_hext:
            uh = uh + h / 6.0 * (k1[3] + 2 * k2[3] + 2 * k3[3] + k4[3])
        if with_materials:
            uA = uA + h / 6.0 * (k1[4] + 2 * k2[4] + 2 * k3[4] + k4[4])
            uKu = uKu + h / 6.0 * (k1[5] + 2 * k2[5] + 2 * k3[5] + k4[5])
        if checkpoints is not None and (s - 1) in checkpoints:
            m = checkpoints[s - 1].copy()
        if a_jumps is not None and (s - 1) in a_jumps:
            a = a + a_jumps[s - 1]
    out = (m, a, u) + ((uh,) if with_hext else ())
    return out + ((uA, uKu) if with_materials else ()) + ((uhn,) if with_hnodal else ())
