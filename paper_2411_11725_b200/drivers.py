"""Host-side drivers around the C-ABI: the adaptive step controller of config 3 and the
adjoint-state gradient loop of config 5.  They hold loop control only — which step to take next,
when to store or restore a checkpoint — and call `nm_rk_step` / `nm_adjoint_rk4_step` for every
piece of arithmetic on the fields (readings C6 and C8).
"""
import torch


def dopri5_next_dt(dt, err_norm, safety=0.9, lo=0.2, hi=5.0):
    """Reading C6: dt_new = dt * clip(0.9 * err^(-1/5), 0.2, 5).  A non-finite error norm (NaN / Inf
    in the trial state) is a rejected step: shrink by the lower clip factor."""
    if err_norm != err_norm or err_norm == float("inf"):
        return dt * lo
    if err_norm <= 0.0:
        return dt * hi
    return dt * min(hi, max(lo, safety * err_norm ** (-0.2)))


def integrate_dopri5(mesh, m, t0, t1, dt0, zeeman=None, rtol=1e-5, atol=1e-5, renormalise=True,
                     max_steps=10 ** 9, on_step=None, dt_min=0.0, max_rejects_in_a_row=50):
    """Advance m in place from t0 to t1 with Dormand-Prince 5(4).  The device takes
    the accept/reject decision (nm_rk_step leaves m untouched on a rejected step) and returns the
    scalar error norm; this loop only adapts dt.  Returns (t, dt, accepted, rejected).  Raises
    ArithmeticError when the step size falls below dt_min or max_rejects_in_a_row trial steps in a
    row are rejected (a non-finite error norm counts as rejected): the state cannot be advanced."""
    t, dt = float(t0), float(dt0)
    acc = rej = 0
    run = 0
    while t < t1 and acc + rej < max_steps:
        h = min(dt, t1 - t)
        err = mesh.nm_rk_step(1, t, h, m, zeeman, renormalise=renormalise, rtol=rtol, atol=atol,
                              want_err=True)
        if err <= 1.0:
            t += h
            acc += 1
            run = 0
            if on_step is not None:
                on_step(t, h, err)
        else:
            rej += 1
            run += 1
        nxt = dopri5_next_dt(h, err)
        # a step clipped to land on t1 says nothing against the step size in use before it
        dt = max(nxt, dt) if (h < dt and err <= 1.0) else nxt
        if run >= max_rejects_in_a_row or not (dt > dt_min):
            raise ArithmeticError("Dormand-Prince: %d trial steps rejected in a row at t = %.6e s "
                                  "(last error norm %r, next dt %.3e s)" % (run, t, err, dt))
    return t, dt, acc, rej


def forward_rk4(mesh, m, dt, n_steps, zeeman=None, checkpoint_every=0, t0=0.0):
    """n_steps fixed RK4 steps in place; returns {step index: clone of m before that step}."""
    ck = {}
    for s in range(n_steps):
        if checkpoint_every and s % checkpoint_every == 0:
            ck[s] = m.clone()
        mesh.nm_rk_step(0, t0 + s * dt, dt, m, zeeman)
    return ck


def adjoint_gradient(mesh, m0, aT_of_mT, dt, n_steps, zeeman=None, checkpoint_every=100, t0=0.0,
                     objectives_at=None, with_hext=False, with_materials=False, with_hnodal=False):
    """Adjoint-state gradient dJ/dMs (Eqs. 27-30; reading C8).

    Forward RK4 from m0 with checkpoints, a(T) = aT_of_mT(m(T)) (the caller's dJ/dm(T)), then the
    backward RK4 of (m, a, u) with step -dt, m replaced by the stored checkpoint whenever one is
    reached.  Returns (m(T), a(0), u(0) = dJ/dMs per cell).

    objectives_at = {step index s < n_steps: callable m(t0 + s dt) -> dL_s/dm}: objective terms at
    further times; each is evaluated on the forward pass and added to the adjoint
    variable when the backward pass arrives at its time (nm_adjoint_add_objective).

    with_hext: also integrate the gradient with respect to a uniform external field h
    (nm_adjoint_rk4_step_hext) and return (m(T), a(0), u(0), u_h(0) = dL/dh as a
    device fp64 3-vector).
    with_materials: also integrate the gradients with respect to the cell-wise A and Ku
    (nm_adjoint_rk4_step_ex) and append (u_A(0), u_Ku(0)) to the returned tuple.
    with_hnodal: also integrate the gradient with respect to a time-constant nodal external field
    (nm_adjoint_extra.u_hn) and append u_hn(0) = dL/dh per node and component, last."""
    m = m0.clone()
    jumps = {}
    if objectives_at:
        ck = {}
        for s in range(n_steps):
            if checkpoint_every and s % checkpoint_every == 0:
                ck[s] = m.clone()
            if s in objectives_at:
                jumps[s] = objectives_at[s](m).clone()
            mesh.nm_rk_step(0, t0 + s * dt, dt, m, zeeman)
    else:
        ck = forward_rk4(mesh, m, dt, n_steps, zeeman, checkpoint_every, t0)
    mT = m.clone()
    a = aT_of_mT(mT).clone()
    u = torch.zeros(mesh.cell_shape_abi, dtype=m.dtype, device=m.device)
    uh = torch.zeros(3, dtype=torch.float64, device=m.device) if with_hext else None
    uA = torch.zeros_like(u) if with_materials else None
    uKu = torch.zeros_like(u) if with_materials else None
    uhn = torch.zeros_like(m) if with_hnodal else None
    for s in range(n_steps, 0, -1):
        if with_materials or with_hnodal:
            mesh.nm_adjoint_rk4_step_ex(t0 + s * dt, dt, m, a, u, u_A=uA, u_Ku=uKu, u_h=uh, zeeman=zeeman, u_hn=uhn)
        elif with_hext:
            mesh.nm_adjoint_rk4_step_hext(t0 + s * dt, dt, m, a, u, uh, zeeman)
        else:
            mesh.nm_adjoint_rk4_step(t0 + s * dt, dt, m, a, u, zeeman)
        if (s - 1) in ck:
            m.copy_(ck[s - 1])
        if (s - 1) in jumps:
            mesh.nm_adjoint_add_objective(a, jumps[s - 1])
    out = (mT, a, u) + ((uh,) if with_hext else ())
    return out + ((uA, uKu) if with_materials else ()) + ((uhn,) if with_hnodal else ())


# ---- field-angle problem of Sec. VII (Eqs. 31-33) ------------------------------
def field_from_angles(Hc, theta, phi):
    """Eq. (31): H_ext = Hc (sin theta cos phi, sin theta sin phi, cos theta)."""
    import math
    return (Hc * math.sin(theta) * math.cos(phi), Hc * math.sin(theta) * math.sin(phi), Hc * math.cos(theta))


def angle_gradient(dLdh, Hc, theta, phi):
    """Chain rule of Eq. (31): (dL/dtheta, dL/dphi) from dL/dh (three host numbers)."""
    import math
    st, ct, sp, cp = math.sin(theta), math.cos(theta), math.sin(phi), math.cos(phi)
    dth = Hc * (ct * cp * dLdh[0] + ct * sp * dLdh[1] - st * dLdh[2])
    dph = Hc * (-st * sp * dLdh[0] + st * cp * dLdh[1])
    return dth, dph


def field_angle_gradient(mesh, m0, loss_grad, Hc, theta, phi, dt, n_steps, checkpoint_every=100,
                         make_zeeman=None):
    """One forward and one backward solve for the field angles: returns
    (m(T), dL/dtheta, dL/dphi).  loss_grad(m(T)) is the caller's dL/dm(T) (the objective is the
    caller's, Eq. 33); the uniform field of Eq. (31) is the only external field unless make_zeeman
    (h_uniform -> Zeeman) adds nodal parts."""
    from . import binding as nm
    h = field_from_angles(Hc, theta, phi)
    z = make_zeeman(h) if make_zeeman else nm.Zeeman(h_uniform=h)
    mT, _, _, uh = adjoint_gradient(mesh, m0, loss_grad, dt, n_steps, z, checkpoint_every, with_hext=True)
    dLdh = uh.cpu().tolist()                       # 24 bytes: the gradient the optimiser steps on
    return (mT,) + angle_gradient(dLdh, Hc, theta, phi)


def optimise_field_angles(mesh, m0, loss, loss_grad, Hc, theta, phi, dt, n_steps, rate, iterations,
                          checkpoint_every=100):
    """Plain gradient descent on (theta, phi) as in Sec. VII ("convergence is achieved after 30-50
    gradient-descent steps").  loss(m(T)) -> float and loss_grad(m(T)) -> dL/dm(T) are
    the caller's objective (Eq. 33).  Returns (theta, phi, [loss per iteration])."""
    history = []
    for _ in range(iterations):
        mT, dth, dph = field_angle_gradient(mesh, m0, loss_grad, Hc, theta, phi, dt, n_steps, checkpoint_every)
        history.append(float(loss(mT)))
        theta -= rate * dth
        phi -= rate * dph
    return theta, phi, history
