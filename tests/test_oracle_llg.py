"""Pins for oracle/llg.py (C6 of SURVEY.md §8(c); Eq. 1, 284-286)."""
import numpy as np
import pytest

from oracle import llg, mesh
from oracle.llg import Problem, TERM_EXCHANGE, TERM_DEMAG, TERM_ANISO, TERM_ZEEMAN


def rand_unit(shape, seed):
    v = np.random.default_rng(seed).standard_normal((3,) + tuple(shape))
    return v / np.sqrt(np.sum(v * v, axis=0))


def small_problem(alpha, terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO | TERM_ZEEMAN, seed=0):
    rng = np.random.default_rng(seed)
    n, dx = (4, 3, 2), (3e-9, 3e-9, 3e-9)
    return Problem(n, dx, rng.uniform(6e5, 8e5, n), rng.uniform(1e-11, 1.3e-11, n),
                   rng.uniform(1e5, 5e5, n), ku_axis=(0.0, 0.6, 0.8), alpha=alpha, terms=terms)


def test_cross_product_against_numpy():
    rng = np.random.default_rng(0)
    a, b = rng.standard_normal((3, 5)), rng.standard_normal((3, 5))
    assert np.allclose(llg.cross(a, b), np.cross(a.T, b.T).T)


def test_rhs_is_perpendicular_to_m_and_matches_eq1_by_hand():
    p = small_problem(0.3)
    m = rand_unit(p.node_shape, 1)
    h = np.array([1e4, -2e4, 5e4])
    f = llg.llg_rhs(p, 0.0, m, lambda t: h)
    assert np.abs(np.sum(m * f, axis=0)).max() < 1e-15 * np.abs(f).max()
    # one node by hand with numpy.cross
    H = llg.effective_field(p, m, h)
    nd = (slice(None), 2, 1, 1)
    gp = p.gamma / (1 + p.alpha ** 2)
    ref = -gp * np.cross(m[nd], H[nd]) - p.alpha * gp * np.cross(m[nd], np.cross(m[nd], H[nd]))
    assert np.allclose(f[nd], ref, rtol=1e-14)


def test_macrospin_closed_form():
    """One cell, Zeeman only, H = H z: phi(t) = phi0 + g' H t, tan(theta/2) = tan(theta0/2) exp(-alpha g' H t)."""
    alpha, Hz = 0.1, 1e5
    p = Problem.uniform((1, 1, 1), (2e-9, 2e-9, 2e-9), 8e5, 1.3e-11, alpha=alpha, terms=TERM_ZEEMAN)
    th0, ph0 = 1.0, 0.3
    m0 = np.array([np.sin(th0) * np.cos(ph0), np.sin(th0) * np.sin(ph0), np.cos(th0)])
    m = np.broadcast_to(m0[:, None, None, None], (3, 2, 2, 2)).copy()
    gp = p.gamma / (1 + alpha ** 2)
    T, nst = 2e-10, 400
    dt = T / nst
    for s in range(nst):
        m = llg.rk4_step(p, s * dt, dt, m, lambda t: np.array([0.0, 0.0, Hz]))
    th = 2 * np.arctan(np.tan(th0 / 2) * np.exp(-alpha * gp * Hz * T))
    ph = ph0 + gp * Hz * T
    ref = np.array([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)])
    assert np.abs(m - ref[:, None, None, None]).max() < 1e-9


def test_energy_conserved_without_damping_and_decays_with_damping():
    h = np.array([0.0, 3e4, 5e4])
    zee = lambda t: h
    p = small_problem(0.0)
    m = rand_unit(p.node_shape, 2)
    E0 = llg.energy(p, m, h)
    dt = 2e-14
    errs = []
    for step_dt in (dt, dt / 2):
        mm = m.copy()
        for s in range(int(round(10 * dt / step_dt))):
            mm = llg.rk4_step(p, 0.0, step_dt, mm, zee, renormalise=False)
        errs.append(abs(llg.energy(p, mm, h) - E0))
    assert 0 < errs[0] < 1e-4 * abs(E0)
    assert errs[1] < errs[0] / 10                     # conserved to O(dt^4) (or better)
    # with damping: dE/dt = -alpha g' sum_n L_n |m x H|^2 <= 0
    p = small_problem(0.5)
    H = llg.effective_field(p, m, h)
    gp = p.gamma / (1 + p.alpha ** 2)
    rate = -p.alpha * gp * np.sum(p.L * np.sum(llg.cross(m, H) ** 2, axis=0))
    eps = 1e-16
    f = llg.llg_from_field(p, m, H)
    dE = (llg.energy(p, m + eps * 1e3 * f, h) - llg.energy(p, m - eps * 1e3 * f, h)) / (2e3 * eps)
    assert rate < 0 and abs(dE - rate) < 1e-6 * abs(rate)
    E_prev = llg.energy(p, m, h)
    mm = m.copy()
    for s in range(20):
        mm = llg.rk4_step(p, 0.0, 5e-15, mm, zee)
        E = llg.energy(p, mm, h)
        assert E < E_prev
        E_prev = E


def test_rk4_is_fourth_order_and_renormalises():
    p = small_problem(0.1)
    m0 = rand_unit(p.node_shape, 3)
    zee = lambda t: np.array([0.0, 0.0, 5e4 * np.cos(1e12 * t)])
    T = 4e-14

    def run(nst, renorm=False):
        m = m0.copy()
        for s in range(nst):
            m = llg.rk4_step(p, s * T / nst, T / nst, m, zee, renormalise=renorm)
        return m
    ref = run(64)
    e1 = np.abs(run(4) - ref).max()
    e2 = np.abs(run(8) - ref).max()
    assert 12 < e1 / e2 < 20                           # halving dt: 16x
    m = run(4, renorm=True)
    assert np.abs(np.sum(m * m, axis=0) - 1).max() < 1e-15


def test_dopri5_tableau_and_order():
    # tableau consistency: rows of A sum to c, weights sum to 1
    for s in range(7):
        assert abs(sum(llg.DP_A[s]) - llg.DP_C[s]) < 1e-15
    assert abs(sum(llg.DP_B5) - 1) < 1e-15 and abs(sum(llg.DP_B4) - 1) < 1e-15
    assert llg.DP_A[6] == llg.DP_B5[:6]                # FSAL property
    # order conditions up to 5 for B5 and up to 4 for B4 on the quadrature conditions sum b c^k = 1/(k+1)
    c = np.array(llg.DP_C)
    for k in range(5):
        assert abs(np.dot(llg.DP_B5, c ** k) - 1 / (k + 1)) < 1e-15
    for k in range(4):
        assert abs(np.dot(llg.DP_B4, c ** k) - 1 / (k + 1)) < 1e-15
    assert abs(np.dot(llg.DP_B4, c ** 4) - 1 / 5) > 1e-4
    p = small_problem(0.1)
    m0 = rand_unit(p.node_shape, 4)
    zee = lambda t: np.array([0.0, 0.0, 5e4 * np.cos(1e12 * t)])
    T = 4e-14

    def run(nst):
        m = m0.copy()
        en = []
        for s in range(nst):
            m, e, ok = llg.dopri5_step(p, s * T / nst, T / nst, m, zee, renormalise=False,
                                       rtol=1e-3, atol=1e-3)
            assert ok
            en.append(e)
        return m, en
    ref, _ = run(32)
    (a, ea), (b, eb) = run(2), run(4)
    r = np.abs(a - ref).max() / np.abs(b - ref).max()
    assert 20 < r < 50                                 # fifth order: 32x
    assert 20 < ea[0] / eb[0] < 50                     # local error estimate ~ dt^5
    # rejection leaves m untouched
    m1, e, ok = llg.dopri5_step(p, 0.0, 2e-12, m0, zee, rtol=1e-9, atol=1e-9)
    assert not ok and e > 1 and m1 is m0
    assert llg.dopri5_next_dt(1.0, 1e-12) == 5.0 and llg.dopri5_next_dt(1.0, 1e12) == 0.2
    assert np.isclose(llg.dopri5_next_dt(2.0, 1.0), 1.8)


def test_dopri5_error_norm_definition():
    """err_norm with k_j replaced by hand: single macrospin where all nodes are identical."""
    p = Problem.uniform((1, 1, 1), (2e-9,) * 3, 8e5, 1.3e-11, alpha=0.05, terms=TERM_ZEEMAN)
    m0 = np.array([0.6, 0.0, 0.8])
    m = np.broadcast_to(m0[:, None, None, None], (3, 2, 2, 2)).copy()
    h = np.array([0.0, 1e5, 0.0])
    dt, rtol, atol = 3e-12, 1e-6, 1e-7
    y5, en, ok = llg.dopri5_step(p, 0.0, dt, m, lambda t: h, renormalise=False, rtol=rtol, atol=atol)
    gp = p.gamma / (1 + p.alpha ** 2)
    f = lambda y: -gp * np.cross(y, h) - p.alpha * gp * np.cross(y, np.cross(y, h))
    k = []
    for s in range(7):
        y = m0 + dt * sum(a * kk for a, kk in zip(llg.DP_A[s], k))
        k.append(f(y))
    y5r = m0 + dt * sum(b * kk for b, kk in zip(llg.DP_B5, k))
    y4r = m0 + dt * sum(b * kk for b, kk in zip(llg.DP_B4, k))
    enr = np.sqrt(np.mean(((y5r - y4r) / (atol + rtol * np.maximum(np.abs(m0), np.abs(y5r)))) ** 2))
    assert np.isclose(en, enr, rtol=1e-9)
    got = y5[:, 0, 0, 0] if ok else None
    if ok:
        assert np.allclose(got, y5r, rtol=1e-13)


def test_normalise_keeps_zero_vectors_zero():
    """Vacuum nodes carry m = 0 by convention: normalise must not turn them into NaN."""
    m = np.zeros((3, 2, 2, 1))
    m[:, 0, 0, 0] = (3.0, 0.0, 4.0)
    m[:, 1, 1, 0] = (0.0, -2.0, 0.0)
    out = llg.normalise(m)
    assert np.all(np.isfinite(out))
    assert np.allclose(out[:, 0, 0, 0], (0.6, 0.0, 0.8)) and np.allclose(out[:, 1, 1, 0], (0.0, -1.0, 0.0))
    assert np.all(out[:, 0, 1, 0] == 0) and np.all(out[:, 1, 0, 0] == 0)
