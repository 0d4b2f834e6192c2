"""Host logic of paper_2411_11725_b200/drivers.py that needs no GPU: the step controller equals
the oracle's (reading C6) and the integration loop takes the steps it should on a fake mesh."""
import numpy as np

from oracle import llg
from paper_2411_11725_b200 import drivers


def test_next_dt_matches_oracle_controller():
    for err in [0.0, 1e-6, 0.03, 0.5, 1.0, 1.7, 40.0, 1e9]:
        assert np.isclose(drivers.dopri5_next_dt(1e-13, err), llg.dopri5_next_dt(1e-13, err), rtol=1e-15)
    assert drivers.dopri5_next_dt(1.0, 1e-12) == 5.0       # clipped above
    assert drivers.dopri5_next_dt(1.0, 1e12) == 0.2        # clipped below


class _FakeMesh:
    """Accepts every second attempt; records (t, dt) of each call."""
    def __init__(self):
        self.calls = []

    def nm_rk_step(self, scheme, t, dt, m, zeeman, renormalise, rtol, atol, want_err):
        assert scheme == 1 and want_err
        self.calls.append((t, dt))
        return 0.5 if len(self.calls) % 2 == 0 else 2.0


def test_integrate_dopri5_loop_control():
    mesh = _FakeMesh()
    t, dt, acc, rej = drivers.integrate_dopri5(mesh, None, 0.0, 1.0, 0.4)
    assert abs(t - 1.0) < 1e-15 and acc >= 2 and rej == acc
    # a rejected attempt is retried from the same time with a smaller step
    for (t0, h0), (t1, h1) in zip(mesh.calls[0::2], mesh.calls[1::2]):
        assert t1 == t0 and h1 < h0
    # the last step is clipped to land on t1 exactly
    assert abs(mesh.calls[-1][0] + mesh.calls[-1][1] - 1.0) < 1e-15


class _NanMesh:
    """Every trial step returns a NaN error norm (a state that went non-finite)."""
    def __init__(self):
        self.calls = []

    def nm_rk_step(self, scheme, t, dt, m, zeeman, renormalise, rtol, atol, want_err):
        self.calls.append(dt)
        return float("nan")


def test_non_finite_error_norm_shrinks_the_step_and_then_fails():
    """a NaN error norm used to read as "no error" (dt * 5 for ever)."""
    import pytest
    assert drivers.dopri5_next_dt(1.0, float("nan")) == 0.2
    assert drivers.dopri5_next_dt(1.0, float("inf")) == 0.2
    assert llg.dopri5_next_dt(1.0, float("nan")) == 0.2 and llg.dopri5_next_dt(1.0, float("inf")) == 0.2
    mesh = _NanMesh()
    with pytest.raises(ArithmeticError):
        drivers.integrate_dopri5(mesh, None, 0.0, 1.0, 0.1, max_rejects_in_a_row=6)
    assert len(mesh.calls) == 6
    assert all(b < a for a, b in zip(mesh.calls, mesh.calls[1:]))     # each retry is smaller
    mesh = _NanMesh()
    with pytest.raises(ArithmeticError):
        drivers.integrate_dopri5(mesh, None, 0.0, 1.0, 0.1, dt_min=1e-3)
    assert len(mesh.calls) == 3                                       # 0.1, 0.02, 0.004 -> 0.0008 < dt_min


class _FakeAdjMesh:
    """Scalar stand-in for the adjoint loops: m += 1 per forward step, m -= 1 per backward step;
    records the order of the calls."""
    cell_shape_abi = (1,)

    def __init__(self):
        self.log = []

    def nm_rk_step(self, scheme, t, dt, m, zeeman):
        m += 1.0
        self.log.append(("fwd", round(t / dt)))

    def nm_adjoint_rk4_step(self, t, dt, m, a, u, zeeman):
        m -= 1.0
        u += a.sum()
        self.log.append(("bwd", round(t / dt)))

    def nm_adjoint_add_objective(self, a, g, scale=1.0):
        a += scale * g
        self.log.append(("jump", float(g.sum())))


def test_adjoint_gradient_loop_adds_objectives_at_their_times():
    """a term L_s(m(t_s)) is evaluated on the forward pass at step s and added to the
    adjoint variable right after the backward step that arrives at t_s (after the checkpoint
    restore of that index)."""
    import torch
    mesh = _FakeAdjMesh()
    m0 = torch.zeros(1, dtype=torch.float64)
    seen = {}

    def at(s):
        def f(m):
            seen[s] = float(m[0])
            return torch.full((1,), 10.0 * s, dtype=torch.float64)
        return f

    mT, a0, u0 = drivers.adjoint_gradient(mesh, m0, lambda m: torch.ones(1, dtype=torch.float64), 1.0, 6,
                                          checkpoint_every=3, objectives_at={2: at(2), 4: at(4)})
    assert seen == {2: 2.0, 4: 4.0}                  # evaluated on m(t_s) of the forward pass
    assert float(mT[0]) == 6.0
    order = [e for e in mesh.log if e[0] != "fwd"]
    assert order == [("bwd", 6), ("bwd", 5), ("jump", 40.0), ("bwd", 4), ("bwd", 3), ("jump", 20.0),
                     ("bwd", 2), ("bwd", 1)]
    assert float(a0[0]) == 1.0 + 40.0 + 20.0
    # u sums a before each backward step: 1, 1, 41, 41, 61, 61
    assert float(u0[0]) == 1 + 1 + 41 + 41 + 61 + 61
    # without further objectives the loop is the plain one
    mesh2 = _FakeAdjMesh()
    drivers.adjoint_gradient(mesh2, m0, lambda m: torch.ones(1, dtype=torch.float64), 1.0, 4, checkpoint_every=2)
    assert [e[0] for e in mesh2.log] == ["fwd"] * 4 + ["bwd"] * 4


def test_field_angle_chain_rule():
    """Eq. (31) and its chain rule against central differences (host arithmetic on three numbers)."""
    Hc, th, ph = 3.0e4, 0.7, -1.1
    g = np.array([0.3, -1.2, 0.8])                                  # some dL/dh
    f = lambda a, b: float(np.dot(g, drivers.field_from_angles(Hc, a, b)))
    e = 1e-6
    dth, dph = drivers.angle_gradient(g, Hc, th, ph)
    assert abs(dth - (f(th + e, ph) - f(th - e, ph)) / (2 * e)) < 1e-5 * Hc
    assert abs(dph - (f(th, ph + e) - f(th, ph - e)) / (2 * e)) < 1e-5 * Hc
    h = drivers.field_from_angles(Hc, th, ph)
    assert abs(np.sqrt(sum(v * v for v in h)) - Hc) < 1e-9 * Hc
    assert drivers.field_from_angles(Hc, 0.0, 0.3)[2] == Hc
