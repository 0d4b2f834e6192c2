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
