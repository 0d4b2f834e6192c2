"""Seeded synthetic inputs for the five BASELINE.json configs.

A module of its own: it holds none of the method's arithmetic and imports neither the CUDA
binding nor `oracle/`; tests feed the same arrays to both sides.  The recipe is stated in
DESIGN.md ("Input recipe").  All draws use numpy.random.default_rng(seed); arrays are made
in fp64 and rounded to the build precision with `round_to`, and the *rounded* values are what
both sides consume.

Index order here is the paper's: nodal fields (3, N1+1, N2+1, N3+1), cell fields (N1, N2, N3).
The C-ABI stores x fastest: `to_abi` / `from_abi` only permute axes.
"""
from dataclasses import dataclass, field

import numpy as np

TERM_EXCHANGE, TERM_DEMAG, TERM_ANISO, TERM_ZEEMAN = 1, 2, 4, 8


def to_abi(a):
    """(..., n1, n2, n3) paper order -> (..., n3, n2, n1) contiguous (x fastest)."""
    a = np.asarray(a)
    lead = tuple(range(a.ndim - 3))
    k = a.ndim
    return np.ascontiguousarray(a.transpose(lead + (k - 1, k - 2, k - 3)))


def from_abi(a):
    """Inverse of to_abi."""
    return to_abi(a)


def round_to(a, dtype):
    """Round an fp64 array to the build precision and return it as fp64 again."""
    return np.asarray(a, dtype=np.float64).astype(dtype).astype(np.float64)


def _unit(v):
    return v / np.sqrt(np.sum(v * v, axis=0, keepdims=True))


def random_unit_field(node_shape, seed):
    rng = np.random.default_rng(seed)
    return _unit(rng.standard_normal((3,) + tuple(node_shape)))


def box_filter3(v):
    """3-point box filter along each node axis, edge-replicated (config 2's smoothing)."""
    for ax in (1, 2, 3):
        pad = [(0, 0)] * 4
        pad[ax] = (1, 1)
        w = np.pad(v, pad, mode="edge")
        sl = lambda s: tuple(slice(None) if d != ax else s for d in range(4))
        v = (w[sl(slice(0, -2))] + w[sl(slice(1, -1))] + w[sl(slice(2, None))]) / 3.0
    return v


@dataclass
class Workload:
    name: str
    n_cells: tuple
    dx: tuple
    Ms: object              # scalar or (N1,N2,N3)
    A: object
    Ku: object = 0.0
    ku_axis: tuple = (0.0, 0.0, 1.0)
    gamma: float = 2.211e5
    alpha: float = 0.02
    terms: int = TERM_EXCHANGE | TERM_DEMAG
    m0: np.ndarray = None
    h_uniform: tuple = (0.0, 0.0, 0.0)
    h_pulse: np.ndarray = None      # nodal (3, nodes) spatial profile of the pulse or None
    pulse: dict = field(default_factory=dict)
    dt: float = 0.0
    n_steps: int = 0
    seed: int = 0

    @property
    def node_shape(self):
        return tuple(n + 1 for n in self.n_cells)

    def cell_array(self, v):
        return np.full(self.n_cells, float(v)) if np.isscalar(v) else np.asarray(v, dtype=np.float64)


def config1_tiny_film():
    """32x8x1 cells, exchange + demag, 200 RK4 steps of 1e-13 s, fp64."""
    n = (32, 8, 1)
    w = Workload("config1_tiny_film", n, (3.125e-9, 3.125e-9, 3e-9), 8e5, 1.3e-11,
                 alpha=0.02, gamma=2.211e5, dt=1e-13, n_steps=200, seed=1)
    w.m0 = random_unit_field(w.node_shape, 1)
    return w


def config2_cube(N=64):
    """Cube N^3 (64 in BASELINE.json), exchange + demag + uniaxial + Zeeman, one H_eff."""
    n = (N, N, N)
    w = Workload("config2_cube%d" % N, n, (2e-9, 2e-9, 2e-9), 8e5, 1.3e-11, Ku=5e5,
                 ku_axis=(0.0, 0.0, 1.0), h_uniform=(0.0, 0.0, 5e4),
                 terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO | TERM_ZEEMAN, seed=2)
    w.m0 = _unit(box_filter3(random_unit_field(w.node_shape, 2)))
    return w


def sinc_pulse(t, amp=1e3, f=50e9, t0=100e-12):
    """amp * sinc(2 pi f (t - t0)), sinc(x) = sin(x)/x, sinc(0) = 1 (reading C6)."""
    x = 2.0 * np.pi * f * (t - t0)
    return amp * (1.0 if x == 0.0 else np.sin(x) / x)


def config3_thin_film(N=512):
    """N x N x 1 film (512 in BASELINE.json) with a sinc Zeeman pulse H_y on a 10-cell stripe."""
    n = (N, N, 1)
    w = Workload("config3_film%d" % N, n, (2e-9, 2e-9, 5e-9), 1.4e5, 3.65e-12, alpha=1e-3,
                 terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ZEEMAN, seed=3)
    rng = np.random.default_rng(3)
    m = 1e-3 * rng.standard_normal((3,) + w.node_shape)
    m[0] += 1.0
    w.m0 = _unit(m)
    hp = np.zeros((3,) + w.node_shape)
    lo = N // 2 - 5                      # nodes n1 in [251, 261] at N = 512
    hp[1, lo:lo + 11, :, :] = 1.0
    w.h_pulse = hp
    w.pulse = dict(amp=1e3, f=50e9, t0=100e-12)
    return w


def config4_sweep(N):
    """Cube N^3, N in {16,32,64,128,192,256}, exchange + demag, random unit m (seed 4+N)."""
    n = (N, N, N)
    w = Workload("config4_sweep%d" % N, n, (2e-9, 2e-9, 2e-9), 8e5, 1.3e-11, alpha=0.02,
                 dt=2e-14, seed=4 + N)
    w.m0 = random_unit_field(w.node_shape, 4 + N)
    return w


def config5_inverse(n=(256, 64, 1), n_steps=2000):
    """Film with cell-wise Ms ~ U[1e5, 1.5e5]; forward RK4, objective mean m_y over the last
    32 node columns, adjoint-state gradient dJ/dMs (C8)."""
    w = Workload("config5_inverse", tuple(n), (4e-9, 4e-9, 5e-9), None, 3.65e-12, alpha=1e-2,
                 h_uniform=(0.0, 2e3, 0.0), terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ZEEMAN,
                 dt=5e-14, n_steps=n_steps, seed=5)
    rng = np.random.default_rng(5)
    w.Ms = rng.uniform(1e5, 1.5e5, size=w.n_cells)
    m = 0.1 * rng.standard_normal((3,) + w.node_shape)
    m[0] += 1.0
    w.m0 = _unit(m)
    return w


def objective_weights(w, columns=32):
    """dJ/dm(T) for J = mean of m_y over nodes with n1 >= N1+1-columns (reading C8)."""
    g = np.zeros((3,) + w.node_shape)
    n1 = w.node_shape[0]
    lo = max(0, n1 - columns)
    cnt = (n1 - lo) * w.node_shape[1] * w.node_shape[2]
    g[1, lo:, :, :] = 1.0 / cnt
    return g


def fd_cells(w, k=8, seed=6):
    """k distinct cells drawn with seed 6 for the finite-difference gradient check."""
    rng = np.random.default_rng(seed)
    flat = rng.choice(int(np.prod(w.n_cells)), size=k, replace=False)
    return [tuple(int(v) for v in np.unravel_index(f, w.n_cells)) for f in flat]


def varied_case(n_cells, dx=(2e-9, 3e-9, 2.5e-9), seed=11, vacuum=False, alpha=0.05):
    """Ragged parity case: every term on, cell-wise random Ms, A, Ku (optionally a vacuum corner
    block with Ms = 0), a tilted anisotropy axis, smoothed random m and a nodal static field.
    Returns (workload, h_static)."""
    n = tuple(int(v) for v in n_cells)
    rng = np.random.default_rng(seed)
    w = Workload("varied_%dx%dx%d" % n, n, tuple(dx), None, None, alpha=alpha,
                 terms=TERM_EXCHANGE | TERM_DEMAG | TERM_ANISO | TERM_ZEEMAN, seed=seed,
                 h_uniform=(1e4, -2e4, 3e4), dt=2e-14)
    w.Ms = rng.uniform(4e5, 9e5, size=n)
    w.A = rng.uniform(0.8e-11, 1.5e-11, size=n)
    w.Ku = rng.uniform(1e5, 5e5, size=n)
    if vacuum:
        w.Ms[: max(1, n[0] // 3), : max(1, n[1] // 2), :] = 0.0
    k = np.array([1.0, 2.0, 2.0])
    w.ku_axis = tuple(k / np.sqrt(np.sum(k * k)))
    w.m0 = _unit(box_filter3(random_unit_field(w.node_shape, seed + 1)))
    h_static = 5e4 * rng.standard_normal((3,) + w.node_shape)
    return w, h_static
