"""Build the two sides of a parity test from one seeded Workload (tests only).

`oracle_problem` feeds the rounded inputs to the fp64 CPU oracle, `gpu_mesh` feeds the same
rounded inputs to libnm.so through the ctypes binding.  Nothing here does any of the method's
arithmetic.
"""
import numpy as np

from paper_2411_11725_b200 import workloads as wl


def rel_l2(x, ref):
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.sqrt(np.sum(ref * ref))
    num = np.sqrt(np.sum((x - ref) ** 2))
    return num / den if den > 0 else num


def max_abs_rel(x, ref):
    """max |x - ref| / max |ref|: the element-wise companion of rel_l2 (one wrong node on a 17 M-node
    grid moves the L2 norm by 1e-6 of itself and this by its full error)."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.max(np.abs(ref))
    num = np.max(np.abs(x - ref))
    return num / den if den > 0 else num


def assert_parity(x, ref, tol, what="", cmax=10.0):
    """north_star's relative-L2 bound and, beside it, max |x - ref| <= cmax * tol * max |ref|."""
    e, m = rel_l2(x, ref), max_abs_rel(x, ref)
    assert e <= tol, "%s: rel L2 %.3e > %.1e" % (what, e, tol)
    assert m <= cmax * tol, "%s: max abs %.3e of max|ref| > %.1e" % (what, m, cmax * tol)
    return e, m


# The oracle's tensor table N(p), p_d = 0..N_d-1, depends on the offset and the cell size only, so the
# table of a smaller grid with the same cells is a sub-block of a larger one (pinned on a tiny case in
# tests/test_oracle_demag.py).  The config-4 grids share their cell size: the __float128 table of the
# largest one asked for so far is kept for the session and sliced.
_TENSOR_CACHE = {}


def oracle_tensor(n_cells, dx):
    from oracle import demag
    n = tuple(int(v) for v in n_cells)
    key = tuple(float(v) for v in dx)
    have = _TENSOR_CACHE.get(key)
    if have is not None and all(a <= b for a, b in zip(n, have.shape[1:])):
        return np.ascontiguousarray(have[:, :n[0], :n[1], :n[2]])
    Nt = demag.demag_tensor(n, key)
    if have is None or Nt.size > have.size:
        _TENSOR_CACHE[key] = Nt
    return Nt


def np_dtype(torch_dtype):
    import torch
    return np.float64 if torch_dtype == torch.float64 else np.float32


def oracle_problem(w, dtype=np.float64, basis=3):
    """oracle.llg.Problem with the materials rounded to the build precision."""
    from oracle import llg
    r = lambda v: wl.round_to(w.cell_array(v), dtype)
    p = llg.Problem(tuple(w.n_cells), tuple(float(v) for v in w.dx), r(w.Ms), r(w.A), r(w.Ku),
                    tuple(w.ku_axis), float(w.gamma), float(w.alpha), int(w.terms), basis=basis)
    if (w.terms & wl.TERM_DEMAG) and int(np.prod(w.n_cells)) >= 32 ** 3:
        p._Nt = oracle_tensor(w.n_cells, w.dx)
    return p


def oracle_zeeman(w, dtype=np.float64, h_static=None):
    """Callable t -> nodal H_ext (paper index order) matching gpu_zeeman, or None."""
    if not (w.terms & wl.TERM_ZEEMAN):
        return None
    hu = wl.round_to(np.asarray(w.h_uniform, dtype=np.float64), dtype)
    hp = wl.round_to(w.h_pulse, dtype) if w.h_pulse is not None else None
    hs = wl.round_to(h_static, dtype) if h_static is not None else None
    shape = tuple(np.asarray(w.m0).shape)          # the basis nodes (a reduced basis has fewer: _sides.reduce_nodal)

    def z(t):
        h = np.broadcast_to(hu[:, None, None, None], shape).copy()
        if hs is not None:
            h += hs
        if hp is not None:
            amp = float(np.asarray(wl.sinc_pulse(t, **w.pulse) if w.pulse else 1.0).astype(dtype))
            h += amp * hp
        return h
    return z


def dev(a, torch_dtype, device=0):
    """Paper-order numpy array -> ABI-order device tensor of the mesh dtype."""
    import torch
    return torch.from_numpy(wl.to_abi(a)).to(device="cuda:%d" % device, dtype=torch_dtype).contiguous()


def host(t):
    """ABI-order device tensor -> paper-order fp64 numpy array."""
    return wl.from_abi(t.detach().cpu().double().numpy())


def reduce_nodal(a, D):
    """A paper-order nodal array of a one-layer mesh restricted to the nodes of a D-dimensional basis
    (Eqs. 23-24): the layer at index 0 of every reduced axis, kept as an axis of extent 1."""
    sl = tuple(slice(None) if d < D else slice(0, 1) for d in range(3))
    return np.ascontiguousarray(np.asarray(a)[(Ellipsis,) + sl])


def gpu_mesh(w, torch_dtype, device=0, basis=3):
    from paper_2411_11725_b200 import binding as nm
    mat = {}
    for name in ("Ms", "A", "Ku"):
        v = getattr(w, name)
        mat[name] = float(v) if np.isscalar(v) else dev(v, torch_dtype, device)
    return nm.Mesh(w.n_cells, w.dx, dtype=torch_dtype, device=device, terms=w.terms, gamma=w.gamma,
                   alpha=w.alpha, ku_axis=w.ku_axis, basis=basis, **mat)


def gpu_zeeman(w, torch_dtype, device=0, h_static=None):
    from paper_2411_11725_b200 import binding as nm
    if not (w.terms & wl.TERM_ZEEMAN):
        return None
    hp = dev(w.h_pulse, torch_dtype, device) if w.h_pulse is not None else None
    hs = dev(h_static, torch_dtype, device) if h_static is not None else None
    amp = (lambda t: wl.sinc_pulse(t, **w.pulse)) if (w.pulse and hp is not None) else None
    return nm.Zeeman(h_uniform=w.h_uniform, h_static=hs, h_pulse=hp, amp=amp)
