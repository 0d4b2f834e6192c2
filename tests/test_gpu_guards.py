"""Out-of-bounds and race evidence without compute-sanitizer (closed on this pool: profiles/r2_sanitizer.md).

Every kernel family is run on a small mesh with
  * the workspace block carved out of a larger allocation whose bytes before and after it hold a
    canary pattern (a kernel that writes past a workspace array at either end of the block trips it;
    arrays inside the block are 256-byte aligned, so an overrun inside it lands in the next array and
    shows as a parity failure in the -m gpu parity tests instead),
  * every input array (m, a, materials, nodal Zeeman field) placed in the middle of a slab filled with
    NaN, so that a read before or after the array poisons the result,
  * every output array placed in the middle of a canary-filled slab,
and the whole sequence (H_eff, right-hand side, RK4 steps incl. graph replay, a Dormand-Prince step,
the adjoint right-hand side, a backward RK4 step with all extra gradients) is repeated three times:
results must be finite, the canaries intact, and the three repetitions bit-identical (an unsynchronised
shared-memory exchange or a barrier-phase slip in the warp-specialised pipelines shows up as run-to-run
differences).  The guarded results must also equal those of a plain run bit for bit.
"""
import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GUARD = 4096            # elements of guard band either side of every array
CANARY = 0x5A


def _cube(n):
    w = wl.config4_sweep(16)
    w.n_cells = tuple(n)
    w.m0 = wl.random_unit_field(w.node_shape, 4 + sum(n))
    return w, None


CASES = [
    ("film 32x8x1 f64 (general path, one layer)", lambda: (wl.config1_tiny_film(), None), "f64", 0),
    ("ragged 12x10x6 all terms (general path)", lambda: wl.varied_case((12, 10, 6), vacuum=True), "f32", 0),
    ("ragged 12x10x6 all terms f64", lambda: wl.varied_case((12, 10, 6), vacuum=True), "f64", 0),
    ("32x32x256 (k_pz_mid)", lambda: _cube((32, 32, 256)), "f32", 1),
    ("32x256x32 (k_py_fwd / k_py_inv)", lambda: _cube((32, 256, 32)), "f32", 1),
    ("32x128x128 (k_pz_mid8, k_py_*8)", lambda: _cube((32, 128, 128)), "f32", 1),
    ("128x32x16 (k_px_*, k_node_col)", lambda: _cube((128, 32, 16)), "f32", 1),
    ("36x64x48 embedded, cell-wise materials", lambda: wl.varied_case((36, 64, 48), vacuum=True), "f32", 2),
    ("32x32x32 f64 (k_fy_*, k_fz_mid)", lambda: _cube((32, 32, 32)), "f64", 1),
    ("128x16x16 f64 (k_px_* f64, k_node_col f64)", lambda: _cube((128, 32, 16)), "f64", 1),
    ("32x256x32 f64 (k_py_fwd / k_py_inv in fp64)", lambda: _cube((32, 256, 32)), "f64", 1),
    ("32x32x256 f64 (k_pz_mid64)", lambda: _cube((32, 32, 256)), "f64", 1),
    ("32x128x128 f64 (k_pz_mid64_8, k_py_*8 in fp64)", lambda: _cube((32, 128, 128)), "f64", 1),
]


class Slabs:
    """Arrays in the middle of guard bands: inputs in NaN, outputs in a byte canary."""

    def __init__(self, td):
        self.td = td
        self.out = []

    def inp(self, a):
        t = torch.from_numpy(wl.to_abi(a)).to(device="cuda:0", dtype=self.td).contiguous()
        slab = torch.full((t.numel() + 2 * GUARD,), float("nan"), dtype=self.td, device="cuda:0")
        v = slab[GUARD:GUARD + t.numel()].view(t.shape)
        v.copy_(t)
        return v

    def outp(self, shape, dtype=None):
        dtype = dtype or self.td
        n = int(np.prod(shape))
        es = torch.empty(0, dtype=dtype).element_size()
        raw = torch.full(((n + 2 * GUARD) * es,), CANARY, dtype=torch.uint8, device="cuda:0")
        v = raw[GUARD * es:(GUARD + n) * es].view(dtype).view(shape)
        self.out.append((raw, GUARD * es, (GUARD + n) * es))
        return v

    def intact(self):
        return all(bool((raw[:lo] == CANARY).all()) and bool((raw[hi:] == CANARY).all()) for raw, lo, hi in self.out)


def _run(make, prec, guarded):
    from paper_2411_11725_b200 import binding as nm
    td = torch.float32 if prec == "f32" else torch.float64
    nd = np.float32 if prec == "f32" else np.float64
    w, hs = make()
    sl = Slabs(td)
    put = sl.inp if guarded else (lambda a: torch.from_numpy(wl.to_abi(a)).to(device="cuda:0", dtype=td).contiguous())
    new = sl.outp if guarded else (lambda shape, dtype=None: torch.empty(shape, dtype=dtype or td, device="cuda:0"))
    mat = {k: (float(getattr(w, k)) if np.isscalar(getattr(w, k)) else put(np.asarray(getattr(w, k), dtype=np.float64)))
           for k in ("Ms", "A", "Ku")}
    desc = nm.make_desc(w.n_cells, w.dx, td, 0, w.terms, w.gamma, w.alpha, w.ku_axis, **mat)
    nbytes = nm.nm_mesh_query_workspace(desc)
    pad = 1 << 16
    big = torch.full((nbytes + 2 * pad + 256,), CANARY, dtype=torch.uint8, device="cuda:0")
    off = (-(big.data_ptr() + pad)) % 256 + pad
    ws = big[off:off + nbytes]
    mesh = nm.Mesh(w.n_cells, w.dx, dtype=td, terms=w.terms, gamma=w.gamma, alpha=w.alpha, ku_axis=w.ku_axis,
                   workspace=ws, **mat)
    z = None
    if w.terms & wl.TERM_ZEEMAN:
        z = nm.Zeeman(h_uniform=w.h_uniform, h_static=put(hs) if hs is not None else None)
    m = put(wl.round_to(w.m0, nd))
    a = put(wl.round_to(np.random.default_rng(3).standard_normal(w.m0.shape), nd))
    dt = w.dt or 2e-14
    reps = []
    for _ in range(3):
        H = mesh.nm_heff(0.0, m, z, new(m.shape))
        f = mesh.nm_llg_rhs(0.0, m, z, new(m.shape))
        y = new(m.shape)
        y.copy_(m)
        for s in range(3):
            mesh.nm_rk_step(0, s * dt, dt, y, z)
        err = mesh.nm_rk_step(1, 3 * dt, dt, y, z, want_err=True)
        f2, da, du = new(m.shape), new(m.shape), new(mesh.cell_shape_abi)
        nm._check(nm.lib().nm_llg_adjoint_rhs(mesh.handle, 0.0, nm._ptr(m), nm._ptr(a), nm._zref(z), nm._ptr(f2),
                                              nm._ptr(da), nm._ptr(du), nm._stream(0)))
        ya, u, uA, uKu = new(m.shape), new(mesh.cell_shape_abi), new(mesh.cell_shape_abi), new(mesh.cell_shape_abi)
        uh = new((3,), torch.float64)
        ya.copy_(a)
        for t_ in (u, uA, uKu, uh):
            t_.zero_()
        mesh.nm_adjoint_rk4_step_ex(4 * dt, dt, y, ya, u, u_A=uA, u_Ku=uKu, u_h=uh, zeeman=z)
        torch.cuda.synchronize()
        reps.append([t_.clone() for t_ in (H, f, y, f2, da, du, ya, u, uA, uKu, uh)] + [torch.tensor([err])])
    ws_ok = bool((big[:off] == CANARY).all()) and bool((big[off + nbytes:] == CANARY).all())
    return reps, (sl.intact() if guarded else True), ws_ok, mesh.nm_debug_demag_path()


@pytest.mark.parametrize("name,make,prec,path", CASES, ids=[c[0] for c in CASES])
def test_guard_bands_and_run_to_run_identity(name, make, prec, path):
    reps, out_ok, ws_ok, got_path = _run(make, prec, guarded=True)
    assert got_path == path
    assert ws_ok, "a kernel wrote outside the workspace block"
    assert out_ok, "a kernel wrote outside an output array"
    for t_ in reps[0]:
        assert bool(torch.isfinite(t_).all()), "an input was read outside its array (NaN guard band)"
    for r in reps[1:]:
        for x, y in zip(reps[0], r):
            assert torch.equal(x, y), "results differ between identical runs"
    plain, _, ws_ok2, _ = _run(make, prec, guarded=False)
    assert ws_ok2
    for x, y in zip(reps[0], plain[0]):
        assert torch.equal(x, y), "guarded and plain runs differ"
