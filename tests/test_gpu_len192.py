"""An axis of 192 cells transformed at its own length (NM_FAST192=1 at nm_mesh_create; Len<12> in nm_fft16.cuh:
192 = 3 x 64, a radix-3 step on top of the 64-point register transforms): nm_heff and nm_llg_rhs against the oracle
for each axis alone and combined, in both precisions -- k_fx_* / k_fy_* / k_fz_mid with M = 12 and, in fp32, the
pipelined z pass k_pz_mid3.  Without the switch the same meshes run zero-extended to 256 cells (the default: it is the
faster of the two, profiles/r2_final.md), and both must agree with the oracle."""
import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import assert_parity, dev, gpu_mesh, host, np_dtype, oracle_problem

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


def _cube(n):
    w = wl.config4_sweep(16)
    w.n_cells = tuple(n)
    w.m0 = wl.random_unit_field(w.node_shape, 4 + sum(n))
    return w


@pytest.mark.parametrize("prec", ["f64", "f32"])
# (the last two: a 192-cell axis beside axes the persistent TMA pipelines serve -- k_py_* with 192 planes, k_pz_mid with
# 385 ky rows, k_px_* feeding k_fy_* with M = 12)
@pytest.mark.parametrize("n", [(192, 32, 16), (32, 192, 32), (32, 32, 192), (192, 64, 192), (32, 256, 192), (256, 192, 32)])
def test_native_192_axis_against_the_oracle(n, prec, monkeypatch):
    from oracle import llg
    td, nd = DT[prec], np_dtype(DT[prec])
    w = _cube(n)
    p = oracle_problem(w, nd)
    m = wl.round_to(w.m0, nd)
    ref_H = llg.effective_field(p, m)
    ref_f = llg.llg_rhs(p, 0.0, m, None)
    monkeypatch.setenv("NM_FAST192", "1")
    mesh = gpu_mesh(w, td)
    assert mesh.nm_debug_demag_path() == 1              # exact fast path, not embedded
    assert_parity(host(mesh.nm_heff(0.0, dev(m, td))), ref_H, TOL[prec], "H, native 192")
    assert_parity(host(mesh.nm_llg_rhs(0.0, dev(m, td))), ref_f, TOL[prec], "f, native 192")
    monkeypatch.delenv("NM_FAST192")
    other = gpu_mesh(w, td)
    assert other.nm_debug_demag_path() in (0, 2)        # zero-extended to 256 (or the general path)
    assert_parity(host(other.nm_heff(0.0, dev(m, td))), ref_H, TOL[prec], "H, default")


@pytest.mark.parametrize("n,prec", [((192, 32, 32), "f32"), ((32, 192, 32), "f32"), ((32, 32, 192), "f32"),
                                    ((32, 32, 192), "f64"), ((192, 192, 32), "f64")])
def test_native_192_guard_bands_and_run_to_run_identity(n, prec, monkeypatch):
    """The checks of tests/test_gpu_guards.py on the 192-cell kernels (k_fx_* / k_fy_* / k_fz_mid with M = 12, k_pz_mid3):
    inputs inside NaN slabs, outputs and the workspace inside canary slabs, every entry point three times over --
    finite, canaries intact, repetitions bit-identical, guarded equal to plain."""
    import test_gpu_guards as gg
    monkeypatch.setenv("NM_FAST192", "1")
    make = lambda: gg._cube(n)
    reps, out_ok, ws_ok, path = gg._run(make, prec, guarded=True)
    assert path == 1 and ws_ok and out_ok
    for t_ in reps[0]:
        assert bool(torch.isfinite(t_).all()), "an input was read outside its array (NaN guard band)"
    for r in reps[1:]:
        for x, y in zip(reps[0], r):
            assert torch.equal(x, y), "results differ between identical runs"
    plain, _, ws_ok2, _ = gg._run(make, prec, guarded=False)
    assert ws_ok2
    for x, y in zip(reps[0], plain[0]):
        assert torch.equal(x, y), "guarded and plain runs differ"
