"""nm_hext_gradient_noalloc (include/nm.h): the uniform-field gradient without a mesh, a workspace or any allocation,
its partial sums in a file-scope device array of libnm.so.  Checked against the existing path
(nm_llg_adjoint_rhs_hext on a mesh, itself held to the oracle in tests/test_gpu_parity.py) on calls in a row that
share the scratch array, and against the oracle directly.

Collected last on purpose (test_zz_*): the suite runs with `pytest -x`, so a failure here hides nothing."""
import numpy as np
import pytest

from paper_2411_11725_b200 import workloads as wl

from _sides import dev, gpu_mesh, np_dtype, oracle_problem

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"f32": 1e-5, "f64": 1e-11}
DT = {"f32": torch.float32, "f64": torch.float64}


def _inputs(n, prec, seed, vacuum):
    td, nd = DT[prec], np_dtype(DT[prec])
    w, _ = wl.varied_case(n, vacuum=vacuum)
    m = wl.round_to(w.m0, nd)
    a = wl.round_to(np.random.default_rng(seed).standard_normal(m.shape), nd)
    return w, m, a, td, nd


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_noalloc_matches_the_mesh_path_on_calls_in_a_row(prec):
    """Three calls in a row on one stream: a mesh that needs several blocks of partial sums, then a smaller one (the
    array still holds the first call's sums beyond what the second overwrites), then the first again; each against
    nm_llg_adjoint_rhs_hext on a mesh of the same inputs, within the tolerance of the parity tests."""
    from paper_2411_11725_b200 import binding as nm
    cases = [((40, 24, 12), 71, True), ((9, 7, 3), 72, True), ((40, 24, 12), 73, True)]
    out = torch.empty(3, dtype=torch.float64, device="cuda:0")
    got, ref = [], []
    for k, (n, seed, vac) in enumerate(cases):
        w, m, a, td, nd = _inputs(n, prec, seed, vac)
        md, ad, Msd = dev(m, td), dev(a, td), dev(wl.round_to(w.Ms, nd), td)
        assert (w.Ms == 0).any()
        mesh = gpu_mesh(w, td)
        ref.append(mesh.nm_llg_adjoint_rhs_hext(md, ad).cpu().numpy())
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(0)[0]
        nm.nm_hext_gradient_noalloc(n, md, ad, Msd, gamma=w.gamma, alpha=w.alpha, out=out)
        torch.cuda.synchronize()
        if k > 0:       # (the first call may load the two kernels)
            assert torch.cuda.mem_get_info(0)[0] >= free0, "the call took device memory"
        got.append(out.cpu().numpy().copy())
    for g, r in zip(got, ref):
        assert np.all(np.isfinite(g)) and np.max(np.abs(r)) > 0
        assert np.max(np.abs(g - r)) <= TOL[prec] * np.max(np.abs(r)), (g, r)
    assert not np.array_equal(got[0], got[2])       # different a: the third call is not the first one's leftovers


def test_noalloc_against_the_oracle_and_without_ms_array():
    """fp64 against oracle adjoint_rhs_hext on a mesh with vacuum nodes; Ms = NULL counts every node."""
    from oracle import adjoint
    from paper_2411_11725_b200 import binding as nm
    n = (17, 9, 5)
    w, m, a, td, nd = _inputs(n, "f64", 74, True)
    p = oracle_problem(w, nd)
    assert np.any(p.L == 0)
    ref = adjoint.adjoint_rhs_hext(p, 0.0, m, a)
    got = nm.nm_hext_gradient_noalloc(n, dev(m, td), dev(a, td), dev(w.Ms, td), gamma=w.gamma, alpha=w.alpha).cpu().numpy()
    assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref))
    gp = w.gamma / (1 + w.alpha ** 2)
    mxa = np.cross(m, a, axis=0)
    b = gp * mxa - w.alpha * gp * np.cross(m, mxa, axis=0)
    every = nm.nm_hext_gradient_noalloc(n, dev(m, td), dev(a, td), None, gamma=w.gamma, alpha=w.alpha).cpu().numpy()
    assert np.max(np.abs(every + b.reshape(3, -1).sum(axis=1))) <= 1e-11 * np.max(np.abs(every))
    assert np.max(np.abs(every - got)) > 1e-6 * np.max(np.abs(every))      # the vacuum nodes do make a difference


def test_noalloc_rejects_what_the_fixed_array_cannot_hold():
    from paper_2411_11725_b200 import binding as nm
    small = torch.zeros((3, 2, 2, 2), dtype=torch.float32, device="cuda:0")
    # 323^3 nodes = 3.37e7 > 2^25: refused before anything is read (the arrays passed are far too small)
    with pytest.raises(nm.NmError) as e:
        nm.nm_hext_gradient_noalloc((322, 322, 322), small, small)
    assert e.value.status == nm.NM_EINVAL and "NM_NOALLOC_MAX_NODES" in str(e.value)
    with pytest.raises(nm.NmError) as e:
        nm.nm_hext_gradient_noalloc((4, 0, 4), small, small)
    assert e.value.status == nm.NM_EINVAL
    assert nm.NM_NOALLOC_MAX_NODES == 1 << 25
    # the largest cube the bench uses fits
    assert 257 ** 3 <= nm.NM_NOALLOC_MAX_NODES
