"""CPU-only checks of the C-ABI boundary: libnm.so loads, exports every symbol include/nm.h
declares, and its host-only entry points validate their arguments (no compute, no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nm():
    from paper_2411_11725_b200 import build
    build.build()
    from paper_2411_11725_b200 import binding
    binding.lib()
    return binding


def _declared():
    src = open(os.path.join(ROOT, "include", "nm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nm_[A-Za-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(nm):
    names = _declared()
    for required in ("nm_mesh_create", "nm_heff", "nm_llg_rhs", "nm_rk_step", "nm_llg_adjoint_rhs"):
        assert required in names            # the five names north_star fixes
    raw = ctypes.CDLL(nm.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), n
    assert sorted(nm.EXPORTS) == names      # the binding covers exactly the header


def test_binding_struct_matches_header_layout(nm):
    # field order of nm_mesh_desc / nm_zeeman as declared in nm.h
    assert [f[0] for f in nm.nm_mesh_desc._fields_] == [
        "n_cells", "cell_size", "dtype", "device", "terms", "gamma", "alpha", "ku_axis", "Ms", "A",
        "Ku", "Ms_scalar", "A_scalar", "Ku_scalar", "basis", "D", "Kc", "D_scalar", "Kc_scalar", "dmi_kind",
        "dmi_normal", "cubic_axes", "rkky_J", "rkky_planes"]
    assert [f[0] for f in nm.nm_zeeman._fields_] == ["h_static", "h_pulse", "h_uniform", "amp", "user"]


def _desc(nm, n=(8, 8, 8), terms=3, dtype_f64=False, dx=(1e-9, 1e-9, 1e-9)):
    import torch
    return nm.make_desc(n, dx, torch.float64 if dtype_f64 else torch.float32, 0, terms, 2.211e5, 0.1,
                        Ms=8e5, A=1.3e-11, Ku=0.0)


def test_query_workspace_validates(nm):
    assert nm.nm_mesh_query_workspace(_desc(nm)) > 0
    # fp64 needs more than fp32; the demag term needs more than exchange alone
    assert nm.nm_mesh_query_workspace(_desc(nm, dtype_f64=True)) > nm.nm_mesh_query_workspace(_desc(nm))
    assert nm.nm_mesh_query_workspace(_desc(nm, terms=3)) > nm.nm_mesh_query_workspace(_desc(nm, terms=1))
    for bad, status in ((dict(n=(0, 8, 8)), nm.NM_EINVAL), (dict(terms=0), nm.NM_EINVAL),
                        (dict(terms=128), nm.NM_EINVAL), (dict(dx=(1e-9, 0.0, 1e-9)), nm.NM_EINVAL),
                        (dict(n=(11, 8, 8)), nm.NM_EUNSUPPORTED), (dict(n=(8, 13, 8), terms=2), nm.NM_EUNSUPPORTED)):
        with pytest.raises(nm.NmError) as e:
            nm.nm_mesh_query_workspace(_desc(nm, **bad))
        assert e.value.status == status, bad
        assert str(e.value)
    # sizes that are not 2^a 3^b 5^c 7^d are fine without the demag term
    assert nm.nm_mesh_query_workspace(_desc(nm, n=(7, 5, 11), terms=1)) > 0
    assert nm.nm_mesh_query_workspace(_desc(nm, n=(10, 7, 35), terms=3)) > 0


def test_workspace_grows_with_the_grid(nm):
    a = nm.nm_mesh_query_workspace(_desc(nm, n=(16, 16, 16)))
    b = nm.nm_mesh_query_workspace(_desc(nm, n=(32, 32, 32)))
    assert 6 * a < b < 10 * a
    # 256^3 fp32 fits one 180 GB GPU with a wide margin
    assert nm.nm_mesh_query_workspace(_desc(nm, n=(256, 256, 256))) < 16 * 2 ** 30


def test_missing_library_fails_loudly(nm, monkeypatch):
    monkeypatch.setattr(nm, "_lib", None)
    monkeypatch.setattr(nm, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libnm.so"))
    with pytest.raises(ImportError):
        nm.lib()
