"""Thin ctypes binding of libnm.so with the names of include/nm.h.

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C-ABI.
PyTorch supplies device memory (`tensor.data_ptr()`) and the current stream, nothing else.
There is no fallback: if libnm.so is missing or a call fails, an exception is raised.

Arrays follow the ABI layout (include/nm.h): nodal vector fields [3][N3+1][N2+1][N1+1], cell
scalars [N3][N2][N1], x fastest, contiguous, in the mesh dtype, on the mesh device.
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnm.so")

NM_F32, NM_F64 = 0, 1
NM_OK, NM_EINVAL, NM_EUNSUPPORTED, NM_ECUDA, NM_ENOMEM = 0, -1, -2, -3, -4
NM_TERM_EXCHANGE, NM_TERM_DEMAG, NM_TERM_ANISO, NM_TERM_ZEEMAN = 1, 2, 4, 8
NM_TERM_DMI, NM_TERM_CUBIC, NM_TERM_RKKY = 16, 32, 64
NM_DMI_BULK, NM_DMI_INTERFACIAL = 0, 1
NM_RK4, NM_DOPRI5 = 0, 1

EXPORTS = ("nm_mesh_query_workspace", "nm_mesh_create", "nm_mesh_set_Ms", "nm_mesh_destroy",
           "nm_last_error", "nm_heff", "nm_llg_rhs", "nm_rk_step", "nm_llg_adjoint_rhs",
           "nm_adjoint_rk4_step", "nm_adjoint_add_objective", "nm_llg_adjoint_rhs_hext", "nm_adjoint_rk4_step_hext",
           "nm_llg_adjoint_rhs_materials", "nm_adjoint_rk4_step_ex", "nm_llg_adjoint_rhs_hnodal", "nm_debug_get_tensor", "nm_debug_get_cell_field",
           "nm_launch_count", "nm_profile_dropped", "nm_debug_demag_path", "nm_profile_class_count", "nm_profile_class_name", "nm_profile_begin",
           "nm_profile_end", "nm_hext_gradient_noalloc")


class nm_mesh_desc(ctypes.Structure):
    _fields_ = [("n_cells", ctypes.c_int * 3),
                ("cell_size", ctypes.c_double * 3),
                ("dtype", ctypes.c_int),
                ("device", ctypes.c_int),
                ("terms", ctypes.c_uint),
                ("gamma", ctypes.c_double),
                ("alpha", ctypes.c_double),
                ("ku_axis", ctypes.c_double * 3),
                ("Ms", ctypes.c_void_p), ("A", ctypes.c_void_p), ("Ku", ctypes.c_void_p),
                ("Ms_scalar", ctypes.c_double), ("A_scalar", ctypes.c_double),
                ("Ku_scalar", ctypes.c_double),
                ("basis", ctypes.c_int),
                ("D", ctypes.c_void_p), ("Kc", ctypes.c_void_p),
                ("D_scalar", ctypes.c_double), ("Kc_scalar", ctypes.c_double),
                ("dmi_kind", ctypes.c_int), ("dmi_normal", ctypes.c_int),
                ("cubic_axes", ctypes.c_double * 9),
                ("rkky_J", ctypes.c_double), ("rkky_planes", ctypes.c_int * 2)]


AMP_FUNC = ctypes.CFUNCTYPE(ctypes.c_double, ctypes.c_double, ctypes.c_void_p)


class nm_zeeman(ctypes.Structure):
    _fields_ = [("h_static", ctypes.c_void_p), ("h_pulse", ctypes.c_void_p),
                ("h_uniform", ctypes.c_double * 3),
                ("amp", AMP_FUNC), ("user", ctypes.c_void_p)]


class nm_adjoint_extra(ctypes.Structure):
    _fields_ = [("u_A", ctypes.c_void_p), ("u_Ku", ctypes.c_void_p), ("u_h", ctypes.c_void_p),
                ("u_hn", ctypes.c_void_p)]


class NmError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("nm status %d: %s" % (status, message))
        self.status = status


_lib = None


def lib():
    """Load libnm.so (built by paper_2411_11725_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libnm.so not found at %s: run `python -m paper_2411_11725_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, dbl, i32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
        L.nm_last_error.restype = ctypes.c_char_p
        L.nm_last_error.argtypes = []
        L.nm_mesh_query_workspace.argtypes = [ctypes.POINTER(nm_mesh_desc), ctypes.POINTER(ctypes.c_size_t)]
        L.nm_mesh_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(nm_mesh_desc), vp, ctypes.c_size_t]
        L.nm_mesh_set_Ms.argtypes = [vp, vp, vp]
        L.nm_mesh_destroy.argtypes = [vp]
        L.nm_heff.argtypes = [vp, dbl, vp, ctypes.POINTER(nm_zeeman), vp, vp]
        L.nm_llg_rhs.argtypes = [vp, dbl, vp, ctypes.POINTER(nm_zeeman), vp, vp]
        L.nm_rk_step.argtypes = [vp, i32, dbl, dbl, vp, ctypes.POINTER(nm_zeeman), i32, dbl, dbl,
                                 ctypes.POINTER(dbl), vp]
        L.nm_llg_adjoint_rhs.argtypes = [vp, dbl, vp, vp, ctypes.POINTER(nm_zeeman), vp, vp, vp, vp]
        L.nm_adjoint_rk4_step.argtypes = [vp, dbl, dbl, vp, vp, vp, ctypes.POINTER(nm_zeeman), i32, vp]
        L.nm_adjoint_add_objective.argtypes = [vp, vp, vp, dbl, vp]
        L.nm_llg_adjoint_rhs_hext.argtypes = [vp, vp, vp, vp, vp]
        L.nm_llg_adjoint_rhs_hnodal.argtypes = [vp, vp, vp, vp, vp]
        L.nm_llg_adjoint_rhs_materials.argtypes = [vp, vp, vp, vp, vp, vp]
        L.nm_adjoint_rk4_step_ex.argtypes = [vp, dbl, dbl, vp, vp, vp, ctypes.POINTER(nm_adjoint_extra),
                                             ctypes.POINTER(nm_zeeman), i32, vp]
        L.nm_adjoint_rk4_step_hext.argtypes = [vp, dbl, dbl, vp, vp, vp, vp, ctypes.POINTER(nm_zeeman), i32, vp]
        L.nm_hext_gradient_noalloc.argtypes = [i32, i32, ctypes.POINTER(i32), vp, vp, vp, dbl, dbl, vp, vp]
        L.nm_debug_get_tensor.argtypes = [vp, vp]
        L.nm_debug_get_cell_field.argtypes = [vp, vp, vp]
        L.nm_launch_count.argtypes = [vp]
        L.nm_launch_count.restype = ctypes.c_longlong
        L.nm_profile_dropped.argtypes = [vp]
        L.nm_profile_dropped.restype = ctypes.c_longlong
        L.nm_debug_demag_path.argtypes = [vp]
        L.nm_debug_demag_path.restype = ctypes.c_int
        L.nm_profile_class_count.argtypes = []
        L.nm_profile_class_name.argtypes = [i32]
        L.nm_profile_class_name.restype = ctypes.c_char_p
        L.nm_profile_begin.argtypes = [vp]
        L.nm_profile_end.argtypes = [vp, vp, ctypes.POINTER(dbl), ctypes.POINTER(ctypes.c_longlong)]
        for name in EXPORTS:
            if name not in ("nm_last_error", "nm_launch_count", "nm_profile_dropped", "nm_profile_dropped", "nm_debug_demag_path", "nm_profile_class_name"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _check(status):
    if status != NM_OK:
        raise NmError(status, lib().nm_last_error().decode("utf-8", "replace"))


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else None


def _stream(device):
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def make_desc(n_cells, cell_size, dtype, device, terms, gamma, alpha, ku_axis=(0.0, 0.0, 1.0),
              Ms=None, A=None, Ku=None, basis=3, D=None, Kc=None, dmi_kind=NM_DMI_BULK, dmi_normal=2,
              cubic_axes=(1.0, 0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0), rkky_J=0.0, rkky_planes=(0, 0)):
    """Fill an nm_mesh_desc.  Ms/A/Ku/D/Kc: python scalar or a device tensor [N3][N2][N1]."""
    d = nm_mesh_desc()
    d.n_cells[:] = [int(v) for v in n_cells]
    d.cell_size[:] = [float(v) for v in cell_size]
    d.dtype = NM_F64 if dtype == torch.float64 else NM_F32
    d.device = int(device)
    d.terms = int(terms)
    d.gamma, d.alpha = float(gamma), float(alpha)
    d.ku_axis[:] = [float(v) for v in ku_axis]
    d.basis = int(basis)
    d.dmi_kind, d.dmi_normal = int(dmi_kind), int(dmi_normal)
    d.rkky_J = float(rkky_J)
    d.rkky_planes[:] = [int(v) for v in rkky_planes]
    d.cubic_axes[:] = [float(v) for row in cubic_axes for v in (row if hasattr(row, "__len__") else (row,))]
    keep = []
    for name, v in (("Ms", Ms), ("A", A), ("Ku", Ku), ("D", D), ("Kc", Kc)):
        if torch.is_tensor(v):
            assert v.is_cuda and v.is_contiguous() and v.dtype == dtype, name
            setattr(d, name, v.data_ptr())
            keep.append(v)
        else:
            setattr(d, name, None)
            setattr(d, name + "_scalar", float(v) if v is not None else 0.0)
    d._keep = keep
    return d


NM_NOALLOC_MAX_NODES = 1 << 25


def nm_hext_gradient_noalloc(n_cells, m, a, Ms=None, gamma=2.211e5, alpha=0.0, out=None):
    """-(df/dh)^T a for a uniform external field without a mesh, a workspace or any allocation inside the library
    (include/nm.h).  m, a: CUDA nodal fields in ABI order; Ms: CUDA cell array or None; out: CUDA fp64 [3] (made here
    if None -- pass one to keep the call itself allocation-free)."""
    if out is None:
        out = torch.empty(3, dtype=torch.float64, device=m.device)
    assert out.dtype == torch.float64 and out.numel() == 3 and out.is_cuda
    dev = m.device.index if m.device.index is not None else torch.cuda.current_device()
    n = (ctypes.c_int * 3)(*[int(v) for v in n_cells])
    _check(lib().nm_hext_gradient_noalloc(dev, NM_F64 if m.dtype == torch.float64 else NM_F32, n, _ptr(m), _ptr(a),
                                          _ptr(Ms), float(gamma), float(alpha), _ptr(out), _stream(dev)))
    return out


def nm_mesh_query_workspace(desc):
    n = ctypes.c_size_t(0)
    _check(lib().nm_mesh_query_workspace(ctypes.byref(desc), ctypes.byref(n)))
    return n.value


class Zeeman:
    """Owner of an nm_zeeman struct: H_ext(t, n) = h_uniform + h_static[n] + amp(t) h_pulse[n]."""

    def __init__(self, h_uniform=(0.0, 0.0, 0.0), h_static=None, h_pulse=None, amp=None):
        self._keep = (h_static, h_pulse, amp)
        z = nm_zeeman()
        z.h_static = h_static.data_ptr() if h_static is not None else None
        z.h_pulse = h_pulse.data_ptr() if h_pulse is not None else None
        z.h_uniform[:] = [float(v) for v in h_uniform]
        self._cb = AMP_FUNC(lambda t, user: float(amp(t))) if amp is not None else AMP_FUNC()
        z.amp = self._cb
        z.user = None
        self.struct = z


def _zref(z):
    return ctypes.byref(z.struct) if z is not None else None


class Mesh:
    """nm_mesh handle plus the torch-allocated workspace block it lives in."""

    def __init__(self, n_cells, cell_size, dtype=torch.float32, device=0, terms=3, gamma=2.211e5,
                 alpha=0.0, ku_axis=(0.0, 0.0, 1.0), Ms=None, A=None, Ku=None, workspace=None, basis=3,
                 D=None, Kc=None, dmi_kind=NM_DMI_BULK, dmi_normal=2,
                 cubic_axes=(1.0, 0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0), rkky_J=0.0, rkky_planes=(0, 0)):
        """workspace: optional caller-made uint8 device tensor (256-byte aligned start, at least
        nm_mesh_query_workspace bytes) to build the mesh in, instead of one allocated here."""
        self.dtype = dtype
        self.device = int(device)
        self.n_cells = tuple(int(v) for v in n_cells)
        self.basis = int(basis) or 3
        self.node_shape_abi = (3, self.n_cells[2] + 1 if self.basis > 2 else 1,
                               self.n_cells[1] + 1 if self.basis > 1 else 1, self.n_cells[0] + 1)
        self.cell_shape_abi = (self.n_cells[2], self.n_cells[1], self.n_cells[0])
        desc = make_desc(n_cells, cell_size, dtype, device, terms, gamma, alpha, ku_axis, Ms, A, Ku, basis,
                         D, Kc, dmi_kind, dmi_normal, cubic_axes, rkky_J, rkky_planes)
        nbytes = nm_mesh_query_workspace(desc)
        self.workspace_bytes = nbytes
        if workspace is None:
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda:%d" % self.device)
            base = (self.workspace.data_ptr() + 255) & ~255
        else:
            assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.numel() >= nbytes
            assert workspace.data_ptr() % 256 == 0
            self.workspace = workspace
            base = workspace.data_ptr()
        h = ctypes.c_void_p()
        torch.cuda.synchronize(self.device)
        _check(lib().nm_mesh_create(ctypes.byref(h), ctypes.byref(desc), ctypes.c_void_p(base), nbytes))
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib().nm_mesh_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C-ABI calls, same names ----
    def nm_mesh_set_Ms(self, Ms):
        _check(lib().nm_mesh_set_Ms(self.handle, _ptr(Ms), _stream(self.device)))

    def nm_heff(self, t, m, zeeman=None, out=None):
        out = torch.empty_like(m) if out is None else out
        _check(lib().nm_heff(self.handle, float(t), _ptr(m), _zref(zeeman), _ptr(out), _stream(self.device)))
        return out

    def nm_llg_rhs(self, t, m, zeeman=None, out=None):
        out = torch.empty_like(m) if out is None else out
        _check(lib().nm_llg_rhs(self.handle, float(t), _ptr(m), _zref(zeeman), _ptr(out), _stream(self.device)))
        return out

    def nm_rk_step(self, scheme, t, dt, m, zeeman=None, renormalise=True, rtol=1e-5, atol=1e-5,
                   want_err=False):
        err = ctypes.c_double(0.0)
        _check(lib().nm_rk_step(self.handle, int(scheme), float(t), float(dt), _ptr(m), _zref(zeeman),
                                1 if renormalise else 0, float(rtol), float(atol),
                                ctypes.byref(err) if want_err else None, _stream(self.device)))
        return err.value if want_err else None

    def nm_llg_adjoint_rhs(self, t, m, a, zeeman=None, want_f=True, want_u=True):
        f = torch.empty_like(m) if want_f else None
        dadt = torch.empty_like(m)
        dudt = torch.empty(self.cell_shape_abi, dtype=self.dtype, device=m.device) if want_u else None
        _check(lib().nm_llg_adjoint_rhs(self.handle, float(t), _ptr(m), _ptr(a), _zref(zeeman), _ptr(f),
                                        _ptr(dadt), _ptr(dudt), _stream(self.device)))
        return f, dadt, dudt

    def nm_adjoint_rk4_step(self, t, dt, m, a, u, zeeman=None, renormalise=True):
        _check(lib().nm_adjoint_rk4_step(self.handle, float(t), float(dt), _ptr(m), _ptr(a), _ptr(u),
                                         _zref(zeeman), 1 if renormalise else 0, _stream(self.device)))

    def nm_llg_adjoint_rhs_hext(self, m, a):
        out = torch.empty(3, dtype=torch.float64, device=m.device)
        _check(lib().nm_llg_adjoint_rhs_hext(self.handle, _ptr(m), _ptr(a), _ptr(out), _stream(self.device)))
        return out

    def nm_adjoint_rk4_step_hext(self, t, dt, m, a, u, u_h, zeeman=None, renormalise=True):
        assert u_h.dtype == torch.float64 and u_h.numel() == 3 and u_h.is_cuda
        _check(lib().nm_adjoint_rk4_step_hext(self.handle, float(t), float(dt), _ptr(m), _ptr(a), _ptr(u),
                                              _ptr(u_h), _zref(zeeman), 1 if renormalise else 0,
                                              _stream(self.device)))

    def nm_llg_adjoint_rhs_materials(self, m, a, want_A=True, want_Ku=True):
        gA = torch.empty(self.cell_shape_abi, dtype=self.dtype, device=m.device) if want_A else None
        gKu = torch.empty(self.cell_shape_abi, dtype=self.dtype, device=m.device) if want_Ku else None
        _check(lib().nm_llg_adjoint_rhs_materials(self.handle, _ptr(m), _ptr(a), _ptr(gA), _ptr(gKu),
                                                  _stream(self.device)))
        return gA, gKu

    def nm_llg_adjoint_rhs_hnodal(self, m, a):
        out = torch.empty_like(m)
        _check(lib().nm_llg_adjoint_rhs_hnodal(self.handle, _ptr(m), _ptr(a), _ptr(out), _stream(self.device)))
        return out

    def nm_adjoint_rk4_step_ex(self, t, dt, m, a, u, u_A=None, u_Ku=None, u_h=None, zeeman=None,
                               renormalise=True, u_hn=None):
        ex = nm_adjoint_extra()
        ex.u_A = u_A.data_ptr() if u_A is not None else None
        ex.u_Ku = u_Ku.data_ptr() if u_Ku is not None else None
        ex.u_h = u_h.data_ptr() if u_h is not None else None
        ex.u_hn = u_hn.data_ptr() if u_hn is not None else None
        _check(lib().nm_adjoint_rk4_step_ex(self.handle, float(t), float(dt), _ptr(m), _ptr(a), _ptr(u),
                                            ctypes.byref(ex), _zref(zeeman), 1 if renormalise else 0,
                                            _stream(self.device)))

    def nm_adjoint_add_objective(self, a, dLdm, scale=1.0):
        _check(lib().nm_adjoint_add_objective(self.handle, _ptr(a), _ptr(dLdm), float(scale),
                                              _stream(self.device)))

    def nm_debug_get_tensor(self):
        import numpy as np
        out = np.empty((6,) + self.cell_shape_abi, dtype=np.float64)
        _check(lib().nm_debug_get_tensor(self.handle, ctypes.c_void_p(out.ctypes.data)))
        return out

    def nm_debug_get_cell_field(self):
        out = torch.empty((3,) + self.cell_shape_abi, dtype=self.dtype, device="cuda:%d" % self.device)
        _check(lib().nm_debug_get_cell_field(self.handle, _ptr(out), _stream(self.device)))
        return out

    def nm_launch_count(self):
        return int(lib().nm_launch_count(self.handle))

    def nm_profile_dropped(self):
        return int(lib().nm_profile_dropped(self.handle))

    def nm_debug_demag_path(self):
        return int(lib().nm_debug_demag_path(self.handle))

    def nm_profile_begin(self):
        _check(lib().nm_profile_begin(self.handle))

    def nm_profile_end(self):
        """{class name: (milliseconds, launches)} since nm_profile_begin; synchronises the stream."""
        n = lib().nm_profile_class_count()
        ms = (ctypes.c_double * n)()
        cnt = (ctypes.c_longlong * n)()
        _check(lib().nm_profile_end(self.handle, _stream(self.device), ms, cnt))
        return {lib().nm_profile_class_name(i).decode(): (ms[i], int(cnt[i])) for i in range(n)}
