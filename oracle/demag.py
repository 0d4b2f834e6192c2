"""Demagnetisation field of the nodal scheme (oracle, fp64).

Test infrastructure only; see oracle/__init__.py.

PAPER.md:175-181 (Sec. III B): the field of homogeneously magnetised cuboidal cells is computed
by FFT-accelerated convolution on the cell grid; a pre- and post-processing step "averages the
values to transition between nodal and cell-centered discretizations".

C4  demag tensor N(c - c'): newell_quad.c (Newell closed form, evaluated in __float128).
C5  M_c  = Ms_c * (1/8) (S^T m)_c        (exact cell mean of the trilinear m^h)
    H_c  = - sum_c' N(c - c') M_c'       (zero-padded FFT convolution, P_d = 2 N_d, or 1 if N_d = 1;
                                          "for 2D computations ... the FFT also reduces to two
                                          dimensions")
    H^d_n = (S (Ms o H^cell))_n / (S Ms)_n   (reading C5: the cell-wise constant field put through
                                          the weak form (7) and lumped (22); plain mean over the
                                          1..8 existing cells when Ms is uniform)
"""
import ctypes
import os
import subprocess

import numpy as np

from .mesh import gather_nodes_to_cells, scatter_cells_to_nodes

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

# component order of the symmetric tensor: index a -> (row, column)
COMPONENTS = ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))


def build_newell_quad(force=False):
    """Compile newell_quad.c next to its source (gcc + libquadmath); returns the .so path."""
    src = os.path.join(_HERE, "newell_quad.c")
    so = os.path.join(_HERE, "_newell_quad.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        tmp = so + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", src,
                               "-lquadmath", "-lm", "-o", tmp])
        os.replace(tmp, so)
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_newell_quad())
        _LIB.newell_tensor_quad.restype = ctypes.c_int
        _LIB.newell_tensor_quad.argtypes = [ctypes.POINTER(ctypes.c_int),
                                            ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]
        _LIB.newell_tensor_quad_at.restype = ctypes.c_int
        _LIB.newell_tensor_quad_at.argtypes = [ctypes.c_void_p, ctypes.c_long,
                                               ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]
    return _LIB


def demag_tensor(n_cells, dx):
    """N[a, p1, p2, p3] for non-negative cell offsets p_d = 0..N_d-1, a in COMPONENTS order."""
    n = (ctypes.c_int * 3)(*[int(v) for v in n_cells])
    d = (ctypes.c_double * 3)(*[float(v) for v in dx])
    out = np.empty((6,) + tuple(int(v) for v in n_cells), dtype=np.float64)
    rc = _lib().newell_tensor_quad(n, d, out.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise MemoryError("newell_tensor_quad")
    return out


def demag_tensor_at(offsets, dx):
    """N[k, a] at the signed cell offsets offsets[k] = (p1, p2, p3), a in COMPONENTS order: the
    same closed form as demag_tensor, evaluated offset by offset (for sampled checks on grids
    whose full table would take minutes)."""
    p = np.ascontiguousarray(np.asarray(offsets, dtype=np.int32).reshape(-1, 3))
    d = (ctypes.c_double * 3)(*[float(v) for v in dx])
    out = np.empty((p.shape[0], 6), dtype=np.float64)
    _lib().newell_tensor_quad_at(p.ctypes.data_as(ctypes.c_void_p), p.shape[0], d,
                                 out.ctypes.data_as(ctypes.c_void_p))
    return out


def tensor_at(Nt, a, p):
    """N_a at a signed cell offset p: diagonal components are even in every argument, the
    off-diagonal component (r,s) is odd in arguments r and s and even in the third."""
    r, s = COMPONENTS[a]
    sign = 1.0
    if r != s:
        for d in (r, s):
            if p[d] < 0:
                sign = -sign
    return sign * Nt[a, abs(p[0]), abs(p[1]), abs(p[2])]


def signed_component(Nt, a):
    """Component a of the tensor over signed offsets p_d = -(N_d-1)..N_d-1, stored at index
    p_d + N_d - 1 (shape 2 N_d - 1 per axis): the parity rule of tensor_at applied to the table."""
    n = Nt.shape[1:]
    idx = [np.abs(np.arange(-(k - 1), k)) for k in n]
    sgn = [np.sign(np.arange(-(k - 1), k) + 0.5) for k in n]
    r, s = COMPONENTS[a]
    blk = Nt[a][np.ix_(idx[0], idx[1], idx[2])]
    if r != s:
        sg = [np.ones(2 * k - 1) for k in n]
        sg[r] = sgn[r]
        sg[s] = sgn[s]
        blk = blk * sg[0][:, None, None] * sg[1][None, :, None] * sg[2][None, None, :]
    return blk


def signed_tensor(Nt):
    """Full array N[a, p1, p2, p3] over signed offsets (all six components of signed_component)."""
    return np.stack([signed_component(Nt, a) for a in range(6)])


def cell_magnetization(m, Ms):
    """M_c = Ms_c * (1/8) sum_i m_{c+i} (C5)."""
    return Ms * gather_nodes_to_cells(m) / 8.0


def demag_field_cells_direct(M, Nt):
    """H_c = - sum_c' N(c - c') M_c' by brute force, O(N_cells^2).  Tiny grids only."""
    n = M.shape[1:]
    Ns = signed_tensor(Nt)
    H = np.zeros_like(M, dtype=np.float64)
    for c1 in range(n[0]):
        for c2 in range(n[1]):
            for c3 in range(n[2]):
                # offsets c - c' for every c': index (c - c') + N - 1
                win = Ns[:, c1 + n[0] - 1 - np.arange(n[0])][:, :, c2 + n[1] - 1 - np.arange(n[1])][
                    :, :, :, c3 + n[2] - 1 - np.arange(n[2])]
                for a, (r, s) in enumerate(COMPONENTS):
                    H[r, c1, c2, c3] -= np.sum(win[a] * M[s])
                    if r != s:
                        H[s, c1, c2, c3] -= np.sum(win[a] * M[r])
    return H


def demag_field_cells_fft(M, Nt):
    """The same sum as a zero-padded circular convolution.

    The kernel is laid out on the padded grid at index (p mod P_d) for the signed offsets
    p_d = -(N_d-1)..N_d-1; axes with N_d = 1 are not padded (P_d = 1).  The six tensor components
    are laid out and transformed one after the other (memory only: a 256^3 mesh then needs one
    padded kernel array at a time instead of six)."""
    n = M.shape[1:]
    P = tuple(2 * k if k > 1 else 1 for k in n)
    idx = [np.arange(-(k - 1), k) % p for k, p in zip(n, P)]
    Mp = np.zeros((3,) + P)
    Mp[:, :n[0], :n[1], :n[2]] = M
    Mk = np.fft.rfftn(Mp, axes=(1, 2, 3))
    del Mp
    Hk = np.zeros_like(Mk)
    for a, (r, s) in enumerate(COMPONENTS):
        ker = np.zeros(P)
        ker[np.ix_(idx[0], idx[1], idx[2])] = signed_component(Nt, a)
        Nk = np.fft.rfftn(ker)
        del ker
        Hk[r] -= Nk * Mk[s]
        if r != s:
            Hk[s] -= Nk * Mk[r]
    del Mk
    Hp = np.fft.irfftn(Hk, s=P, axes=(1, 2, 3))
    return np.ascontiguousarray(Hp[:, :n[0], :n[1], :n[2]])


def demag_field_nodes(Hc, Ms):
    """H^d_n = (S (Ms o H^cell))_n / (S Ms)_n; nodes with S Ms = 0 get 0 (reading C3(iii))."""
    num = scatter_cells_to_nodes(Ms * Hc)
    den = scatter_cells_to_nodes(Ms)
    out = np.zeros_like(num)
    ok = den > 0
    out[:, ok] = num[:, ok] / den[ok]
    return out


def demag_field(m, Ms, Nt, direct=False):
    """Nodal demag field of nodal m: average -> convolution -> average."""
    M = cell_magnetization(m, Ms)
    Hc = demag_field_cells_direct(M, Nt) if direct else demag_field_cells_fft(M, Nt)
    return demag_field_nodes(Hc, Ms)
