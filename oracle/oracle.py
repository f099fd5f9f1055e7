"""ctypes wrapper of the CPU oracle (oracle/gint_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package except nothing at all: inputs
arrive as plain numpy arrays (built by paper_2409_09399_b200.workloads, the shared seeded
input generator that holds none of the method's arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "gint_oracle.c")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (no tuning flags beyond that)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.oracle_pairs.restype = C.c_longlong
        _lib.oracle_threads.restype = C.c_int
    return _lib


def threads() -> int:
    return int(lib().oracle_threads())


def _basis_args(b):
    return (C.c_int(b.n_species), _p(np.ascontiguousarray(b.n_shell, np.int32), C.c_int),
            _p(np.ascontiguousarray(b.shell_l, np.int32), C.c_int), _p(np.ascontiguousarray(b.rcut, np.float64), C.c_double),
            C.c_double(b.dr), _p(np.ascontiguousarray(b.n_knot, np.int32), C.c_int),
            _p(np.ascontiguousarray(b.tab_y, np.float64), C.c_double), _p(np.ascontiguousarray(b.tab_y2, np.float64), C.c_double))


def phi(basis, species: int, d) -> np.ndarray:
    out = np.zeros(basis.norb[species])
    d = np.ascontiguousarray(d, np.float64)
    rc = lib().oracle_phi(*_basis_args(basis), C.c_int(species), _p(d, C.c_double), _p(out, C.c_double))
    assert rc >= 0
    return out


def pairs(w):
    """(A, B, R[n,3], offset[n+1]) in lexicographic order."""
    b = w.basis
    sp = np.ascontiguousarray(w.atom_species, np.int32)
    pos = np.ascontiguousarray(w.atom_pos, np.float64)
    cell = np.ascontiguousarray(w.cell, np.float64)
    head = (C.c_int(b.n_species), _p(np.ascontiguousarray(b.n_shell, np.int32), C.c_int),
            _p(np.ascontiguousarray(b.shell_l, np.int32), C.c_int), _p(np.ascontiguousarray(b.rcut, np.float64), C.c_double),
            C.c_int(len(sp)), _p(sp, C.c_int), _p(pos, C.c_double), _p(cell, C.c_double))
    n = lib().oracle_pairs(*head, None, None, None, None)
    assert n >= 0
    A = np.zeros(n, np.int32); B = np.zeros(n, np.int32); R = np.zeros((n, 3), np.int32); off = np.zeros(n + 1, np.int64)
    n2 = lib().oracle_pairs(*head, _p(A, C.c_int), _p(B, C.c_int), _p(R, C.c_int), _p(off, C.c_longlong))
    assert n2 == n
    return A, B, R, off


def _common(w):
    sp = np.ascontiguousarray(w.atom_species, np.int32)
    pos = np.ascontiguousarray(w.atom_pos, np.float64)
    cell = np.ascontiguousarray(w.cell, np.float64)
    mesh = np.ascontiguousarray(w.mesh, np.int32)
    keep = (sp, pos, cell, mesh)
    return keep, (C.c_int(len(sp)), _p(sp, C.c_int), _p(pos, C.c_double), _p(cell, C.c_double), _p(mesh, C.c_int))


def vlocal(w, V, plist, sel=None, H=None) -> np.ndarray:
    """H values (all blocks, or only the pair indices in `sel`; other entries stay as given / zero)."""
    A, B, R, off = plist
    V = np.ascontiguousarray(V, np.float64)
    assert V.size == w.n_points
    if H is None:
        H = np.zeros(int(off[-1]))
    keep, geo = _common(w)
    if sel is None:
        nsel, selp = C.c_longlong(0), None
    else:
        sel = np.ascontiguousarray(sel, np.int64); nsel, selp = C.c_longlong(len(sel)), _p(sel, C.c_longlong)
    Rc = np.ascontiguousarray(R, np.int32)
    rc = lib().oracle_vlocal(*_basis_args(w.basis), *geo, _p(V, C.c_double), C.c_longlong(len(A)),
                             _p(A, C.c_int), _p(B, C.c_int), _p(Rc, C.c_int), _p(off, C.c_longlong),
                             _p(H, C.c_double), nsel, selp)
    assert rc == 0, rc
    return H


def rho(w, D, plist, sel=None, out=None) -> np.ndarray:
    """rho on the mesh (all points, or only the mesh indices in `sel`)."""
    A, B, R, off = plist
    D = np.ascontiguousarray(D, np.float64)
    assert D.size == off[-1]
    if out is None:
        out = np.zeros(w.n_points)
    keep, geo = _common(w)
    if sel is None:
        nsel, selp = C.c_longlong(0), None
    else:
        sel = np.ascontiguousarray(sel, np.int64); nsel, selp = C.c_longlong(len(sel)), _p(sel, C.c_longlong)
    Rc = np.ascontiguousarray(R, np.int32)
    rc = lib().oracle_rho(*_basis_args(w.basis), *geo, _p(D, C.c_double), C.c_longlong(len(A)),
                          _p(A, C.c_int), _p(B, C.c_int), _p(Rc, C.c_int), _p(off, C.c_longlong),
                          _p(out, C.c_double), nsel, selp)
    assert rc == 0, rc
    return out


def dphi(basis, species: int, d):
    """(values[norb], gradients[norb, 3]) of the orbitals of `species` at displacement d."""
    out = np.zeros(basis.norb[species]); grad = np.zeros((basis.norb[species], 3))
    d = np.ascontiguousarray(d, np.float64)
    rc = lib().oracle_dphi(*_basis_args(basis), C.c_int(species), _p(d, C.c_double), _p(out, C.c_double), _p(grad, C.c_double))
    assert rc >= 0
    return out, grad


def force_stress(w, V, D, plist, sel=None):
    """Pulay force F[n_atoms, 3] and stress sigma[3, 3] of the local-potential energy (Eq. 4 / Eq. 5, reading R15).
    sel: only the forces of these atoms (other rows stay zero; sigma is None)."""
    A, B, R, off = plist
    V = np.ascontiguousarray(V, np.float64); D = np.ascontiguousarray(D, np.float64)
    assert V.size == w.n_points and D.size == off[-1]
    F = np.zeros((w.n_atoms, 3)); sigma = np.zeros((3, 3))
    keep, geo = _common(w)
    if sel is None:
        nsel, selp = C.c_longlong(0), None
    else:
        sel = np.ascontiguousarray(sel, np.int64); nsel, selp = C.c_longlong(len(sel)), _p(sel, C.c_longlong)
    Rc = np.ascontiguousarray(R, np.int32)
    rc = lib().oracle_force_stress(*_basis_args(w.basis), *geo, _p(V, C.c_double), _p(D, C.c_double), C.c_longlong(len(A)),
                                   _p(A, C.c_int), _p(B, C.c_int), _p(Rc, C.c_int), _p(off, C.c_longlong),
                                   _p(F, C.c_double), _p(sigma, C.c_double), nsel, selp)
    assert rc == 0, rc
    return F, (sigma if sel is None else None)
