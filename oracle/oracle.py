"""ctypes wrapper over oracle/liboracle.so (TEST INFRASTRUCTURE; see ani_oracle.c).

All inputs are the fp32 arrays of `paper_2207_14276_b200.workloads`; hyper-parameters are the fp32
values of `AniParams`, converted exactly to fp64 here.  Nothing in this file does arithmetic of the
method: it marshals arguments and sums per-atom energies per molecule.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

_NR, _NAMAX, _NZMAX = 16, 8, 8


class _Params(C.Structure):
    _fields_ = [("rcr", C.c_double), ("rca", C.c_double), ("eta_r", C.c_double), ("eta_a", C.c_double),
                ("zeta", C.c_double), ("alpha", C.c_double),
                ("shf_r", C.c_double * _NR), ("shf_a", C.c_double * _NAMAX), ("shf_z", C.c_double * _NZMAX),
                ("n_a", C.c_int), ("n_z", C.c_int)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.ora_pairs.restype = C.c_int64
        lib.ora_pairs.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_double,
                                  C.c_void_p, C.c_void_p, C.c_int64]
        lib.ora_aev.restype = None
        lib.ora_aev.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p,
                                C.POINTER(_Params), C.c_void_p, C.c_int64, C.c_void_p]
        lib.ora_mlp.restype = None
        lib.ora_mlp.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int, C.c_double,
                                C.c_void_p, C.c_void_p]
        lib.ora_energy_forces.restype = None
        lib.ora_energy_forces.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p,
                                          C.POINTER(_Params), C.c_void_p, C.c_int, C.c_void_p, C.c_int64,
                                          C.c_void_p, C.c_void_p, C.c_void_p]
        lib.ora_aev_dim.restype = C.c_int
        lib.ora_net_params.restype = C.c_int
        lib.ora_num_threads.restype = C.c_int
        _lib = lib
    return _lib


AEV_DIM = 1008
NET_PARAMS = 338689


def num_threads() -> int:
    return int(_load().ora_num_threads())


def _params(p) -> _Params:
    q = _Params()
    q.rcr, q.rca = float(np.float32(p.rcr)), float(np.float32(p.rca))
    q.eta_r, q.eta_a = float(np.float32(p.eta_r)), float(np.float32(p.eta_a))
    q.zeta, q.alpha = float(np.float32(p.zeta)), float(np.float32(p.celu_alpha))
    for i in range(_NR):
        q.shf_r[i] = float(np.float32(p.shf_r[i]))
    q.n_a, q.n_z = len(p.shf_a), len(p.shf_z)
    assert q.n_a * q.n_z == 32 and q.n_a <= _NAMAX and q.n_z <= _NZMAX
    for i in range(q.n_a):
        q.shf_a[i] = float(np.float32(p.shf_a[i]))
    for i in range(q.n_z):
        q.shf_z[i] = float(np.float32(p.shf_z[i]))
    return q


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _mol_id(n: int, mol_offsets: Optional[np.ndarray]) -> Optional[np.ndarray]:
    if mol_offsets is None:
        return None
    off = np.asarray(mol_offsets, dtype=np.int64)
    return np.repeat(np.arange(off.size - 1, dtype=np.int32), np.diff(off)).astype(np.int32)


def _prep(pos, species, box):
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    species = np.ascontiguousarray(species, dtype=np.int32)
    box = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
    return pos, species, box


def pairs(pos, box, rc, mol_offsets=None):
    """Brute-force full pair list: (row_ptr int64 [N+1], col int32 [nnz]), columns ascending."""
    lib = _load()
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    box = None if box is None else np.ascontiguousarray(box, dtype=np.float32)
    n = pos.shape[0]
    mid = _mol_id(n, mol_offsets)
    rc = float(np.float32(rc))
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    nnz = lib.ora_pairs(_ptr(pos), n, _ptr(box), _ptr(mid), rc, _ptr(row_ptr), None, 0)
    col = np.zeros(max(int(nnz), 1), dtype=np.int32)
    got = lib.ora_pairs(_ptr(pos), n, _ptr(box), _ptr(mid), rc, _ptr(row_ptr), _ptr(col), int(nnz))
    assert got == nnz
    return row_ptr, col[:nnz]


def aev(pos, species, box, params, centres=None, mol_offsets=None):
    """AEV rows (fp64 [n_centres, 1008]) of the listed centres (default: all atoms)."""
    lib = _load()
    pos, species, box = _prep(pos, species, box)
    n = pos.shape[0]
    centres = np.arange(n, dtype=np.int32) if centres is None else np.ascontiguousarray(centres, dtype=np.int32)
    mid = _mol_id(n, mol_offsets)
    out = np.zeros((centres.size, AEV_DIM), dtype=np.float64)
    q = _params(params)
    lib.ora_aev(_ptr(pos), _ptr(species), n, _ptr(box), _ptr(mid), C.byref(q), _ptr(centres), centres.size, _ptr(out))
    return out


def mlp(aev_rows, species, weights, n_models, params, want_grad=True):
    """Networks on given AEV rows: (E [n], dE/dG [n,1008] or None), ensemble mean."""
    lib = _load()
    a = np.ascontiguousarray(aev_rows, dtype=np.float64)
    sp = np.ascontiguousarray(species, dtype=np.int32)
    w = np.ascontiguousarray(weights, dtype=np.float32)
    assert w.size == n_models * 7 * NET_PARAMS
    E = np.zeros(a.shape[0], dtype=np.float64)
    g = np.zeros_like(a) if want_grad else None
    lib.ora_mlp(_ptr(a), _ptr(sp), a.shape[0], _ptr(w), n_models, float(np.float32(params.celu_alpha)), _ptr(E), _ptr(g))
    return E, g


def energy_forces(pos, species, box, params, weights, n_models, centres=None, mol_offsets=None, want_dEdG=False):
    """(E_atom [n_centres], F [N,3], dEdG or None): atomic energies of the centres and the forces
    those centres exert on every atom.  With all atoms as centres these are the totals."""
    lib = _load()
    pos, species, box = _prep(pos, species, box)
    n = pos.shape[0]
    centres = np.arange(n, dtype=np.int32) if centres is None else np.ascontiguousarray(centres, dtype=np.int32)
    mid = _mol_id(n, mol_offsets)
    w = np.ascontiguousarray(weights, dtype=np.float32)
    assert w.size == n_models * 7 * NET_PARAMS
    E = np.zeros(centres.size, dtype=np.float64)
    F = np.zeros((n, 3), dtype=np.float64)
    g = np.zeros((centres.size, AEV_DIM), dtype=np.float64) if want_dEdG else None
    q = _params(params)
    lib.ora_energy_forces(_ptr(pos), _ptr(species), n, _ptr(box), _ptr(mid), C.byref(q), _ptr(w), n_models,
                          _ptr(centres), centres.size, _ptr(E), _ptr(F), _ptr(g))
    return E, F, g


def total_energy_forces(system, params, weights):
    """Convenience for a `workloads.System`: (E [max(1,n_mol)], F [N,3])."""
    E_atom, F, _ = energy_forces(system.pos, system.species, system.box, params, weights, system.n_models,
                                 mol_offsets=system.mol_offsets)
    if system.mol_offsets is None:
        return np.array([E_atom.sum()]), F
    off = np.asarray(system.mol_offsets, dtype=np.int64)
    return np.add.reduceat(E_atom, off[:-1]), F
