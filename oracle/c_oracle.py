"""ORACLE -- ctypes loader for oracle/nbody_oracle.c (test infrastructure, not product code).

`build()` compiles the C form with gcc (-O2, OpenMP, no fast-math);
`force()` / `predict()` call it on fp64 arrays.  The arithmetic is in the .c
file; this module only marshals arguments.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nbody_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_D = ctypes.POINTER(ctypes.c_double)
_I = ctypes.POINTER(ctypes.c_int64)


def build(force_rebuild: bool = False) -> str:
    if force_rebuild or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_force.restype = ctypes.c_int
        _lib.oracle_force.argtypes = [ctypes.c_int64, _D, _D, _D, ctypes.c_double, ctypes.c_int64, _I,
                                      _D, _D, ctypes.c_uint, _D, _D, _D]
        _lib.oracle_predict.restype = ctypes.c_int
        _lib.oracle_predict.argtypes = [ctypes.c_int64, ctypes.c_double, _D, _D, _D, _D, _D, _D, _D]
        _lib.oracle_nearest.restype = ctypes.c_int
        _lib.oracle_nearest.argtypes = [ctypes.c_int64, _D, ctypes.c_int64, _I, _D, _I, _D]
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(_D)


def _c64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def force(m, x, v, eps, i_index=None, want_jerk=True, xi=None, vi=None):
    lib = _load()
    m, x, v, xi, vi = _c64(m), _c64(x), _c64(v), _c64(xi), _c64(vi)
    n = m.shape[0]
    if i_index is None:
        i_index = np.arange(n)
    idx = np.ascontiguousarray(i_index, dtype=np.int64)
    n_i = idx.shape[0]
    acc = np.zeros((n_i, 3))
    jrk = np.zeros((n_i, 3))
    pot = np.zeros(n_i)
    rc = lib.oracle_force(n, _p(m), _p(x), _p(v), float(eps), n_i, idx.ctypes.data_as(_I), _p(xi), _p(vi),
                          1 if want_jerk else 0, _p(acc), _p(jrk) if want_jerk else None, _p(pot))
    if rc != 0:
        raise ValueError("oracle_force: bad arguments")
    return acc, jrk, pot


def nearest_neighbour(x, i_index=None, xi=None):
    lib = _load()
    x, xi = _c64(x), _c64(xi)
    n = x.shape[0]
    if i_index is None:
        i_index = np.arange(n)
    idx = np.ascontiguousarray(i_index, dtype=np.int64)
    nn = np.empty(idx.shape[0], dtype=np.int64)
    r2 = np.empty(idx.shape[0])
    rc = lib.oracle_nearest(n, _p(x), idx.shape[0], idx.ctypes.data_as(_I), _p(xi),
                            nn.ctypes.data_as(_I), _p(r2))
    if rc != 0:
        raise ValueError("oracle_nearest: bad arguments")
    return nn, r2


def predict(t, tj, x, v, a, jerk):
    lib = _load()
    tj, x, v, a, jerk = _c64(tj), _c64(x), _c64(v), _c64(a), _c64(jerk)
    xp, vp = np.empty_like(x), np.empty_like(v)
    rc = lib.oracle_predict(tj.shape[0], float(t), _p(tj), _p(x), _p(v), _p(a), _p(jerk), _p(xp), _p(vp))
    if rc != 0:
        raise ValueError("oracle_predict: bad arguments")
    return xp, vp
