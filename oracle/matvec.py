"""ctypes loader for oracle/matvec_c.c (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

build() compiles the C file with gcc (-O2 -fopenmp) next to the source; matvec_rows() evaluates
u_j = sum_{i != j} A_ji x_i for selected targets (Eq. I21) without storing A.
"""
import ctypes
import os
import subprocess

import numpy as np

from .modes import n_modes
from .translation import coupling_tables

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_matvec.so")
_SRC = os.path.join(_HERE, "matvec_c.c")
_lib = None


def build(force=False):
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads():
    return int(_load().oracle_num_threads())


def matvec_rows(lmax, k, pos, x, rows=None, win_ptr=None):
    """u[rows] = (A x)[rows];  pos (N,3), x (N,L) complex, rows int array (default all).  Returns (len(rows), L)."""
    lib = _load()
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.complex128)
    N = pos.shape[0]
    L = n_modes(lmax)
    assert x.shape == (N, L)
    rows = np.arange(N, dtype=np.int32) if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    wp = np.array([0, N], dtype=np.int32) if win_ptr is None else np.ascontiguousarray(win_ptr, dtype=np.int32)
    coef, mu = coupling_tables(lmax)
    coef = np.ascontiguousarray(coef, dtype=np.complex128)
    mu = np.ascontiguousarray(mu, dtype=np.int32)
    y = np.zeros((rows.size, L), dtype=np.complex128)
    vp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    lib.oracle_matvec_rows(ctypes.c_int(lmax), ctypes.c_double(k), ctypes.c_int(N), vp(pos), vp(wp),
                           ctypes.c_int(wp.size - 1), vp(coef), vp(mu), ctypes.c_int(rows.size), vp(rows),
                           vp(x), vp(y))
    return y
