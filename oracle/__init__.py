"""ctypes front end of the CPU oracle (oracle/bem_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, bench.py's cpu_baseline /
--impl reference legs and __graft_entry__.smoke() may import this package; the
CUDA library (paper_1905_01341_b200/) never does and shares no code with it.

The arithmetic is all in bem_oracle.c (plain C, fp64, direct O(N * 3T) sums of
the discretised operator y = S[q] - D[phi] of PAPER.md:127-146, Eqs. 11-13);
this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bem_oracle.c")
_LIB = os.path.join(_HERE, "libbem_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile bem_oracle.c with gcc (-O2 -fopenmp).  Building the checker is
    not using it (graft build() calls this)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else ctypes.c_void_p(0)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def g3_apply(V, F, q, phi, eta=2.5, rows=None, return_near=False):
    """y[r] = (S q - D phi)(rows[r]) in mode G3 (3-pt Gauss + exact near
    correction).  q or phi may be None (zero density)."""
    lib = _load()
    V = _f64(V); F = np.ascontiguousarray(F, dtype=np.int32)
    q = _f64(q); phi = _f64(phi)
    N, T = V.shape[0], F.shape[0]
    rows = np.arange(N, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    y = np.zeros(rows.shape[0])
    near = np.zeros(rows.shape[0], dtype=np.int64)
    rc = lib.oracle_g3_apply_rows(_p(V), ctypes.c_int64(N), _p(F), ctypes.c_int64(T), _p(q), _p(phi),
                                  ctypes.c_double(eta), _p(rows), ctypes.c_int64(rows.shape[0]),
                                  _p(y), _p(near))
    assert rc == 0
    return (y, near) if return_near else y


def g3_dense(V, F, eta=2.5, rows=None):
    """Dense rows of S and D (tiny meshes only)."""
    lib = _load()
    V = _f64(V); F = np.ascontiguousarray(F, dtype=np.int32)
    N, T = V.shape[0], F.shape[0]
    rows = np.arange(N, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    S = np.zeros((rows.shape[0], N)); D = np.zeros((rows.shape[0], N))
    rc = lib.oracle_g3_dense_rows(_p(V), ctypes.c_int64(N), _p(F), ctypes.c_int64(T),
                                  ctypes.c_double(eta), _p(rows), ctypes.c_int64(rows.shape[0]),
                                  _p(S), _p(D))
    assert rc == 0
    return S, D


def v1_vertex_weights(V, F):
    lib = _load()
    V = _f64(V); F = np.ascontiguousarray(F, dtype=np.int32)
    N, T = V.shape[0], F.shape[0]
    s = np.zeros(N); n = np.zeros((N, 3))
    lib.oracle_v1_vertex_weights(_p(V), ctypes.c_int64(N), _p(F), ctypes.c_int64(T), _p(s), _p(n))
    return s, n


def v1_apply(V, F, q, phi, rows=None, return_diag=False):
    """Mode V1: the paper's Eq. 17 with the diagonal of Eqs. 19-21."""
    lib = _load()
    V = _f64(V); F = np.ascontiguousarray(F, dtype=np.int32)
    q = _f64(q); phi = _f64(phi)
    N, T = V.shape[0], F.shape[0]
    rows = np.arange(N, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    y = np.zeros(rows.shape[0]); Ld = np.zeros(rows.shape[0]); Md = np.zeros(rows.shape[0])
    rc = lib.oracle_v1_apply_rows(_p(V), ctypes.c_int64(N), _p(F), ctypes.c_int64(T), _p(q), _p(phi),
                                  _p(rows), ctypes.c_int64(rows.shape[0]), _p(y), _p(Ld), _p(Md))
    assert rc == 0
    return (y, Ld, Md) if return_diag else y


def exact_weights(tri, x, incident_local=-1):
    """Exact int_T lambda_a G and int_T lambda_a dG/dn of one flat triangle seen from x."""
    lib = _load()
    tri = _f64(tri).reshape(9); x = _f64(x).reshape(3)
    WS = np.zeros(3); WD = np.zeros(3)
    lib.oracle_exact_weights(_p(tri), _p(x), ctypes.c_int(incident_local), _p(WS), _p(WD))
    return WS, WD


def gauss3_coeffs(tri, x):
    lib = _load()
    tri = _f64(tri).reshape(9); x = _f64(x).reshape(3)
    cS = np.zeros(3); cD = np.zeros(3)
    lib.oracle_gauss3_coeffs(_p(tri), _p(x), _p(cS), _p(cD))
    return cS, cD


def monopole_sum(src, m, tgt):
    """y[r] = sum_j m_j / (4 pi |tgt_r - src_j|), coincident points skipped
    (the workload of the paper's Table 1)."""
    lib = _load()
    src = _f64(src); m = _f64(m); tgt = _f64(tgt)
    y = np.zeros(tgt.shape[0])
    lib.oracle_monopole_sum(_p(src), _p(m), ctypes.c_int64(src.shape[0]), _p(tgt),
                            ctypes.c_int64(tgt.shape[0]), _p(y))
    return y


def point_sum(src, m, d, tgt):
    """y[r] = sum_j [ m_j / (4 pi |x_r - y_j|) - d_j.(x_r - y_j) / (4 pi |x_r - y_j|^3) ], coincident points skipped
    (Eq. 13); m [ns] or d [ns, 3] may be None."""
    lib = _load()
    src = _f64(src); tgt = _f64(tgt)
    m = None if m is None else _f64(m)
    d = None if d is None else _f64(d)
    y = np.zeros(tgt.shape[0])
    lib.oracle_point_sum(_p(src), _p(m), _p(d), ctypes.c_int64(src.shape[0]), _p(tgt), ctypes.c_int64(tgt.shape[0]), _p(y))
    return y


def g3_evaluate(V, F, q, phi, X, eta=2.5, return_near=False):
    """u(x) = S[q](x) - D[phi](x) at points x OFF the surface (Eq. 11), mode G3."""
    lib = _load()
    V = _f64(V); F = np.ascontiguousarray(F, dtype=np.int32); X = _f64(X)
    q = None if q is None else _f64(q)
    phi = None if phi is None else _f64(phi)
    y = np.zeros(X.shape[0]); near = np.zeros(X.shape[0], dtype=np.int64)
    rc = lib.oracle_g3_evaluate(_p(V), ctypes.c_int64(V.shape[0]), _p(F), ctypes.c_int64(F.shape[0]), _p(q), _p(phi),
                                ctypes.c_double(eta), _p(X), ctypes.c_int64(X.shape[0]), _p(y), _p(near))
    assert rc == 0
    return (y, near) if return_near else y
