"""ctypes wrapper of the CPU oracle (oracle/wdref.c).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import this package.  It shares no code with ``paper_2407_00041_b200`` and does
not import it.  See oracle/wdref.c for what each function follows in the paper.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwdref.so")
_SRCS = [os.path.join(_HERE, "wdref.c"), os.path.join(_HERE, "wdref.h")]
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (in-tree).  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(map(os.path.getmtime, _SRCS)):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRCS[0], "-lm"]
        )
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        i, d, p = ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        lib.wdref_apply.argtypes = [i, i, i, i, d, p, p, p, p, i]
        lib.wdref_build_clover.argtypes = [i, i, i, i, d, d, p, p]
        lib.wdref_build_clover_full.argtypes = [i, i, i, i, d, d, p, p]
        lib.wdref_dense.argtypes = [i, i, i, i, d, d, p, p]
        lib.wdref_gamma.argtypes = [i, p]
        lib.wdref_gamma.restype = None
        lib.wdref_set_num_threads.argtypes = [i]
        lib.wdref_set_num_threads.restype = None
        _lib = lib
    return _lib


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def apply(dims, m0, U, C, psi) -> np.ndarray:
    """out = D psi.  psi: [nrhs][V][12][2] (or [V][12][2]); C may be None (pure Wilson)."""
    T, Z, Y, X = dims
    V = T * Z * Y * X
    psi = _f64(psi)
    squeeze = psi.ndim == 3
    psi4 = psi.reshape(-1, V, 12, 2)
    U = _f64(U)
    assert U.size == V * 72, U.shape
    out = np.empty_like(psi4)
    cptr = None
    if C is not None:
        C = _f64(C)
        assert C.size == V * 84, C.shape
        cptr = C.ctypes.data
    rc = _load().wdref_apply(T, Z, Y, X, float(m0), U.ctypes.data, cptr, out.ctypes.data,
                             psi4.ctypes.data, psi4.shape[0])
    if rc != 0:
        raise RuntimeError(f"wdref_apply failed: {rc}")
    return out[0] if squeeze else out


def build_clover(dims, m0, csw, U) -> np.ndarray:
    T, Z, Y, X = dims
    V = T * Z * Y * X
    U = _f64(U)
    C = np.empty((V, 42, 2), dtype=np.float64)
    rc = _load().wdref_build_clover(T, Z, Y, X, float(m0), float(csw), U.ctypes.data, C.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"wdref_build_clover failed: {rc}")
    return C


def build_clover_full(dims, m0, csw, U) -> np.ndarray:
    """[V][12][12] complex128."""
    T, Z, Y, X = dims
    V = T * Z * Y * X
    U = _f64(U)
    S = np.empty((V, 12, 12, 2), dtype=np.float64)
    rc = _load().wdref_build_clover_full(T, Z, Y, X, float(m0), float(csw), U.ctypes.data, S.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"wdref_build_clover_full failed: {rc}")
    return S.view(np.complex128)[..., 0]


def dense(dims, m0, csw, U) -> np.ndarray:
    """[12V][12V] complex128."""
    T, Z, Y, X = dims
    N = 12 * T * Z * Y * X
    U = _f64(U)
    M = np.empty((N, N, 2), dtype=np.float64)
    rc = _load().wdref_dense(T, Z, Y, X, float(m0), float(csw), U.ctypes.data, M.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"wdref_dense failed: {rc}")
    return M.view(np.complex128)[..., 0]


def gamma(mu: int) -> np.ndarray:
    g = np.empty((4, 4, 2), dtype=np.float64)
    _load().wdref_gamma(mu, g.ctypes.data)
    return g.view(np.complex128)[..., 0]


def num_threads() -> int:
    return int(_load().wdref_num_threads())


def set_num_threads(n: int) -> None:
    _load().wdref_set_num_threads(int(n))
