"""ctypes binding of libwdbench.so (include/wd_bench.h): measurement helpers for bench.py's roofline
denominators — a register-only FP64 FMA microbenchmark and streaming ceilings of the device memory.
Not part of the product path: libwd.so exports none of this.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwdbench.so")
_i, _d, _sz = ctypes.c_int, ctypes.c_double, ctypes.c_size_t
SIGNATURES = {
    "wdb_measure_fp64": (_i, [_i, _i, _i, _i, ctypes.POINTER(_d), ctypes.POINTER(_d)]),
    "wdb_measure_stream": (_i, [_i, _sz, _i, ctypes.POINTER(_d)]),
    "wdb_measure_lds": (_i, [_i, ctypes.POINTER(_d)]),
}
_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2407_00041_b200.build`")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def wdb_measure_fp64(threads_per_sm: int, ilp: int, one_cta_per_sm: bool = False,
                     distinct_operands: bool = False) -> tuple[float, float]:
    tf, cyc = _d(0.0), _d(0.0)
    rc = lib().wdb_measure_fp64(threads_per_sm, ilp, 1 if one_cta_per_sm else 0, 1 if distinct_operands else 0,
                                ctypes.byref(tf), ctypes.byref(cyc))
    if rc != 0:
        raise RuntimeError(f"wdb_measure_fp64 failed: {rc}")
    return tf.value, cyc.value


def wdb_measure_stream(mode: int, nbytes: int, reps: int = 5) -> float:
    """GB/s of a grid-stride streaming kernel: mode 0 read only, 1 copy, 2 seven reads per write."""
    g = _d(0.0)
    rc = lib().wdb_measure_stream(mode, nbytes, reps, ctypes.byref(g))
    if rc != 0:
        raise RuntimeError(f"wdb_measure_stream failed: {rc}")
    return g.value


LDS_PATTERNS = ["512 distinct bytes", "lane & 7 (same 128 B in each quarter-warp)", "lane >> 2 (one address per 4 adjacent lanes)",
                "one address", "4 aligned segments by lane & 3", "4 aligned segments by lane >> 3", "lane >> 1 (pairs)"]


def wdb_measure_lds(pattern: int) -> float:
    """SM cycles per warp-level LDS.128 for a lane-to-address pattern (index into LDS_PATTERNS)."""
    c = _d(0.0)
    rc = lib().wdb_measure_lds(pattern, ctypes.byref(c))
    if rc != 0:
        raise RuntimeError(f"wdb_measure_lds failed: {rc}")
    return c.value
