"""Seeded synthetic input fields shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NONE of the method's arithmetic (no gamma matrices, no operator, no clover
construction) — only counter-based random numbers shaped into the input distributions listed in
DESIGN.md ("Input recipe").  It imports neither ``oracle`` nor ``paper_2407_00041_b200``.

Layouts (canonical host layouts of include/wd.h):
  spinor  float64 [nrhs][V][12][2]      site-major, component 3*spin+colour, (re, im)
  gauge   float64 [V][4][3][3][2]       mu = T,Z,Y,X forward links of the own site, row-major 3x3
  selfcpl float64 [V][42][2]            the 42 entries of D_sc (R6)
with site index i = ((t*Z + z)*Y + y)*X + x.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwdinputs.so")
_SRC = os.path.join(_HERE, "gen.c")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c into libwdinputs.so with gcc (in-tree)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp, u64, f64 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_double
        lib.wdin_gaussian.argtypes = [dp, u64, u64]
        lib.wdin_su3_haar.argtypes = [dp, u64, u64]
        lib.wdin_su3_exp.argtypes = [dp, u64, u64, f64]
        lib.wdin_su3_unit.argtypes = [dp, u64]
        lib.wdin_selfcoupling_random.argtypes = [dp, u64, u64, f64, f64]
        lib.wdin_gaussian_sites.argtypes = [dp, dp, u64, u64, u64]
        lib.wdin_su3_haar_sites.argtypes = [dp, dp, u64, u64]
        lib.wdin_su3_exp_sites.argtypes = [dp, dp, u64, u64, f64]
        for f in (lib.wdin_gaussian, lib.wdin_su3_haar, lib.wdin_su3_exp, lib.wdin_su3_unit,
                  lib.wdin_selfcoupling_random, lib.wdin_gaussian_sites, lib.wdin_su3_haar_sites, lib.wdin_su3_exp_sites):
            f.restype = None
        _lib = lib
    return _lib


def volume(dims) -> int:
    T, Z, Y, X = dims
    return T * Z * Y * X


def gaussian(n: int, seed: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().wdin_gaussian(out.ctypes.data, n, seed)
    return out


def spinor(dims, seed: int, nrhs: int = 1) -> np.ndarray:
    """[nrhs][V][12][2]; RHS r is the independent stream seed + r (BASELINE.json cfg 5)."""
    V = volume(dims)
    out = np.empty((nrhs, V, 12, 2), dtype=np.float64)
    for r in range(nrhs):
        _load().wdin_gaussian(out[r].ctypes.data, V * 24, seed + r)
    return out


def spinor_sites(seed: int, sites, nrhs: int = 1) -> np.ndarray:
    """The rows spinor(dims, seed, nrhs)[:, sites] without generating the rest: [nrhs][len(sites)][12][2].  `sites`: global
    canonical site indices (int64), e.g. Decomposition.global_sites(rank)."""
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((nrhs, len(sites), 12, 2), dtype=np.float64)
    for r in range(nrhs):
        _load().wdin_gaussian_sites(out[r].ctypes.data, sites.ctypes.data, len(sites), 24, seed + r)
    return out


def config_gauge_sites(cfg: dict, sites) -> np.ndarray:
    """The rows config_gauge(cfg)[sites] without generating the rest: [len(sites)][4][3][3][2]."""
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    U = np.empty((len(sites), 4, 3, 3, 2), dtype=np.float64)
    g = cfg["gauge"]
    if g[0] == "haar":
        _load().wdin_su3_haar_sites(U.ctypes.data, sites.ctypes.data, len(sites), g[1])
    elif g[0] == "exp":
        _load().wdin_su3_exp_sites(U.ctypes.data, sites.ctypes.data, len(sites), g[1], g[2])
    else:
        raise ValueError(g)
    return U


def gauge_haar(dims, seed: int) -> np.ndarray:
    V = volume(dims)
    U = np.empty((V, 4, 3, 3, 2), dtype=np.float64)
    _load().wdin_su3_haar(U.ctypes.data, V * 4, seed)
    return U


def gauge_exp(dims, seed: int, eps: float) -> np.ndarray:
    V = volume(dims)
    U = np.empty((V, 4, 3, 3, 2), dtype=np.float64)
    _load().wdin_su3_exp(U.ctypes.data, V * 4, seed, eps)
    return U


def gauge_unit(dims) -> np.ndarray:
    V = volume(dims)
    U = np.empty((V, 4, 3, 3, 2), dtype=np.float64)
    _load().wdin_su3_unit(U.ctypes.data, V * 4)
    return U


def su3_field(dims, seed: int) -> np.ndarray:
    """One Haar SU(3) matrix per site, [V][3][3][2] (e.g. a random gauge transformation)."""
    V = volume(dims)
    g = np.empty((V, 3, 3, 2), dtype=np.float64)
    _load().wdin_su3_haar(g.ctypes.data, V, seed)
    return g


def selfcoupling_random(dims, seed: int, shift: float = 3.6, scale: float = 0.2) -> np.ndarray:
    V = volume(dims)
    C = np.empty((V, 42, 2), dtype=np.float64)
    _load().wdin_selfcoupling_random(C.ctypes.data, V, seed, shift, scale)
    return C


# The five workloads of BASELINE.json "configs"; seeds as proposed there.
CONFIGS = {
    1: dict(name="cfg1_4^4_wilson", dims=(4, 4, 4, 4), m0=-0.5, csw=0.0, nrhs=1,
            gauge=("haar", 1001), spinor_seed=2001),
    2: dict(name="cfg2_8^4_clover", dims=(8, 8, 8, 8), m0=-0.4, csw=1.0, nrhs=1,
            gauge=("exp", 1002, 0.3), spinor_seed=2002),
    3: dict(name="cfg3_32^4_clover", dims=(32, 32, 32, 32), m0=-0.4, csw=1.0, nrhs=1,
            gauge=("exp", 1003, 0.5), spinor_seed=2003),
    4: dict(name="cfg4_64^4_clover", dims=(64, 64, 64, 64), m0=-0.4, csw=1.0, nrhs=1,
            gauge=("haar", 1004), spinor_seed=2004),
    5: dict(name="cfg5_48^3x96_clover_12rhs", dims=(96, 48, 48, 48), m0=-0.4, csw=1.0, nrhs=12,
            gauge=("haar", 1005), spinor_seed=2005),
}


def config_gauge(cfg: dict, dims=None) -> np.ndarray:
    dims = dims or cfg["dims"]
    g = cfg["gauge"]
    if g[0] == "haar":
        return gauge_haar(dims, g[1])
    if g[0] == "exp":
        return gauge_exp(dims, g[1], g[2])
    raise ValueError(g)
