"""Seeded synthetic SU(3) gauge-field generators -- the one module oracle tests and CUDA tests share.

Holds no gauge-fixing arithmetic (see gfi_gen.c header).  Fields come back as numpy complex128 arrays in the
canonical layout ``U[s, mu, row, col]`` with ``s = x + Nx*(y + Ny*(z + Nz*t))``, which
both ``oracle`` and ``paper_1209_4008_b200`` take (the latter through ``gf_pack``).

Recipes follow BASELINE.json ``configs`` / SURVEY.md sec. 8(d); they stand in for the paper's Monte-Carlo
configurations, which are not available.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gfi_gen.c")
_LIB = os.path.join(_HERE, "libgfi.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gfi_gen.c -> libgfi.so with gcc (host code only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.gfi_generate.argtypes = [
            ctypes.POINTER(ctypes.c_int), ctypes.c_int, ctypes.c_double, ctypes.c_uint64, ctypes.c_void_p,
        ]
        lib.gfi_generate.restype = ctypes.c_int
        lib.gfi_haar_su3.argtypes = [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p]
        lib.gfi_haar_su3.restype = None
        lib.gfi_philox4x32_10.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.gfi_philox4x32_10.restype = None
        _lib = lib
    return _lib


KIND_TRIVIAL_ORBIT, KIND_SMOOTH, KIND_HOT, KIND_SMOOTH_NOGAUGE = 0, 1, 2, 3


def _generate(dims, kind: int, eps: float, seed: int) -> np.ndarray:
    dims = tuple(int(d) for d in dims)
    assert len(dims) == 4 and all(d >= 1 for d in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    assert V < 2**32
    U = np.empty((V, 4, 3, 3), dtype=np.complex128)
    N = (ctypes.c_int * 4)(*dims)
    rc = _load().gfi_generate(N, kind, float(eps), int(seed), U.ctypes.data)
    if rc != 0:
        raise ValueError(f"gfi_generate failed rc={rc}")
    return U


def trivial_orbit(dims, seed: int) -> np.ndarray:
    """U_mu(x) = g(x) g(x+mu)^dagger with Haar-random g(x) (BASELINE.json configs[0])."""
    return _generate(dims, KIND_TRIVIAL_ORBIT, 0.0, seed)


def smooth_random(dims, eps: float, seed: int) -> np.ndarray:
    """U_mu(x) = g(x) exp(i eps H_mu(x)) g(x+mu)^dagger (BASELINE.json configs[1..4])."""
    return _generate(dims, KIND_SMOOTH, eps, seed)


def smooth_nogauge(dims, eps: float, seed: int) -> np.ndarray:
    """U_mu(x) = exp(i eps H_mu(x)): same links as smooth_random before the random gauge transformation."""
    return _generate(dims, KIND_SMOOTH_NOGAUGE, eps, seed)


def hot(dims, seed: int) -> np.ndarray:
    """Every link an independent Haar SU(3) matrix (disordered field; oracle pins)."""
    return _generate(dims, KIND_HOT, 0.0, seed)


def haar_su3(seed: int, s: int, f: int = 4) -> np.ndarray:
    g = np.empty((3, 3), dtype=np.complex128)
    _load().gfi_haar_su3(int(seed), int(s), int(f), g.ctypes.data)
    return g


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    _load().gfi_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out
