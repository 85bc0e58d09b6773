"""Seeded synthetic SU(3) gauge fields: the input generator shared by the oracle tests and
the CUDA path.  It holds none of the gauge-fixing arithmetic (see gen_links.c header) and
imports neither ``oracle`` nor ``paper_1210_8018_b200``.

Recipe: BASELINE.json ``configs`` / DESIGN.md "Input recipe".  Stands in for the paper's
Wilson-action configurations, which are not available.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen_links.c")
_LIB = os.path.join(_HERE, "libgen_links.so")
_lib = None

#: seeds of the BASELINE.json configs: 12108018 + N for the N^4 lattice
BASE_SEED = 12108018


def build(force: bool = False) -> str:
    """Compile gen_links.c with gcc (OpenMP) into gen/libgen_links.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.gen_links.argtypes = [
            ctypes.POINTER(ctypes.c_int), ctypes.c_double, ctypes.c_uint64, ctypes.c_int,
            ctypes.c_void_p,
        ]
        lib.gen_links.restype = None
        lib.gen_haar_field.argtypes = [ctypes.POINTER(ctypes.c_int), ctypes.c_uint64, ctypes.c_void_p]
        lib.gen_haar_field.restype = None
        _lib = lib
    return _lib


def _dims(N):
    if isinstance(N, int):
        N = (N, N, N, N)
    N = tuple(int(n) for n in N)
    assert len(N) == 4
    return N


def gen_links(N, sigma: float, seed: int, haar: bool = True, out=None) -> np.ndarray:
    """Links in the interchange layout: complex128 array [V, 4, 3, 3], site index
    s = ix + Nx*(iy + Ny*(iz + Nz*it)) (x fastest), direction mu = 0..3 <-> x, y, z, t."""
    N = _dims(N)
    V = N[0] * N[1] * N[2] * N[3]
    if out is None:
        out = np.empty((V, 4, 3, 3), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous and out.size == V * 36
    cN = (ctypes.c_int * 4)(*N)
    _load().gen_links(cN, float(sigma), int(seed), int(bool(haar)), out.ctypes.data)
    return out


def gen_haar_field(N, seed: int) -> np.ndarray:
    """Haar-random SU(3) matrix per site, complex128 [V, 3, 3] (the g0 used by gen_links)."""
    N = _dims(N)
    V = N[0] * N[1] * N[2] * N[3]
    out = np.empty((V, 3, 3), dtype=np.complex128)
    cN = (ctypes.c_int * 4)(*N)
    _load().gen_haar_field(cN, int(seed), out.ctypes.data)
    return out


#: the five BASELINE.json configs: name -> (extents, sigma, seed)
CONFIGS = {
    "8^4": ((8, 8, 8, 8), 0.3, BASE_SEED + 8),
    "16^4": ((16, 16, 16, 16), 0.5, BASE_SEED + 16),
    "32^4": ((32, 32, 32, 32), 0.5, BASE_SEED + 32),
    "48^4": ((48, 48, 48, 48), 0.5, BASE_SEED + 48),
    "64^4": ((64, 64, 64, 64), 0.6, BASE_SEED + 64),
}


def gen_config(name: str) -> np.ndarray:
    N, sigma, seed = CONFIGS[name]
    return gen_links(N, sigma, seed)
