"""ctypes access to the CPU oracle (oracle/lgf_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports neither the CUDA package
nor the input generator.  Argument marshalling only; every formula lives in the C file.

Arrays are numpy complex128, C-contiguous:
  links U [V,4,3,3];  Delta / w / g [V,3,3];  scalar field [V];  s = ix + Nx*(iy + Ny*(iz + Nz*it)).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lgf_oracle.c")
_LIB = os.path.join(_HERE, "liblgf_oracle.so")
_lib = None

_c_int4 = ctypes.c_int * 4
_vp = ctypes.c_void_p
_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (single-threaded, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.orc_momentum_tables.argtypes = [_c_int4, _vp, _dp]
        L.orc_mask.argtypes = [_c_int4, _vp]
        L.orc_measure.argtypes = [_c_int4, _vp, _vp, _dp, _dp]
        L.orc_fft1d.argtypes = [ctypes.c_int, _vp, ctypes.c_int]
        L.orc_fft4d.argtypes = [_c_int4, _vp, ctypes.c_int]
        L.orc_fourier_accelerate.argtypes = [_c_int4, _vp, _vp]
        L.orc_build_g.argtypes = [ctypes.c_int64, _vp, ctypes.c_double, _vp]
        L.orc_build_g_exp.argtypes = [ctypes.c_int64, _vp, ctypes.c_double, _vp]
        L.orc_set_exponential.argtypes = [ctypes.c_int]
        L.orc_update_links.argtypes = [_c_int4, _vp, _vp]
        L.orc_iterate.argtypes = [_c_int4, _vp, ctypes.c_double, ctypes.c_int64, _vp]
        L.orc_fix.argtypes = [_c_int4, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int64,
                              _dp, _dp, _vp, ctypes.c_int64]
        L.orc_fix.restype = ctypes.c_int64
        L.orc_plaquette.argtypes = [_c_int4, _vp]
        L.orc_plaquette.restype = ctypes.c_double
        for f in (L.orc_momentum_tables, L.orc_mask, L.orc_measure, L.orc_fft1d, L.orc_fft4d,
                  L.orc_fourier_accelerate, L.orc_build_g, L.orc_build_g_exp, L.orc_set_exponential,
                  L.orc_update_links, L.orc_iterate):
            f.restype = None
        _lib = L
    return _lib


def _dims(N):
    if isinstance(N, int):
        N = (N,) * 4
    N = tuple(int(n) for n in N)
    assert len(N) == 4
    return N, _c_int4(*N), N[0] * N[1] * N[2] * N[3]


def _c128(a, size):
    assert isinstance(a, np.ndarray) and a.dtype == np.complex128 and a.flags.c_contiguous, "need contiguous complex128"
    assert a.size == size, (a.size, size)
    return a.ctypes.data


def momentum_tables(N):
    """Per-axis tables s_mu[k] = 4 sin^2(pi k/N_mu) and p_max^2 (O0)."""
    N, cN, V = _dims(N)
    tab = np.empty(sum(N), dtype=np.float64)
    pmax2 = ctypes.c_double()
    _load().orc_momentum_tables(cN, tab.ctypes.data, ctypes.byref(pmax2))
    offs = np.cumsum((0,) + N)
    return [tab[offs[i]:offs[i + 1]].copy() for i in range(4)], pmax2.value


def mask(N):
    """M(k) = p_max^2/p^2(k), M(0) = 0, as a float64 array [V] (O0)."""
    N, cN, V = _dims(N)
    M = np.empty(V, dtype=np.float64)
    _load().orc_mask(cN, M.ctypes.data)
    return M


def measure(N, U, want_delta=True):
    """(Delta [V,3,3] or None, F, theta) of links U (O1)."""
    N, cN, V = _dims(N)
    D = np.empty((V, 3, 3), dtype=np.complex128) if want_delta else None
    F, th = ctypes.c_double(), ctypes.c_double()
    _load().orc_measure(cN, _c128(U, V * 36), D.ctypes.data if want_delta else None,
                        ctypes.byref(F), ctypes.byref(th))
    return D, F.value, th.value


def fft1d(x, sign):
    """Unnormalised 1D DFT of a copy of x; sign=-1 forward, +1 backward."""
    y = np.ascontiguousarray(x, dtype=np.complex128).copy()
    _load().orc_fft1d(y.size, y.ctypes.data, int(sign))
    return y


def fft4d(N, f, sign):
    """Unnormalised 4D DFT of a copy of the scalar field f [V] (O3 / O5 without 1/V)."""
    N, cN, V = _dims(N)
    y = np.ascontiguousarray(f, dtype=np.complex128).copy()
    _load().orc_fft4d(cN, _c128(y, V), int(sign))
    return y


def fourier_accelerate(N, Delta):
    """w = F^-1 [ p_max^2/p^2 ] F Delta, all 9 elements, normalised (O3-O5)."""
    N, cN, V = _dims(N)
    w = np.empty((V, 3, 3), dtype=np.complex128)
    _load().orc_fourier_accelerate(cN, _c128(Delta, V * 9), w.ctypes.data)
    return w


def build_g(w, alpha):
    """g(x) = reunit(1 + (alpha/2) w(x)) (O6)."""
    V = w.size // 9
    g = np.empty((V, 3, 3), dtype=np.complex128)
    _load().orc_build_g(V, _c128(w, V * 9), float(alpha), g.ctypes.data)
    return g


def build_g_exp(w, alpha):
    """g(x) = exp((alpha/2) w(x)): eq. 1.2 as written, the variant of SURVEY 8(f4)."""
    V = w.size // 9
    g = np.empty((V, 3, 3), dtype=np.complex128)
    _load().orc_build_g_exp(V, _c128(w, V * 9), float(alpha), g.ctypes.data)
    return g


def set_exponential(on):
    """iterate / fix form g by the exact exponential (True) or by first order + reunitarisation (False, default)."""
    _load().orc_set_exponential(1 if on else 0)


def update_links(N, U, g):
    """In place: U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger (O7)."""
    N, cN, V = _dims(N)
    _load().orc_update_links(cN, _c128(U, V * 36), _c128(g, V * 9))
    return U


def iterate(N, U, alpha, n):
    """Exactly n iterations in place; returns history array [n+1, 2] of (F, theta)."""
    N, cN, V = _dims(N)
    hist = np.empty((n + 1, 2), dtype=np.float64)
    _load().orc_iterate(cN, _c128(U, V * 36), float(alpha), int(n), hist.ctypes.data)
    return hist


def fix(N, U, alpha=0.08, eps=1e-15, max_iter=100000, hist_cap=4096):
    """Algorithm 1 in place.  Returns (iterations, F, theta, history[iterations+1, 2])."""
    N, cN, V = _dims(N)
    hist = np.full((hist_cap, 2), np.nan, dtype=np.float64)
    F, th = ctypes.c_double(), ctypes.c_double()
    it = _load().orc_fix(cN, _c128(U, V * 36), float(alpha), float(eps), int(max_iter),
                         ctypes.byref(F), ctypes.byref(th), hist.ctypes.data, hist_cap)
    n = min(it if it >= 0 else max_iter, hist_cap - 1)
    return it, F.value, th.value, hist[: n + 1].copy()


def plaquette(N, U):
    """Average plaquette (gauge invariant; pin P11 only)."""
    N, cN, V = _dims(N)
    return _load().orc_plaquette(cN, _c128(U, V * 36))
