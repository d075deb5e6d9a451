"""ctypes wrapper around oracle/gene_nl_oracle.c (plain C, FP64, OpenMP over planes).

TEST INFRASTRUCTURE ONLY -- see the header of gene_nl_oracle.c.  Array convention on the Python
side: a plane is a complex128 numpy array of shape (nky0, nx0) (kx fastest, BASELINE.json
configs[0]); a stack of planes has shape (P, nky0, nx0).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

DFT_NAIVE = 0       # O(N^2) definition of the 1-D DFT
DFT_RECURSIVE = 1   # plain recursive radix-2/3 decimation

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gene_nl_oracle.c")
_LIB = os.path.join(_HERE, "libgene_nl_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA involved).  Returns the path of the shared object."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            dp = ctypes.POINTER(ctypes.c_double)
            lib.oracle_dft.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp]
            lib.oracle_dft.restype = None
            lib.oracle_nl_pseudospectral.argtypes = [
                ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                ctypes.c_long, dp, ctypes.POINTER(ctypes.c_long), dp, dp, ctypes.c_double]
            lib.oracle_nl_pseudospectral.restype = None
            lib.oracle_nl_convolution_plane.argtypes = [
                ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, dp, dp, dp]
            lib.oracle_nl_convolution_plane.restype = None
            ip = ctypes.POINTER(ctypes.c_int)
            lib.oracle_nl_convolution_modes.argtypes = [
                ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, dp, dp,
                ctypes.c_int, ip, ip, dp]
            lib.oracle_nl_convolution_modes.restype = None
            lib.oracle_nlx_convolution_plane.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp, dp, dp, dp]
            lib.oracle_nlx_convolution_plane.restype = None
            lib.oracle_nlx_pseudospectral.argtypes = [
                ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_long, dp, dp, dp, dp, dp, dp, ctypes.c_double]
            lib.oracle_nlx_pseudospectral.restype = None
            _lib = lib
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def num_threads() -> int:
    """Threads the OpenMP loops of the oracle will use (OMP_NUM_THREADS or all host cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        try:
            return max(1, int(env.split(",")[0]))
        except ValueError:
            pass
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def dft(x, sign: int, backend: int = DFT_NAIVE) -> np.ndarray:
    """Unnormalised 1-D DFT, out[k] = sum_n x[n] exp(sign*2*pi*i*n*k/N)."""
    x = _c128(x)
    out = np.empty_like(x)
    _load().oracle_dft(int(backend), int(x.size), int(sign), _dptr(x), _dptr(out))
    return out


def nl_pseudospectral(chi, g, rhs, scale: float, kxmin: float, kymin: float,
                      chi_index=None, backend: int = DFT_RECURSIVE) -> np.ndarray:
    """rhs + scale*N(chi, g) for a stack of planes, by the algorithm of PAPER.md:61.

    g, rhs: (P, nky0, nx0); chi: (Q, nky0, nx0); chi_index[p] in [0, Q) is the chi plane that g
    plane p uses (default: identity, Q == P).  Returns a new array; inputs are not modified.
    """
    g = _c128(g)
    chi = _c128(chi)
    out = _c128(rhs).copy()
    if g.ndim == 2:
        g, chi, out = g[None], chi[None], out[None]
    P, nky0, nx0 = g.shape
    assert out.shape == g.shape and chi.shape[1:] == g.shape[1:]
    if chi_index is None:
        assert chi.shape[0] == P
        chi_index = np.arange(P)
    ci = np.ascontiguousarray(chi_index, dtype=np.int64)
    assert ci.shape == (P,) and ci.min(initial=0) >= 0 and ci.max(initial=0) < chi.shape[0]
    _load().oracle_nl_pseudospectral(
        int(backend), nx0, nky0, float(kxmin), float(kymin), P, _dptr(chi),
        ci.ctypes.data_as(ctypes.POINTER(ctypes.c_long)), _dptr(g), _dptr(out), float(scale))
    return out


def nl_convolution_plane(chi, g, kxmin: float, kymin: float) -> np.ndarray:
    """N(chi, g) of ONE plane by the definition (direct truncated spectral convolution)."""
    g = _c128(g)
    chi = _c128(chi)
    nky0, nx0 = g.shape
    out = np.zeros_like(g)
    _load().oracle_nl_convolution_plane(nx0, nky0, float(kxmin), float(kymin),
                                        _dptr(chi), _dptr(g), _dptr(out))
    return out


def nl_convolution_modes(chi, g, kxmin: float, kymin: float, i_idx, j_idx) -> np.ndarray:
    """N(chi, g) of ONE plane at the stored indices (i_idx[t], j_idx[t]) only, by the definition."""
    g = _c128(g)
    chi = _c128(chi)
    nky0, nx0 = g.shape
    ii = np.ascontiguousarray(i_idx, dtype=np.int32)
    jj = np.ascontiguousarray(j_idx, dtype=np.int32)
    out = np.zeros(ii.size, dtype=np.complex128)
    ip = ctypes.POINTER(ctypes.c_int)
    _load().oracle_nl_convolution_modes(nx0, nky0, float(kxmin), float(kymin), _dptr(chi), _dptr(g),
                                        int(ii.size), ii.ctypes.data_as(ip), jj.ctypes.data_as(ip),
                                        _dptr(out))
    return out


# ---- x-global variant: planes of shape (nky0, nx), x fastest ----
def nlx_convolution_plane(vex, vey, dxg, dyg) -> np.ndarray:
    """N^(x, ky) = sum over ky' of [vex dxg + vey dyg] for ONE plane, by the definition (truncated convolution)."""
    vex, vey, dxg, dyg = (_c128(a) for a in (vex, vey, dxg, dyg))
    nky0, nx = vex.shape
    out = np.zeros_like(vex)
    _load().oracle_nlx_convolution_plane(nx, nky0, _dptr(vex), _dptr(vey), _dptr(dxg), _dptr(dyg), _dptr(out))
    return out


def nlx_pseudospectral(vex, vey, dxg, dyg, pref, rhs, scale: float, backend: int = DFT_RECURSIVE) -> np.ndarray:
    """rhs + scale*pref[x]*N^ for a stack of planes (P, nky0, nx), by the algorithm of PAPER.md:61."""
    vex, vey, dxg, dyg = (_c128(a) for a in (vex, vey, dxg, dyg))
    out = _c128(rhs).copy()
    single = vex.ndim == 2
    if single:
        vex, vey, dxg, dyg, out = vex[None], vey[None], dxg[None], dyg[None], out[None]
    P, nky0, nx = vex.shape
    assert all(a.shape == vex.shape for a in (vey, dxg, dyg, out))
    pref = np.ascontiguousarray(pref, dtype=np.float64)
    assert pref.shape == (nx,)
    _load().oracle_nlx_pseudospectral(int(backend), nx, nky0, P, _dptr(vex), _dptr(vey), _dptr(dxg), _dptr(dyg),
                                      _dptr(pref), _dptr(out), float(scale))
    return out[0] if single else out
