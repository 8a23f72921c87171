"""Seeded synthetic inputs for the DWF Dhop path (gauge fields and spinors).

The one module shared by the CPU oracle tests and the CUDA path.  It contains no
Dhop arithmetic: only counter-based random fills of the canonical layouts
declared in ``include/dwf.h`` (recipes: SURVEY.md section 8(c) #12-#15, DESIGN.md
"Input recipe").  Backed by ``gen.c`` (plain C + OpenMP), built on first use.

Canonical layouts (real index, C order):
  gauge   [x][mu][a][b][reim]          x = x0 + L0*(x1 + L1*(x2 + L2*x3))
  spinor  [site][s][spin][colour][reim]   site = x (full) or x>>1 (half field)
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libdwfinputs.so")

# stream ids
STREAM_GAUGE, STREAM_SPINOR, STREAM_SPINOR2, STREAM_TRANSFORM = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile gen.c into libdwfinputs.so (in-tree)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64 = ctypes.c_uint64
        lib.dwfin_gaussian.argtypes = [u64, u64, u64, u64, ctypes.c_int, ctypes.c_void_p]
        lib.dwfin_su3_random.argtypes = [u64, u64, u64, u64, ctypes.c_int, ctypes.c_void_p]
        lib.dwfin_su3_near_unit.argtypes = [u64, u64, u64, u64, ctypes.c_double, ctypes.c_int,
                                            ctypes.c_void_p]
        for f in (lib.dwfin_gaussian, lib.dwfin_su3_random, lib.dwfin_su3_near_unit):
            f.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dtype(prec: int):
    if prec == 4:
        return np.float32
    if prec == 8:
        return np.float64
    raise ValueError("prec must be 4 or 8 (bytes per real)")


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def gaussian(n: int, seed: int, stream: int, prec: int = 8, first: int = 0, out=None):
    """n reals iid N(0,1): elements first..first+n-1 of the (seed, stream) sequence."""
    if out is None:
        out = np.empty(n, dtype=_dtype(prec))
    assert out.flags.c_contiguous and out.size == n and out.dtype == _dtype(prec)
    rc = _load().dwfin_gaussian(seed, stream, first, n, prec, out.ctypes.data)
    assert rc == 0
    return out


def spinor_gaussian(nsites: int, Ls: int, seed: int, stream: int = STREAM_SPINOR, prec: int = 8):
    """Gaussian spinor field in the canonical layout, shape (nsites, Ls, 4, 3, 2)."""
    out = np.empty((nsites, Ls, 4, 3, 2), dtype=_dtype(prec))
    gaussian(out.size, seed, stream, prec, out=out.reshape(-1))
    return out


def gauge_random(dims, seed: int, stream: int = STREAM_GAUGE, prec: int = 8):
    """Random SU(3) gauge field, canonical layout, shape (V4, 4, 3, 3, 2)."""
    v4 = volume(dims)
    out = np.empty((v4, 4, 3, 3, 2), dtype=_dtype(prec))
    rc = _load().dwfin_su3_random(seed, stream, 0, v4 * 4, prec, out.ctypes.data)
    assert rc == 0
    return out


def gauge_near_unit(dims, seed: int, eps: float = 0.2, stream: int = STREAM_GAUGE, prec: int = 8):
    """Near-unit gauge field U = exp(i*eps*H) projected to SU(3), shape (V4, 4, 3, 3, 2)."""
    v4 = volume(dims)
    out = np.empty((v4, 4, 3, 3, 2), dtype=_dtype(prec))
    rc = _load().dwfin_su3_near_unit(seed, stream, 0, v4 * 4, float(eps), prec, out.ctypes.data)
    assert rc == 0
    return out


def gauge_unit(dims, prec: int = 8):
    """Unit gauge field (free field), shape (V4, 4, 3, 3, 2)."""
    out = np.zeros((volume(dims), 4, 3, 3, 2), dtype=_dtype(prec))
    for a in range(3):
        out[:, :, a, a, 0] = 1.0
    return out


def su3_random(n: int, seed: int, stream: int = STREAM_TRANSFORM, prec: int = 8):
    """n random SU(3) matrices, shape (n, 3, 3, 2) (e.g. a gauge transformation g(x))."""
    out = np.empty((n, 3, 3, 2), dtype=_dtype(prec))
    rc = _load().dwfin_su3_random(seed, stream, 0, n, prec, out.ctypes.data)
    assert rc == 0
    return out


def site_parity(dims) -> np.ndarray:
    """(V4,) array of (x0+x1+x2+x3)&1 in lexicographic site order."""
    L0, L1, L2, L3 = (int(d) for d in dims)
    x = np.arange(L0 * L1 * L2 * L3, dtype=np.int64)
    return ((x % L0) + (x // L0) % L1 + (x // (L0 * L1)) % L2 + x // (L0 * L1 * L2)) & 1


def split_parity(full: np.ndarray, dims, parity: int) -> np.ndarray:
    """Half field of `parity` (sites in increasing x) taken from a full canonical field."""
    return np.ascontiguousarray(full[site_parity(dims) == parity])
