"""CPU oracle for the DWF hopping term Dhop -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports, links or
calls anything of ``paper_2203_06777_b200`` (the CUDA path), and that package
never imports this one.

The arithmetic lives in ``dhop_oracle.c`` (plain C, fp64, OpenMP over sites): the
definition of the operator written out with full 4x4 gamma matrices, see that
file's header for the passages it follows (PAPER.md L43/L223/L254 name the
operator; BASELINE.json north_star states it; SURVEY.md 8(c) fixes conventions),
and in ``dwf5d_oracle.c``: the rest of the red-black Shamir domain-wall operator
 as dense linear algebra on the (4 Ls) x (4 Ls) matrix of its
4D-site-diagonal part.  This module only marshals numpy arrays (canonical layouts
of include/dwf.h).

Pins: tests/test_oracle_pins.py (P1-P9 of SURVEY.md 8(c)) and
tests/test_oracle_pins_dwf.py (the 8(f2) functions); nothing is unpinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = [os.path.join(_HERE, "dhop_oracle.c"), os.path.join(_HERE, "dwf5d_oracle.c")]
_LIB = os.path.join(_HERE, "liboracle.so")

PERIODIC, ANTIPERIODIC_T, OPEN_T = 0, 1, 2     # OPEN_T: hops that would wrap in time contribute nothing
EVEN, ODD = 0, 1


def build(force: bool = False) -> str:
    """Compile dhop_oracle.c into liboracle.so (in-tree).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fcx-limited-range", "-fopenmp", "-fPIC", "-shared",
             "-o", tmp, *_SRCS, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, ci, i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        i4 = ctypes.POINTER(ctypes.c_int)
        lib.orc_gamma.argtypes = [ci, vp]
        lib.orc_gamma.restype = None
        lib.orc_check_gamma.restype = ci
        lib.orc_dhop.argtypes = [i4, ci, ci, vp, ci, vp, ci, vp]
        lib.orc_dhop.restype = ci
        lib.orc_dhop_cb.argtypes = [i4, ci, ci, ci, vp, ci, vp, ci, vp]
        lib.orc_dhop_cb.restype = ci
        lib.orc_dhop_dag.argtypes = lib.orc_dhop.argtypes
        lib.orc_dhop_dag.restype = ci
        lib.orc_dhop_cb_dag.argtypes = lib.orc_dhop_cb.argtypes
        lib.orc_dhop_cb_dag.restype = ci
        lib.orc_dhop_sites.argtypes = [i4, ci, ci, vp, ci, vp, ci, ci, vp, i64, vp]
        lib.orc_dhop_sites.restype = ci
        lib.orc_norm2.argtypes = [vp, ci, i64]
        lib.orc_norm2.restype = ctypes.c_double
        lib.orc_inner.argtypes = [vp, vp, ci, i64, vp]
        lib.orc_inner.restype = None
        lib.orc_num_threads.restype = ci
        dbl = ctypes.c_double
        lib.orc_mooee_matrix.argtypes = [ci, dbl, dbl, ci, vp]
        lib.orc_mooee_matrix.restype = ci
        lib.orc_mooee.argtypes = [i64, ci, dbl, dbl, ci, vp, ci, vp]
        lib.orc_mooee.restype = ci
        lib.orc_ddwf.argtypes = [i4, ci, ci, dbl, dbl, ci, vp, ci, vp, ci, vp]
        lib.orc_ddwf.restype = ci
        lib.orc_schur.argtypes = [i4, ci, ci, dbl, dbl, ci, ci, vp, ci, vp, ci, vp]
        lib.orc_schur.restype = ci
        if lib.orc_check_gamma() != 0:
            raise RuntimeError("oracle gamma matrices fail their algebra self-check")
        _lib = lib
    return _lib


def _prec(a: np.ndarray) -> int:
    if a.dtype == np.float32:
        return 4
    if a.dtype == np.float64:
        return 8
    raise TypeError("fields must be float32 or float64 arrays of reals")


def _dims(dims):
    d = (ctypes.c_int * 4)(*[int(v) for v in dims])
    return d, int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def _c(a: np.ndarray) -> np.ndarray:
    if not a.flags.c_contiguous:
        raise ValueError("arrays must be C-contiguous")
    return a


def num_threads() -> int:
    return int(_load().orc_num_threads())


def gamma(mu: int) -> np.ndarray:
    """The oracle's own gamma_mu as a complex (4,4) array (for the pins)."""
    out = np.zeros((4, 4, 2))
    _load().orc_gamma(mu, out.ctypes.data)
    return out[..., 0] + 1j * out[..., 1]


def dhop(dims, Ls: int, bc_time: int, U: np.ndarray, psi: np.ndarray, dagger: bool = False) -> np.ndarray:
    """Full Dhop (dagger: its matrix adjoint).  U (V4,4,3,3,2), psi (V4,Ls,4,3,2) -> fp64 (V4,Ls,4,3,2)."""
    d, v4 = _dims(dims)
    assert U.size == v4 * 72 and psi.size == v4 * Ls * 24
    out = np.empty((v4, Ls, 4, 3, 2), dtype=np.float64)
    fn = _load().orc_dhop_dag if dagger else _load().orc_dhop
    rc = fn(d, Ls, bc_time, _c(U).ctypes.data, _prec(U),
                          _c(psi).ctypes.data, _prec(psi), out.ctypes.data)
    if rc:
        raise ValueError("orc_dhop: bad arguments")
    return out


def dhop_cb(dims, Ls: int, bc_time: int, parity_out: int, U: np.ndarray,
            psi_half: np.ndarray, dagger: bool = False) -> np.ndarray:
    """Checkerboarded Dhop onto parity_out (ODD: DhopOE, EVEN: DhopEO).
    psi_half (V4/2,Ls,4,3,2) lives on the opposite parity -> fp64 (V4/2,Ls,4,3,2)."""
    d, v4 = _dims(dims)
    assert U.size == v4 * 72 and psi_half.size == (v4 // 2) * Ls * 24
    out = np.empty((v4 // 2, Ls, 4, 3, 2), dtype=np.float64)
    fn = _load().orc_dhop_cb_dag if dagger else _load().orc_dhop_cb
    rc = fn(d, Ls, bc_time, parity_out, _c(U).ctypes.data, _prec(U),
                             _c(psi_half).ctypes.data, _prec(psi_half), out.ctypes.data)
    if rc:
        raise ValueError("orc_dhop_cb: bad arguments (extents must be even)")
    return out


def dhop_oe(dims, Ls, bc_time, U, psi_even):
    """DhopOE: even in -> odd out (SURVEY.md 8(c) reading #6)."""
    return dhop_cb(dims, Ls, bc_time, ODD, U, psi_even)


def dhop_eo(dims, Ls, bc_time, U, psi_odd):
    """DhopEO: odd in -> even out."""
    return dhop_cb(dims, Ls, bc_time, EVEN, U, psi_odd)


def dhop_sites(dims, Ls: int, bc_time: int, U: np.ndarray, psi: np.ndarray, psi_is_half: bool,
               sites) -> np.ndarray:
    """Dhop at the listed output sites (lexicographic indices) -> fp64 (n,Ls,4,3,2)."""
    d, v4 = _dims(dims)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    assert U.size == v4 * 72
    assert psi.size == (v4 // 2 if psi_is_half else v4) * Ls * 24
    assert sites.size == 0 or (0 <= sites.min() and sites.max() < v4)
    out = np.empty((sites.size, Ls, 4, 3, 2), dtype=np.float64)
    rc = _load().orc_dhop_sites(d, Ls, bc_time, _c(U).ctypes.data, _prec(U),
                                _c(psi).ctypes.data, _prec(psi), int(bool(psi_is_half)),
                                sites.ctypes.data, sites.size, out.ctypes.data)
    if rc:
        raise ValueError("orc_dhop_sites: bad arguments")
    return out


def norm2(x: np.ndarray) -> float:
    """sum of squares of all reals of x (fp64, compensated)."""
    return float(_load().orc_norm2(_c(x).ctypes.data, _prec(x), x.size))


def inner(a: np.ndarray, b: np.ndarray) -> complex:
    """sum conj(a) * b over all complex entries (last axis = re, im)."""
    assert a.shape == b.shape and a.dtype == b.dtype and a.size % 2 == 0
    out = np.zeros(2)
    _load().orc_inner(_c(a).ctypes.data, _c(b).ctypes.data, _prec(a), a.size // 2, out.ctypes.data)
    return complex(out[0], out[1])


def reconstruct12(U: np.ndarray) -> np.ndarray:
    """SURVEY.md 8(f4), 12-real link storage: the links an SU(3)-compressed path works with.  Rows 0 and 1 of
    every U_mu(x) are kept (promoted exactly to fp64), row 2 is REPLACED by conj(row0 x row1) -- for a matrix of
    SU(3) that is its own third row (unitarity + det = 1), for the fp32-rounded links of the inputs it differs
    from the stored third row at the 1e-7 level.  Plain numpy, fp64 out, shape of U."""
    Uc = U.astype(np.float64)
    z = Uc[..., 0] + 1j * Uc[..., 1]                     # (..., 3, 3) complex, row a, column b
    r0, r1 = z[..., 0, :], z[..., 1, :]
    r2 = np.conj(np.cross(r0, r1))
    out = np.stack([r0, r1, r2], axis=-2)
    return np.ascontiguousarray(np.stack([out.real, out.imag], axis=-1))


# ---------------------------------------------------------------------------------------------
# the rest of the red-black Shamir domain-wall operator (dwf5d_oracle.c)
# ---------------------------------------------------------------------------------------------
M5_APPLY, M5_DAG, M5_INV, M5_INV_DAG = 0, 1, 2, 3


def mooee_matrix(Ls: int, M5: float, mass: float, op: int = M5_APPLY) -> np.ndarray:
    """The oracle's dense (4 Ls, 4 Ls) real matrix of Mooee (index s*4 + spin), its transpose, inverse
    or inverse transpose (for the pins)."""
    out = np.empty((4 * Ls, 4 * Ls), dtype=np.float64)
    if _load().orc_mooee_matrix(int(Ls), float(M5), float(mass), int(op), out.ctypes.data):
        raise ValueError("orc_mooee_matrix: bad arguments or singular matrix")
    return out


def mooee(Ls: int, M5: float, mass: float, psi: np.ndarray, op: int = M5_APPLY) -> np.ndarray:
    """The 4D-site-diagonal part of the Shamir DWF matrix applied to a field (nsites, Ls, 4, 3, 2):
    op = M5_APPLY (Mooee), M5_DAG (its adjoint), M5_INV (inverse), M5_INV_DAG.  fp64 out."""
    assert psi.ndim == 5 and psi.shape[1:] == (Ls, 4, 3, 2)
    out = np.empty(psi.shape, dtype=np.float64)
    if _load().orc_mooee(psi.shape[0], int(Ls), float(M5), float(mass), int(op), _c(psi).ctypes.data, _prec(psi),
                         out.ctypes.data):
        raise ValueError("orc_mooee: bad arguments")
    return out


def ddwf(dims, Ls: int, bc_time: int, M5: float, mass: float, U: np.ndarray, psi: np.ndarray,
         dagger: bool = False) -> np.ndarray:
    """Full Shamir DWF matrix M = Mooee - Dhop/2 on a full field (V4, Ls, 4, 3, 2) -> fp64."""
    d, v4 = _dims(dims)
    assert U.size == v4 * 72 and psi.size == v4 * Ls * 24
    out = np.empty((v4, Ls, 4, 3, 2), dtype=np.float64)
    if _load().orc_ddwf(d, Ls, bc_time, float(M5), float(mass), int(bool(dagger)), _c(U).ctypes.data, _prec(U),
                        _c(psi).ctypes.data, _prec(psi), out.ctypes.data):
        raise ValueError("orc_ddwf: bad arguments")
    return out


def schur(dims, Ls: int, bc_time: int, M5: float, mass: float, parity: int, U: np.ndarray,
          psi_half: np.ndarray, dagger: bool = False) -> np.ndarray:
    """Schur complement S = Mooee - M_pq Mooee^-1 M_qp on parity p (half field in, half field out)."""
    d, v4 = _dims(dims)
    assert U.size == v4 * 72 and psi_half.size == (v4 // 2) * Ls * 24
    out = np.empty((v4 // 2, Ls, 4, 3, 2), dtype=np.float64)
    if _load().orc_schur(d, Ls, bc_time, float(M5), float(mass), int(bool(dagger)), int(parity),
                         _c(U).ctypes.data, _prec(U), _c(psi_half).ctypes.data, _prec(psi_half), out.ctypes.data):
        raise ValueError("orc_schur: bad arguments")
    return out
