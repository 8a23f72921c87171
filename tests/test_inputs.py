"""Seeded input generators (dwf_inputs): determinism, SU(3) properties, distributions.  CPU only."""
import numpy as np

import dwf_inputs as gen
from _util import cplx


def test_gaussian_deterministic_and_offset_consistent():
    a = gen.gaussian(1000, seed=7, stream=1)
    b = gen.gaussian(1000, seed=7, stream=1)
    assert np.array_equal(a, b)
    tail = gen.gaussian(400, seed=7, stream=1, first=600)
    assert np.array_equal(a[600:], tail)                      # slab fills agree with one big fill
    assert not np.array_equal(a, gen.gaussian(1000, seed=8, stream=1))
    assert not np.array_equal(a, gen.gaussian(1000, seed=7, stream=2))
    f = gen.gaussian(1000, seed=7, stream=1, prec=4)
    assert f.dtype == np.float32 and np.array_equal(f, a.astype(np.float32))   # rounded once


def test_gaussian_moments():
    x = gen.gaussian(400000, seed=3, stream=1)
    assert abs(x.mean()) < 0.01 and abs(x.var() - 1.0) < 0.01
    assert abs(np.mean(x ** 4) - 3.0) < 0.1
    assert abs(np.corrcoef(x[0::2], x[1::2])[0, 1]) < 0.01


def _check_su3(U, tol):
    M = cplx(U.astype(np.float64)).reshape(-1, 3, 3)
    eye = np.eye(3)[None]
    assert np.max(np.abs(M @ M.conj().transpose(0, 2, 1) - eye)) < tol
    assert np.max(np.abs(np.linalg.det(M) - 1.0)) < tol
    return M


def test_random_su3_links():
    dims = (4, 2, 2, 4)
    M = _check_su3(gen.gauge_random(dims, seed=1001), 1e-13)
    assert np.mean(np.abs(M - np.eye(3)[None])) > 0.3            # far from unit: a "hot" field
    _check_su3(gen.gauge_random(dims, seed=1001, prec=4), 1e-6)


def test_near_unit_links():
    dims = (4, 2, 2, 4)
    M = _check_su3(gen.gauge_near_unit(dims, seed=1004, eps=0.2), 1e-13)
    dev = np.abs(M - np.eye(3)[None]).max(axis=(1, 2))
    assert 0.02 < dev.mean() < 0.6 and dev.max() < 1.5           # close to, but not equal to, 1
    M0 = _check_su3(gen.gauge_near_unit(dims, seed=1004, eps=0.0), 1e-14)
    assert np.max(np.abs(M0 - np.eye(3)[None])) < 1e-14


def test_spinor_shapes_and_parity_split():
    dims, Ls = (4, 2, 2, 2), 3
    V = gen.volume(dims)
    psi = gen.spinor_gaussian(V, Ls, seed=5)
    assert psi.shape == (V, Ls, 4, 3, 2)
    par = gen.site_parity(dims)
    assert par.sum() == V // 2 and par[0] == 0 and par[1] == 1 and par[dims[0]] == 1
    e = gen.split_parity(psi, dims, 0)
    o = gen.split_parity(psi, dims, 1)
    assert e.shape == (V // 2, Ls, 4, 3, 2) and o.shape == e.shape
    x = np.arange(V)
    assert np.array_equal(e[x[par == 0] >> 1], psi[par == 0])
