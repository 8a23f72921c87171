"""Pins for the oracle of SURVEY.md 8(f2): the rest of the red-black Shamir domain-wall operator
(oracle/dwf5d_oracle.c).  CPU only.

The paper prints no formula for these kernels (PAPER.md L223, L250, L254 only name "all kernels
involved in the DWF Dirac operator"); reading #22 states the definition:

    (M psi)(x,s) = (5 - M5) psi(x,s) - 1/2 Dhop psi(x,s) - P_- psi(x,s+1) - P_+ psi(x,s-1),
    psi(x,Ls) = -m psi(x,0),  psi(x,-1) = -m psi(x,Ls-1),  P_+- = (1 +- gamma5)/2.

Every oracle function is checked against something other than itself: a dense matrix over
(spin, s, site, colour) assembled with numpy Kronecker products from Pauli-matrix gammas (tests/_util.py),
numpy.linalg on that matrix (inverse, Schur complement), closed forms (Ls = 1, periodic /
antiperiodic fifth dimension) and the gamma5 R5 hermiticity of the operator.
"""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import GAMMA5, cplx, dense_dhop_matrix, reals, rel_err

M5, MASS = 1.8, 0.07


def dense_s_matrices(Ls, mass):
    """(Ls, Ls) shift matrices with the wall mass: (Sp psi)(s) = psi(s+1), psi(Ls) = -m psi(0);
    (Sm psi)(s) = psi(s-1), psi(-1) = -m psi(Ls-1)."""
    Sp, Sm = np.zeros((Ls, Ls)), np.zeros((Ls, Ls))
    for s in range(Ls):
        if s + 1 < Ls:
            Sp[s, s + 1] += 1.0
        else:
            Sp[s, 0] += -mass
        if s - 1 >= 0:
            Sm[s, s - 1] += 1.0
        else:
            Sm[s, Ls - 1] += -mass
    return Sp, Sm


def dense_mooee(Ls, m5, mass):
    """Mooee on one 4D site and colour, index (s, spin): a second statement of the definition."""
    Pp, Pm = 0.5 * (np.eye(4) + GAMMA5.real), 0.5 * (np.eye(4) - GAMMA5.real)
    Sp, Sm = dense_s_matrices(Ls, mass)
    return (5.0 - m5) * np.eye(4 * Ls) - np.kron(Sp, Pm) - np.kron(Sm, Pp)


def dense_dwf_matrix(dims, Ls, U, bc, m5, mass):
    """Full M over index (s, spin, site, colour): Mooee (x) 1 - 1/2 1_s (x) Dhop."""
    V = int(np.prod(dims))
    D = dense_dhop_matrix(dims, U, bc == oracle.ANTIPERIODIC_T)           # index (spin, site, colour)
    A = dense_mooee(Ls, m5, mass)                                          # index (s, spin)
    return np.kron(A, np.eye(3 * V)) - 0.5 * np.kron(np.eye(Ls), D)


def to_vec(psi):
    """canonical (V, Ls, 4, 3, 2) -> complex vector indexed (s, spin, site, colour)"""
    return cplx(psi.astype(np.float64)).transpose(1, 2, 0, 3).reshape(-1)


def from_vec(v, V, Ls):
    return reals(v.reshape(Ls, 4, V, 3).transpose(2, 0, 1, 3))


@pytest.mark.parametrize("Ls", [1, 2, 3, 4, 8, 16])
@pytest.mark.parametrize("mass", [0.0, 0.07, 1.0, -1.0])
def test_mooee_matrix_is_the_definition(Ls, mass):
    A = oracle.mooee_matrix(Ls, M5, mass)
    want = dense_mooee(Ls, M5, mass)
    assert np.array_equal(A, want)                                       # exact: entries are sums of a few literals
    assert np.array_equal(oracle.mooee_matrix(Ls, M5, mass, oracle.M5_DAG), want.T)
    Ainv = oracle.mooee_matrix(Ls, M5, mass, oracle.M5_INV)
    assert np.abs(Ainv - np.linalg.inv(want)).max() < 1e-14
    assert np.abs(A @ Ainv - np.eye(4 * Ls)).max() < 1e-14
    assert np.abs(oracle.mooee_matrix(Ls, M5, mass, oracle.M5_INV_DAG) - np.linalg.inv(want).T).max() < 1e-14


@pytest.mark.parametrize("Ls", [1, 2, 5, 16])
@pytest.mark.parametrize("op", [oracle.M5_APPLY, oracle.M5_DAG, oracle.M5_INV, oracle.M5_INV_DAG])
def test_mooee_apply_against_numpy(Ls, op):
    n = 37
    psi = gen.spinor_gaussian(n, Ls, seed=61)
    A = dense_mooee(Ls, M5, MASS)
    B = {oracle.M5_APPLY: A, oracle.M5_DAG: A.T, oracle.M5_INV: np.linalg.inv(A), oracle.M5_INV_DAG: np.linalg.inv(A).T}[op]
    z = cplx(psi).reshape(n, 4 * Ls, 3)
    want = reals(np.einsum("rq,xqc->xrc", B, z).reshape(n, Ls, 4, 3))
    assert rel_err(oracle.mooee(Ls, M5, MASS, psi, op), want) < 1e-14
    # fp32 inputs are promoted exactly
    psi32 = psi.astype(np.float32)
    z = cplx(psi32.astype(np.float64)).reshape(n, 4 * Ls, 3)
    want = reals(np.einsum("rq,xqc->xrc", B, z).reshape(n, Ls, 4, 3))
    assert rel_err(oracle.mooee(Ls, M5, MASS, psi32, op), want) < 1e-14


@pytest.mark.parametrize("Ls", [2, 4, 16])
def test_mooee_inverse_composes_to_identity(Ls):
    psi = gen.spinor_gaussian(50, Ls, seed=62)
    for a, b in ((oracle.M5_APPLY, oracle.M5_INV), (oracle.M5_INV, oracle.M5_APPLY), (oracle.M5_DAG, oracle.M5_INV_DAG)):
        back = oracle.mooee(Ls, M5, MASS, oracle.mooee(Ls, M5, MASS, psi, a), b)
        assert rel_err(back, psi) < 1e-14


def test_mooee_ls1_is_a_mass_term():
    """Ls = 1: both wraps land on the same slice, Mooee = (5 - M5) + m (P_- + P_+) = 5 - M5 + m."""
    psi = gen.spinor_gaussian(20, 1, seed=63)
    assert rel_err(oracle.mooee(1, M5, MASS, psi), (5.0 - M5 + MASS) * psi) < 1e-15
    assert rel_err(oracle.mooee(1, M5, MASS, psi, oracle.M5_INV), psi / (5.0 - M5 + MASS)) < 1e-15


@pytest.mark.parametrize("mass,Ls,n", [(-1.0, 8, 3), (-1.0, 6, 0), (1.0, 8, 2), (1.0, 5, 4)])
def test_mooee_plane_wave_in_s(mass, Ls, n):
    """m = -1 makes the fifth dimension periodic, m = +1 antiperiodic; psi(s) = e^{ips} chi is then an
    eigenvector per chirality: (5 - M5 - e^{-ip}) on P_+ chi (it sees psi(s-1)), (5 - M5 - e^{+ip}) on
    P_- chi (it sees psi(s+1))."""
    p = 2 * np.pi * n / Ls if mass < 0 else (2 * n + 1) * np.pi / Ls
    rng = np.random.default_rng(7)
    chi = rng.normal(size=(11, 4, 3)) + 1j * rng.normal(size=(11, 4, 3))
    psi = np.exp(1j * p * np.arange(Ls))[None, :, None, None] * chi[:, None]
    lam = np.array([5 - M5 - np.exp(-1j * p)] * 2 + [5 - M5 - np.exp(1j * p)] * 2)   # gamma5 = diag(+,+,-,-)
    want = lam[None, None, :, None] * psi
    assert rel_err(oracle.mooee(Ls, M5, mass, reals(psi)), reals(want)) < 1e-14
    assert rel_err(oracle.mooee(Ls, M5, mass, reals(psi), oracle.M5_INV), reals(psi / lam[None, None, :, None])) < 1e-13


@pytest.mark.parametrize("dims,Ls,bc", [((2, 2, 2, 2), 1, 0), ((2, 2, 2, 2), 2, 1), ((2, 2, 2, 2), 4, 0), ((4, 2, 2, 2), 3, 1)])
@pytest.mark.parametrize("dagger", [False, True])
def test_ddwf_dense_matrix(dims, Ls, bc, dagger):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=64)
    psi = gen.spinor_gaussian(V, Ls, seed=64)
    M = dense_dwf_matrix(dims, Ls, U, bc, M5, MASS)
    if dagger:
        M = M.conj().T
    want = from_vec(M @ to_vec(psi), V, Ls)
    assert rel_err(oracle.ddwf(dims, Ls, bc, M5, MASS, U, psi, dagger=dagger), want) < 1e-14


def test_ddwf_ls1_is_the_wilson_matrix():
    """Ls = 1: M = (5 - M5 + m) - Dhop/2, the Wilson matrix built from the pinned Dhop oracle."""
    dims, bc = (4, 2, 4, 2), 1
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=65)
    psi = gen.spinor_gaussian(V, 1, seed=65)
    want = (5.0 - M5 + MASS) * psi - 0.5 * oracle.dhop(dims, 1, bc, U, psi)
    assert rel_err(oracle.ddwf(dims, 1, bc, M5, MASS, U, psi), want) < 1e-15


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 4, 0), ((2, 4, 2, 4), 5, 1)])
def test_gamma5_r5_hermiticity(dims, Ls, bc):
    """M^dagger = (gamma5 R5) M (gamma5 R5), R5: s -> Ls-1-s; the oracle's dagger entry point agrees
    with that sandwich of its plain one, and <phi, M psi> = <M^dag phi, psi>."""
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=66)
    psi = gen.spinor_gaussian(V, Ls, seed=66, stream=gen.STREAM_SPINOR)
    phi = gen.spinor_gaussian(V, Ls, seed=66, stream=gen.STREAM_SPINOR2)
    g5 = np.array([1, 1, -1, -1.0])[None, None, :, None, None]

    def G5R5(f):
        return np.ascontiguousarray(g5 * f[:, ::-1])

    sandwich = G5R5(oracle.ddwf(dims, Ls, bc, M5, MASS, U, G5R5(phi)))
    dag = oracle.ddwf(dims, Ls, bc, M5, MASS, U, phi, dagger=True)
    assert rel_err(dag, sandwich) < 1e-14
    lhs = oracle.inner(phi, oracle.ddwf(dims, Ls, bc, M5, MASS, U, psi))
    rhs = oracle.inner(dag, psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # without the reflection R5 the sandwich is NOT the adjoint (the pin has teeth)
    no_r5 = np.ascontiguousarray(g5 * oracle.ddwf(dims, Ls, bc, M5, MASS, U, np.ascontiguousarray(g5 * phi)))
    assert rel_err(no_r5, dag) > 1e-3


@pytest.mark.parametrize("dims,Ls,bc", [((2, 2, 2, 2), 2, 0), ((2, 2, 2, 2), 4, 1), ((4, 2, 2, 2), 3, 0)])
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("dagger", [False, True])
def test_schur_against_dense_schur_complement(dims, Ls, bc, parity, dagger):
    """S_pp = M_pp - M_pq M_qq^{-1} M_qp taken with numpy from the dense full matrix."""
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=67)
    M = dense_dwf_matrix(dims, Ls, U, bc, M5, MASS)
    par = gen.site_parity(dims)
    # index (s, spin, site, colour): parity of each matrix index
    ipar = np.broadcast_to(par[None, None, :, None], (Ls, 4, V, 3)).reshape(-1)
    P, Q = np.nonzero(ipar == parity)[0], np.nonzero(ipar == 1 - parity)[0]
    S = M[np.ix_(P, P)] - M[np.ix_(P, Q)] @ np.linalg.solve(M[np.ix_(Q, Q)], M[np.ix_(Q, P)])
    if dagger:
        S = S.conj().T
    half = gen.spinor_gaussian(V // 2, Ls, seed=67)
    vec = cplx(half).transpose(1, 2, 0, 3).reshape(-1)                   # (s, spin, cb site, colour): same order as P
    want = reals((S @ vec).reshape(Ls, 4, V // 2, 3).transpose(2, 0, 1, 3))
    assert rel_err(oracle.schur(dims, Ls, bc, M5, MASS, parity, U, half, dagger=dagger), want) < 1e-13


def test_schur_solves_the_full_system():
    """The red-black reduction: with x_p = S^{-1}(b_p - M_pq Mooee^{-1} b_q) and
    x_q = Mooee^{-1}(b_q - M_qp x_p) the full M x = b holds -- checked by applying the oracle's M to a
    solution obtained from the dense matrix."""
    dims, Ls, bc = (2, 2, 2, 2), 3, 1
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=68)
    b = gen.spinor_gaussian(V, Ls, seed=68)
    M = dense_dwf_matrix(dims, Ls, U, bc, M5, MASS)
    x = from_vec(np.linalg.solve(M, to_vec(b)), V, Ls)
    assert rel_err(oracle.ddwf(dims, Ls, bc, M5, MASS, U, x), b) < 1e-13
    # and the even Schur system of that solution
    par = gen.site_parity(dims)
    xe, be, bo = (np.ascontiguousarray(f[par == p]) for f, p in ((x, 0), (b, 0), (b, 1)))
    rhs = be + 0.5 * oracle.dhop_cb(dims, Ls, bc, 0, U, oracle.mooee(Ls, M5, MASS, bo, oracle.M5_INV))
    assert rel_err(oracle.schur(dims, Ls, bc, M5, MASS, 0, U, xe), rhs) < 1e-13
