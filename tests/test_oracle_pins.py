"""Pins for the CPU oracle.  CPU only.

Each pin checks oracle/ against something other than itself: a dense matrix assembled a
different way, a closed form, or an invariant of the operator.  A dropped term, a wrong sign
or index, a transposed link or a wrong parity rule fails at least one of them.
"""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import (GAMMA5, apply_dense, coords, cplx, dense_dhop_matrix, lex, pauli_gammas, reals,
                   rel_err, shift_index)

TINY = [((2, 2, 2, 2), 2), ((4, 2, 4, 2), 3), ((2, 4, 2, 6), 1)]


def test_gamma_algebra_and_basis():
    g_or = [oracle.gamma(mu) for mu in range(4)]
    g_pa = pauli_gammas()
    for mu in range(4):
        assert np.array_equal(g_or[mu], g_or[mu].conj().T)
        assert np.allclose(g_or[mu], g_pa[mu], atol=0)           # same basis, built two ways
        for nu in range(4):
            anti = g_or[mu] @ g_or[nu] + g_or[nu] @ g_or[mu]
            assert np.allclose(anti, 2 * np.eye(4) * (mu == nu), atol=0)
    assert np.allclose(g_or[0] @ g_or[1] @ g_or[2] @ g_or[3], GAMMA5, atol=0)


@pytest.mark.parametrize("dims,Ls", TINY)
@pytest.mark.parametrize("bc", [oracle.PERIODIC, oracle.ANTIPERIODIC_T])
def test_p1_dense_matrix(dims, Ls, bc):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=11)
    psi = gen.spinor_gaussian(V, Ls, seed=11)
    D = dense_dhop_matrix(dims, U, bc == oracle.ANTIPERIODIC_T)
    want = apply_dense(D, psi)
    got = oracle.dhop(dims, Ls, bc, U, psi)
    assert rel_err(got, want) < 1e-14


def test_p1_dense_matrix_4x4x4x4():
    dims, Ls = (4, 4, 4, 4), 1
    V = 256
    U = gen.gauge_random(dims, seed=1001)
    psi = gen.spinor_gaussian(V, Ls, seed=1001)
    D = dense_dhop_matrix(dims, U, True)
    assert rel_err(oracle.dhop(dims, Ls, oracle.ANTIPERIODIC_T, U, psi), apply_dense(D, psi)) < 1e-14


def test_p1_dense_matrix_fp32_inputs_promoted_exactly():
    dims, Ls = (2, 4, 2, 2), 2
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=5, prec=4)
    psi = gen.spinor_gaussian(V, Ls, seed=5, prec=4)
    D = dense_dhop_matrix(dims, U, False)
    assert rel_err(oracle.dhop(dims, Ls, 0, U, psi), apply_dense(D, psi)) < 1e-14


@pytest.mark.parametrize("dims,n,bc", [
    ((4, 4, 4, 4), (0, 0, 0, 0), 0),
    ((4, 6, 2, 8), (1, 2, 1, 3), 0),
    ((4, 6, 2, 8), (3, 5, 0, 2), 1),
    ((8, 8, 8, 8), (7, 1, 4, 5), 1),
])
def test_p2_free_field_plane_wave(dims, n, bc):
    Ls = 3
    V = int(np.prod(dims))
    U = gen.gauge_unit(dims)
    p = np.array([2 * np.pi * n[mu] / dims[mu] for mu in range(4)])
    if bc:
        p[3] = (2 * n[3] + 1) * np.pi / dims[3]
    rng = np.random.default_rng(3)
    chi = rng.normal(size=(Ls, 4, 3)) + 1j * rng.normal(size=(Ls, 4, 3))
    phase = np.exp(1j * (coords(dims) @ p))
    psi = phase[:, None, None, None] * chi[None]
    g = pauli_gammas()
    M = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * g[mu] for mu in range(4))
    want = np.einsum("ab,xsbc->xsac", M, psi)
    got = oracle.dhop(dims, Ls, bc, U, reals(psi))
    assert rel_err(got, reals(want)) < 1e-13
    if not bc and not any(n):
        assert rel_err(got, 8 * reals(psi)) < 1e-14           # p = 0: Dhop psi = 8 psi


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 2, 0), ((4, 4, 2, 6), 3, 1)])
def test_p3_gamma5_hermiticity(dims, Ls, bc):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=21)
    psi = gen.spinor_gaussian(V, Ls, seed=21, stream=gen.STREAM_SPINOR)
    phi = gen.spinor_gaussian(V, Ls, seed=21, stream=gen.STREAM_SPINOR2)
    g5 = np.array([1, 1, -1, -1.0])[None, None, :, None, None]
    lhs = oracle.inner(phi, oracle.dhop(dims, Ls, bc, U, psi))
    g5Dg5phi = g5 * oracle.dhop(dims, Ls, bc, U, np.ascontiguousarray(g5 * phi))
    rhs = oracle.inner(np.ascontiguousarray(g5Dg5phi), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # and Dhop is NOT hermitian without the gamma5's (the test has teeth)
    plain = oracle.inner(oracle.dhop(dims, Ls, bc, U, phi), psi)
    assert abs(lhs - plain) / abs(lhs) > 1e-3


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 2, 0), ((2, 4, 4, 4), 2, 1)])
def test_p4_gauge_covariance(dims, Ls, bc):
    V = int(np.prod(dims))
    U = cplx(gen.gauge_random(dims, seed=31))                     # (V,4,3,3)
    psi = cplx(gen.spinor_gaussian(V, Ls, seed=31))               # (V,Ls,4,3)
    g = cplx(gen.su3_random(V, seed=31))                          # (V,3,3)
    Ut = np.empty_like(U)
    for mu in range(4):
        gp = g[shift_index(dims, mu, +1)]
        Ut[:, mu] = np.einsum("xab,xbc,xdc->xad", g, U[:, mu], gp.conj())
    psit = np.einsum("xab,xsib->xsia", g, psi)
    lhs = oracle.dhop(dims, Ls, bc, reals(Ut), reals(psit))
    rhs = np.einsum("xab,xsib->xsia", g, cplx(oracle.dhop(dims, Ls, bc, reals(U), reals(psi))))
    assert rel_err(lhs, reals(rhs)) < 1e-14


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 2, 0), ((2, 2, 4, 6), 3, 1), ((4, 4, 4, 4), 2, 1)])
def test_p5_even_odd_reassembly(dims, Ls, bc):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=41)
    psi = gen.spinor_gaussian(V, Ls, seed=41)
    par = gen.site_parity(dims)
    full = oracle.dhop(dims, Ls, bc, U, psi)
    out_o = oracle.dhop_oe(dims, Ls, bc, U, gen.split_parity(psi, dims, 0))
    out_e = oracle.dhop_eo(dims, Ls, bc, U, gen.split_parity(psi, dims, 1))
    # half-field index must be x>>1 within each parity
    x = np.arange(V)
    assert np.array_equal(np.sort(x[par == 0] >> 1), np.arange(V // 2))
    re = np.empty_like(full)
    re[x[par == 1]] = out_o[x[par == 1] >> 1]
    re[x[par == 0]] = out_e[x[par == 0] >> 1]
    assert rel_err(re, full) < 1e-15
    # Dhop of an even-only field has exactly zero even components
    psi_e = psi.copy()
    psi_e[par == 1] = 0
    assert np.all(oracle.dhop(dims, Ls, bc, U, psi_e)[par == 0] == 0)


def test_p5_cb_rejects_odd_extent():
    with pytest.raises(ValueError):
        oracle.dhop_cb((3, 2, 2, 2), 1, 0, 1, gen.gauge_unit((3, 2, 2, 2)),
                       np.zeros((12, 1, 4, 3, 2)))


def test_p6_s_equivariance():
    dims, Ls = (2, 4, 2, 4), 5
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=51)
    psi = gen.spinor_gaussian(V, Ls, seed=51)
    perm = np.array([3, 0, 4, 1, 2])
    a = oracle.dhop(dims, Ls, 1, U, psi)
    b = oracle.dhop(dims, Ls, 1, U, np.ascontiguousarray(psi[:, perm]))
    assert np.array_equal(a[:, perm], b)
    one = oracle.dhop(dims, 1, 1, U, np.ascontiguousarray(psi[:, 2:3]))
    assert np.array_equal(one[:, 0], a[:, 2])


def test_p7_linearity_and_translation():
    dims, Ls = (4, 2, 2, 4), 2
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=61)
    psi = cplx(gen.spinor_gaussian(V, Ls, seed=61, stream=1))
    phi = cplx(gen.spinor_gaussian(V, Ls, seed=61, stream=2))
    a, b = 0.3 - 1.1j, -2.0 + 0.5j
    D = lambda z: cplx(oracle.dhop(dims, Ls, 0, U, reals(z)))
    assert rel_err(reals(D(a * psi + b * phi)), reals(a * D(psi) + b * D(phi))) < 1e-14
    # translation by one site in each direction (periodic): shifting U and psi shifts the output
    for mu in range(4):
        nb = shift_index(dims, mu, +1)
        Us = np.ascontiguousarray(U[nb])
        shifted = cplx(oracle.dhop(dims, Ls, 0, Us, reals(psi[nb])))
        assert rel_err(reals(shifted), reals(D(psi)[nb])) < 1e-15


def test_p8_norm_bound_and_unitary_links():
    dims, Ls = (8, 8, 8, 8), 2
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=71)
    psi = gen.spinor_gaussian(V, Ls, seed=71)
    out = oracle.dhop(dims, Ls, 1, U, psi)
    ratio = np.sqrt(oracle.norm2(out) / oracle.norm2(psi))
    assert 1.0 < ratio <= 8.0


def test_p9_norm2_and_inner():
    assert oracle.norm2(np.full(1000, 0.5)) == 250.0
    rng = np.random.default_rng(0)
    for dt, tol in ((np.float64, 1e-14), (np.float32, 1e-14)):
        x = rng.normal(size=(501, 2)).astype(dt)
        y = rng.normal(size=(501, 2)).astype(dt)
        ref = np.sum(x.astype(np.float64) ** 2)
        assert abs(oracle.norm2(x) - ref) / ref < tol
        want = np.vdot(cplx(x.astype(np.float64)), cplx(y.astype(np.float64)))
        assert abs(oracle.inner(x, y) - want) / abs(want) < 1e-13
    # compensated sum survives a cancellation-prone sequence
    z = np.array([1e8, 1.0, 1e-4] * 1000)
    assert abs(oracle.norm2(z) - 1000 * (1e16 + 1.0 + 1e-8)) / 1e19 < 1e-15


def test_sites_subset_matches_full_and_cb():
    dims, Ls, bc = (4, 4, 2, 6), 2, 1
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=81, prec=4)
    psi = gen.spinor_gaussian(V, Ls, seed=81, prec=4)
    full = oracle.dhop(dims, Ls, bc, U, psi)
    sites = np.array([0, 5, 17, V - 1, V // 2])
    assert np.array_equal(oracle.dhop_sites(dims, Ls, bc, U, psi, False, sites), full[sites])
    par = gen.site_parity(dims)
    odd = np.arange(V)[par == 1][[0, 3, 40, -1]]
    sub = oracle.dhop_sites(dims, Ls, bc, U, gen.split_parity(psi, dims, 0), True, odd)
    assert np.array_equal(sub, full[odd])


# ---- Dhop^dagger: the oracle's projector swap against the matrix adjoint ------------

@pytest.mark.parametrize("dims,Ls", TINY)
@pytest.mark.parametrize("bc", [oracle.PERIODIC, oracle.ANTIPERIODIC_T])
def test_dagger_is_the_adjoint_of_the_dense_matrix(dims, Ls, bc):
    """numpy's conjugate transpose of the brute-force matrix knows nothing about projectors."""
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=21)
    psi = gen.spinor_gaussian(V, Ls, seed=21)
    D = dense_dhop_matrix(dims, U, bc == oracle.ANTIPERIODIC_T)
    assert rel_err(oracle.dhop(dims, Ls, bc, U, psi, dagger=True), apply_dense(D.conj().T, psi)) < 1e-14
    assert rel_err(oracle.dhop(dims, Ls, bc, U, psi, dagger=True), oracle.dhop(dims, Ls, bc, U, psi)) > 0.1


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 2, 0), ((4, 4, 2, 6), 3, 1)])
def test_dagger_is_gamma5_dhop_gamma5_and_adjoint_under_the_inner_product(dims, Ls, bc):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=22)
    psi = gen.spinor_gaussian(V, Ls, seed=22, stream=gen.STREAM_SPINOR)
    phi = gen.spinor_gaussian(V, Ls, seed=22, stream=gen.STREAM_SPINOR2)
    g5 = np.array([1.0, 1.0, -1.0, -1.0]).reshape(1, 1, 4, 1, 1)
    # gamma5-hermiticity, using only the plain (non-dagger) oracle on the right-hand side
    assert rel_err(oracle.dhop(dims, Ls, bc, U, psi, dagger=True), g5 * oracle.dhop(dims, Ls, bc, U, g5 * psi)) < 1e-14
    # <phi, D psi> = <D^dag phi, psi>
    lhs = oracle.inner(phi, oracle.dhop(dims, Ls, bc, U, psi))
    rhs = oracle.inner(oracle.dhop(dims, Ls, bc, U, phi, dagger=True), psi)
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


@pytest.mark.parametrize("dims,Ls,bc", [((4, 2, 4, 2), 2, 0), ((2, 2, 4, 6), 3, 1)])
def test_dagger_even_odd_reassembly(dims, Ls, bc):
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=23)
    psi = gen.spinor_gaussian(V, Ls, seed=23)
    full = oracle.dhop(dims, Ls, bc, U, psi, dagger=True)
    par = gen.site_parity(dims)
    for p_out in (0, 1):
        half = gen.split_parity(psi, dims, 1 - p_out)
        got = oracle.dhop_cb(dims, Ls, bc, p_out, U, half, dagger=True)
        assert rel_err(got, full[par == p_out]) < 1e-15


def test_wilson_combination_is_the_dense_matrix_a_plus_b_dhop():
    """a x + b Dhop x, as the GPU's fused axpy tests form it from the oracle, against (a 1 + b D) x."""
    dims, Ls, bc = (4, 2, 4, 2), 2, oracle.ANTIPERIODIC_T
    V = int(np.prod(dims))
    U = gen.gauge_random(dims, seed=31)
    psi = gen.spinor_gaussian(V, Ls, seed=31)
    a, b = 4.3, -0.5
    D = dense_dhop_matrix(dims, U, True)
    M = a * np.eye(D.shape[0]) + b * D
    assert rel_err(a * psi + b * oracle.dhop(dims, Ls, bc, U, psi), apply_dense(M, psi)) < 1e-14


def test_golden_fixture():
    """tests/golden/dhop_2x2x2x2.txt (written by tests/golden/make_golden.py from the oracle alone):
    the oracle still produces it, and the stored numbers satisfy the dense-matrix pin themselves."""
    import os
    here = os.path.dirname(os.path.abspath(__file__))
    stored = np.loadtxt(os.path.join(here, "golden", "dhop_2x2x2x2.txt"))
    dims, Ls, seed = (2, 2, 2, 2), 1, 2203
    U = gen.gauge_random(dims, seed)
    psi = gen.spinor_gaussian(16, Ls, seed)
    d = oracle.dhop(dims, Ls, oracle.ANTIPERIODIC_T, U, psi)
    dd = oracle.dhop(dims, Ls, oracle.ANTIPERIODIC_T, U, psi, dagger=True)
    assert np.allclose(stored[:, 0], d.ravel(), rtol=0, atol=1e-14)
    assert np.allclose(stored[:, 1], dd.ravel(), rtol=0, atol=1e-14)
    D = dense_dhop_matrix(dims, U, True)
    assert rel_err(stored[:, 0].reshape(d.shape), apply_dense(D, psi)) < 1e-14
    assert rel_err(stored[:, 1].reshape(d.shape), apply_dense(D.conj().T, psi)) < 1e-14


def test_reconstruct12_is_the_identity_on_su3_and_pins_the_third_row():
    """SURVEY.md 8(f4) oracle helper: for exact SU(3) links (fp64 generator) the rebuilt third row IS the third row
    (unitarity and det = 1 fix it); independent statement: the rebuilt matrix is unitary with determinant 1
    (numpy.linalg), whatever the third row of the input was; rows 0, 1 are untouched bit for bit."""
    dims = (4, 2, 4, 2)
    U = gen.gauge_random(dims, 31, prec=8)
    R = oracle.reconstruct12(U)
    assert np.abs(R - U).max() <= 1e-13
    junk = U.copy()
    junk[..., 2, :, :] = 7.0                                  # a wrong third row is ignored and replaced
    R2 = oracle.reconstruct12(junk)
    assert np.array_equal(R2[..., :2, :, :], U[..., :2, :, :])
    z = R2[..., 0] + 1j * R2[..., 1]
    eye = np.einsum("...ab,...cb->...ac", z, z.conj())
    assert np.abs(eye - np.eye(3)).max() <= 1e-13
    assert np.abs(np.linalg.det(z) - 1.0).max() <= 1e-13
    # fp32-rounded links: rows 0, 1 are the fp32 values exactly, row 2 moves by a few fp32 ulps only
    U32 = gen.gauge_random(dims, 31, prec=4)
    R32 = oracle.reconstruct12(U32)
    assert R32.dtype == np.float64 and np.array_equal(R32[..., :2, :, :], U32[..., :2, :, :].astype(np.float64))
    assert 0 < np.abs(R32 - U32).max() <= 5e-7


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 4, 2), (2, 4, 2, 6)])
def test_open_time_boundary_against_dense_matrix_and_slab_identity(dims):
    """SURVEY.md 8(f3) / DESIGN.md reading #26: bc code 2 drops the hops that wrap in time.  Pins: the dense
    Kronecker matrix with the wrapping blocks of W_3 left out (full, checkerboarded, dagger); and the slab identity
    the domain decomposition rests on: the periodic (antiperiodic) Dhop on the whole lattice, restricted to a
    time slab, equals the open-boundary Dhop of the slab plus terms that involve ONLY the neighbouring slabs'
    boundary layers (changing the other slab's interior does not change the difference)."""
    Ls = 2
    U = gen.gauge_random(dims, 17, prec=8)
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 17, prec=8)
    D = dense_dhop_matrix(dims, U, 2)
    assert rel_err(oracle.dhop(dims, Ls, oracle.OPEN_T, U, psi), apply_dense(D, psi)) <= 1e-14
    assert rel_err(oracle.dhop(dims, Ls, oracle.OPEN_T, U, psi, dagger=True), apply_dense(D.conj().T, psi)) <= 1e-14
    par = gen.site_parity(dims)
    full = oracle.dhop(dims, Ls, oracle.OPEN_T, U, psi)
    for p_out in (0, 1):
        got = oracle.dhop_cb(dims, Ls, oracle.OPEN_T, p_out, U, gen.split_parity(psi, dims, 1 - p_out))
        assert rel_err(got, full[par == p_out]) <= 1e-14
    if dims[3] >= 4:
        # two slabs along time: lower = x3 < L3/2.  V4 is lexicographic with x3 slowest, so a slab is a contiguous block
        L3h = dims[3] // 2
        ld = dims[:3] + (L3h,)
        nl = gen.volume(ld)
        Ul = U.reshape(gen.volume(dims), 4, 3, 3, 2)[:nl]
        for bc in (oracle.PERIODIC, oracle.ANTIPERIODIC_T):
            glob = oracle.dhop(dims, Ls, bc, U, psi)[:nl]
            loc = oracle.dhop(ld, Ls, oracle.OPEN_T, Ul, psi[:nl])
            diff = glob - loc
            # the difference lives on the slab's two boundary layers only ...
            layer = gen.volume(ld[:3] + (1,))
            assert np.abs(diff[layer:nl - layer]).max() == 0.0 if L3h > 2 else True
            assert np.abs(diff).max() > 0.1
            # ... and does not see the interior of the other slab
            psi2 = psi.copy()
            if dims[3] - L3h > 2:
                psi2[nl + layer:-layer] = 0.0
                glob2 = oracle.dhop(dims, Ls, bc, U, psi2)[:nl]
                assert np.array_equal(glob2 - loc, diff)
