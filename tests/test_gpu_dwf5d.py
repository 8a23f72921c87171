"""GPU parity of SURVEY.md 8(f2): the rest of the red-black Shamir domain-wall operator (csrc/dwf5d.cu)
against the oracle (oracle/dwf5d_oracle.c), element by element on identical seeded inputs, through
the C ABI.  Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64) per operator application (the bars of
north_star for Dhop; each of these operators is a short composition of such steps, the Schur complement
the longest: two Dhops and two fifth-dimension passes, held to 2x the bar).  The solver is checked by
the oracle: its solution must satisfy the oracle's Schur operator to the stated residual."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}
M5, MASS = 1.8, 0.07
OPS = [(False, False, oracle.M5_APPLY), (False, True, oracle.M5_DAG), (True, False, oracle.M5_INV), (True, True, oracle.M5_INV_DAG)]


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("dims,Ls", [((4, 4, 4, 4), 1), ((4, 4, 4, 4), 2), ((8, 4, 6, 4), 5), ((8, 8, 8, 8), 8), ((12, 6, 2, 4), 12),
                                     ((32, 4, 4, 4), 16), ((4, 2, 6, 14), 24), ((6, 4, 4, 2), 32), ((4, 4, 2, 2), 40)])
def test_mooee_and_inverse_full_and_half(lib, dims, Ls, prec):
    V = gen.volume(dims)
    psi = gen.spinor_gaussian(V, Ls, 71, prec=prec)
    half = gen.split_parity(psi, dims, 1)
    with lib.Geometry(dims, Ls, prec) as g:
        f, fh = g.import_spinor(psi, lib.FULL), g.import_spinor(half, lib.ODD)
        for inv, dag, op in OPS:
            fn = g.mooee_inv if inv else g.mooee
            got = g.export_spinor(fn(f, lib.FULL, M5, MASS, dagger=dag), lib.FULL)
            assert rel_err(got, oracle.mooee(Ls, M5, MASS, psi, op)) <= TOL[prec], (inv, dag)
            got = g.export_spinor(fn(fh, lib.ODD, M5, MASS, dagger=dag), lib.ODD)
            assert rel_err(got, oracle.mooee(Ls, M5, MASS, half, op)) <= TOL[prec], (inv, dag)
        # the pair composes to the identity on the device, and the in-place form gives the same bits
        back = g.mooee_inv(g.mooee(fh, lib.ODD, M5, MASS), lib.ODD, M5, MASS)
        assert rel_err(g.export_spinor(back, lib.ODD), half) <= TOL[prec]
        if Ls <= 32:
            import torch
            ref = g.mooee_inv(fh, lib.ODD, M5, MASS, dagger=True)
            buf = fh.clone()
            lib.dwf_mooee_inv(g.handle, buf, buf, lib.ODD, M5, MASS, True)
            assert torch.equal(buf, ref)
        else:
            with pytest.raises(lib.DwfError) as e:
                lib.dwf_mooee(g.handle, fh, fh, lib.ODD, M5, MASS)
            assert e.value.code == lib.ERR_UNSUPPORTED


@pytest.mark.parametrize("prec", [4, 8])
def test_mooee_degenerate_masses(lib, prec):
    """m = 0 (open fifth dimension), m = +-1 ((anti)periodic), Ls = 1 (a pure mass term), large mass."""
    dims = (4, 4, 4, 6)
    for Ls, mass in ((8, 0.0), (8, 1.0), (8, -1.0), (1, 0.3), (3, 25.0)):
        half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 72, prec=prec)
        with lib.Geometry(dims, Ls, prec) as g:
            fh = g.import_spinor(half, lib.EVEN)
            for inv, dag, op in OPS:
                fn = g.mooee_inv if inv else g.mooee
                got = g.export_spinor(fn(fh, lib.EVEN, M5, mass, dagger=dag), lib.EVEN)
                assert rel_err(got, oracle.mooee(Ls, M5, mass, half, op)) <= TOL[prec], (Ls, mass, inv, dag)
    with lib.Geometry(dims, 4, prec) as g:
        fh = g.new_field(lib.EVEN)
        with pytest.raises(lib.DwfError) as e:
            g.mooee_inv(fh, lib.EVEN, 5.0, 0.1)                   # 5 - M5 = 0: singular
        assert e.value.code == lib.ERR_INVALID_ARG


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("dims,Ls,bc", [((4, 4, 4, 4), 4, 0), ((8, 8, 8, 8), 8, 1), ((16, 4, 6, 4), 5, 1), ((32, 8, 8, 8), 4, 0)])
def test_ddwf_full_matrix(lib, dims, Ls, bc, prec):
    V = gen.volume(dims)
    U = gen.gauge_random(dims, 73, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, 73, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        f = g.import_spinor(psi, lib.FULL)
        for dag in (False, True):
            got = g.export_spinor(g.ddwf(f, M5, MASS, dagger=dag), lib.FULL)
            assert rel_err(got, oracle.ddwf(dims, Ls, bc, M5, MASS, U, psi, dagger=dag)) <= TOL[prec], dag
        for kernel in (1,):                                      # the direct kernel's fused a x + b Dhop epilogue
            g.set_option("kernel", kernel)
            got = g.export_spinor(g.ddwf(f, M5, MASS), lib.FULL)
            assert rel_err(got, oracle.ddwf(dims, Ls, bc, M5, MASS, U, psi)) <= TOL[prec]


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("dims,Ls,bc", [((8, 8, 8, 8), 8, 1), ((32, 8, 8, 8), 4, 0), ((12, 4, 6, 4), 6, 1), ((16, 16, 16, 16), 16, 0)])
def test_schur_complement(lib, dims, Ls, bc, prec):
    U = gen.gauge_random(dims, 74, prec=prec)
    for parity in (lib.EVEN, lib.ODD):
        half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 74 + parity, prec=prec)
        with lib.Geometry(dims, Ls, prec, bc) as g:
            g.load_gauge(U)
            fh = g.import_spinor(half, parity)
            for dag in (False, True):
                got = g.export_spinor(g.schur(fh, parity, M5, MASS, dagger=dag), parity)
                want = oracle.schur(dims, Ls, bc, M5, MASS, parity, U, half, dagger=dag)
                assert rel_err(got, want) <= 2 * TOL[prec], (parity, dag)
            with pytest.raises(lib.DwfError):
                lib.dwf_schur(g.handle, fh, fh, parity, M5, MASS, g.new_work(lib.dwf_schur_work_bytes(g.handle)))


def test_schur_c4_full_size_sampled_properties(lib):
    """C4 shape (32^4 x 16, fp32, near-unit gauge), the launch configuration bench.py --workload schur
    times: the four kernels against the oracle's Schur operator on the WHOLE even half field."""
    dims, Ls, prec, bc, seed = (32, 32, 32, 32), 16, 4, 0, 1004
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, seed, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        got = g.export_spinor(g.schur(g.import_spinor(half, lib.EVEN), lib.EVEN, M5, 0.01), lib.EVEN)
    want = oracle.schur(dims, Ls, bc, M5, 0.01, 0, U, half)
    assert rel_err(got, want) <= 2 * TOL[prec]


@pytest.mark.parametrize("prec,tol,bar", [(8, 1e-10, 1e-9), (4, 1e-5, 2e-4)])
def test_cg_on_schur_normal_equations_16x16(lib, prec, tol, bar):
    """16^4 x 16: conjugate gradients on S^dag S reach the requested residual; the ORACLE checks the
    solution: |b - S_oracle x| / |b| <= bar (fp64: 1e-9; fp32: 2e-4, the attainable accuracy of a
    single-precision recursive residual on a system of condition number ~1e3)."""
    dims, Ls, bc = (16, 16, 16, 16), 16, 1
    mass = 0.05
    U = gen.gauge_near_unit(dims, 75, 0.2, prec=prec)
    b = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 75, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fb = g.import_spinor(b, lib.EVEN)
        x, iters, res = g.cg_schur(fb, lib.EVEN, M5, mass, tol, 2000)
        sol = g.export_spinor(x, lib.EVEN)
        assert 0 < iters < 2000
        assert res <= bar
        # restart from the solution's residual is not needed: the oracle applies S to the solution
        r = b.astype(np.float64) - oracle.schur(dims, Ls, bc, M5, mass, 0, U, sol)
        true_res = np.linalg.norm(r.ravel()) / np.linalg.norm(b.astype(np.float64).ravel())
        assert true_res <= bar
        assert abs(true_res - res) <= 0.5 * bar                   # the library's own report of it agrees
        # max_iter = 0 returns x = 0 and residual 1
        x0, it0, res0 = g.cg_schur(fb, lib.EVEN, M5, mass, tol, 0)
        assert it0 == 0 and res0 == pytest.approx(1.0) and float(x0.abs().max()) == 0.0


@pytest.mark.parametrize("prec", [4, 8])
def test_red_black_solve_reproduces_the_full_system(lib, prec):
    """The whole red-black chain on the device (prepare source, Schur CG, reconstruct the odd sites) gives
    a full-lattice solution that the ORACLE's unpreconditioned matrix maps back onto the source."""
    dims, Ls, bc, mass = (8, 8, 8, 8), 8, 1, 0.1
    V = gen.volume(dims)
    U = gen.gauge_random(dims, 76, prec=prec)
    eta = gen.spinor_gaussian(V, Ls, 76, prec=prec)
    par = gen.site_parity(dims)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fe, fo = g.import_spinor(gen.split_parity(eta, dims, 0), lib.EVEN), g.import_spinor(gen.split_parity(eta, dims, 1), lib.ODD)
        # b_e = eta_e - M_eo Mooee^{-1} eta_o = eta_e + 1/2 DhopEO Mooee^{-1} eta_o
        rhs = g.dhop_eo_axpy(g.mooee_inv(fo, lib.ODD, M5, mass), fe, 1.0, 0.5)
        xe, iters, res = g.cg_schur(rhs, lib.EVEN, M5, mass, 1e-11 if prec == 8 else 1e-6, 4000)
        # x_o = Mooee^{-1} (eta_o - M_oe x_e) = Mooee^{-1} (eta_o + 1/2 DhopOE x_e)
        xo = g.mooee_inv(g.dhop_oe_axpy(xe, fo, 1.0, 0.5), lib.ODD, M5, mass)
        sol = np.empty_like(eta)
        sol[par == 0], sol[par == 1] = g.export_spinor(xe, lib.EVEN), g.export_spinor(xo, lib.ODD)
    back = oracle.ddwf(dims, Ls, bc, M5, mass, U, sol)
    assert rel_err(back, eta) <= (1e-9 if prec == 8 else 2e-4)
