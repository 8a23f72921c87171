"""The small cases that are run under compute-sanitizer:

    compute-sanitizer --tool memcheck  python -m pytest tests/test_gpu_sanitizer_cases.py -x -q
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_cases.py -x -q

(one tool per GPU call; the summaries are under profiles/).  Every kernel family of the library on a
shape that spans several tiles per CTA: C1, C2, the staged fp32 kernel (all MODEs) and the staged
fp64 kernel on (32,16,16,16) x 4 with a tile switch, the direct kernel, the reductions, the
fifth-dimension passes, the Schur complement and two CG iterations.  Each case is also an ordinary
parity test against the oracle, so the file runs in the plain `-m gpu` suite as well."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}
M5, MASS = 1.8, 0.05


def test_sanitize_c1_full_fp64(lib):
    dims, Ls = (4, 4, 4, 4), 4
    U = gen.gauge_random(dims, 1001, prec=8)
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 1001, prec=8)
    with lib.Geometry(dims, Ls, 8, lib.PERIODIC) as g:
        g.load_gauge(U)
        out = g.dhop(g.import_spinor(psi, lib.FULL))
        assert rel_err(g.export_spinor(out, lib.FULL), oracle.dhop(dims, Ls, 0, U, psi)) <= TOL[8]
        n = g.norm2(out, lib.FULL)
        assert abs(n - oracle.norm2(g.export_spinor(out, lib.FULL))) <= 1e-12 * n


def test_sanitize_c2_full_and_eo_fp64(lib):
    dims, Ls, bc = (8, 8, 8, 8), 8, 1
    U = gen.gauge_random(dims, 1002, prec=8)
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 1002, prec=8)
    with lib.Geometry(dims, Ls, 8, bc) as g:
        g.load_gauge(U)
        out = g.dhop(g.import_spinor(psi, lib.FULL))
        assert rel_err(g.export_spinor(out, lib.FULL), oracle.dhop(dims, Ls, bc, U, psi)) <= TOL[8]
        for p_out in (1, 0):
            half = gen.split_parity(psi, dims, 1 - p_out)
            fin = g.import_spinor(half, 1 - p_out)
            got = g.export_spinor(g.dhop_oe(fin) if p_out else g.dhop_eo(fin), p_out)
            assert rel_err(got, oracle.dhop_cb(dims, Ls, bc, p_out, U, half)) <= TOL[8]


@pytest.mark.parametrize("prec", [4, 8])
def test_sanitize_staged_multi_tile_all_modes(lib, prec):
    """(32,16,16,16) x 4: 256 (fp32) tiles on 148 CTAs, i.e. tile switches with link refill; plain, dagger,
    fused norm2 and fused a x + b Dhop instances of the staged kernels."""
    dims, Ls, bc = (32, 16, 16, 16), 4, 1
    U = gen.gauge_random(dims, 81, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 81, prec=prec)
    xh = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 82, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        fin, fx = g.import_spinor(half, lib.EVEN), g.import_spinor(xh, lib.ODD)
        want = oracle.dhop_cb(dims, Ls, bc, 1, U, half)
        assert rel_err(g.export_spinor(g.dhop_oe(fin), lib.ODD), want) <= TOL[prec]
        fo, n2 = g.dhop_oe_norm2(fin)
        assert abs(n2 - oracle.norm2(g.export_spinor(fo, lib.ODD))) <= 1e-12 * n2
        want_d = oracle.dhop_cb(dims, Ls, bc, 1, U, half, dagger=True)
        assert rel_err(g.export_spinor(g.dhop_oe_dag(fin), lib.ODD), want_d) <= TOL[prec]
        got = g.export_spinor(g.dhop_oe_axpy(fin, fx, 0.75, -0.5), lib.ODD)
        assert rel_err(got, 0.75 * xh.astype(np.float64) - 0.5 * want) <= TOL[prec]


@pytest.mark.parametrize("prec", [4, 8])
def test_sanitize_direct_kernel_and_reductions(lib, prec):
    dims, Ls, bc = (12, 6, 4, 6), 5, 1
    U = gen.gauge_random(dims, 83, prec=prec)
    a = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 83, prec=prec)
    b = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 84, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 1)
        fa, fb = g.import_spinor(a, lib.ODD), g.import_spinor(b, lib.ODD)
        got = g.export_spinor(g.dhop_eo(fa), lib.EVEN)
        assert rel_err(got, oracle.dhop_cb(dims, Ls, bc, 0, U, a)) <= TOL[prec]
        ip = g.inner_product(fa, fb, lib.ODD)
        want = oracle.inner(a, b)
        assert abs(ip - want) <= 1e-12 * np.sqrt(oracle.norm2(a) * oracle.norm2(b))


@pytest.mark.parametrize("prec", [4, 8])
def test_sanitize_fifth_dimension_schur_and_cg(lib, prec):
    dims, Ls, bc = (16, 8, 8, 8), 8, 1
    U = gen.gauge_random(dims, 85, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 85, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fh = g.import_spinor(half, lib.EVEN)
        for inv, op in ((False, oracle.M5_APPLY), (True, oracle.M5_INV)):
            fn = g.mooee_inv if inv else g.mooee
            got = g.export_spinor(fn(fh, lib.EVEN, M5, MASS), lib.EVEN)
            assert rel_err(got, oracle.mooee(Ls, M5, MASS, half, op)) <= TOL[prec]
        got = g.export_spinor(g.schur(fh, lib.EVEN, M5, MASS), lib.EVEN)
        assert rel_err(got, oracle.schur(dims, Ls, bc, M5, MASS, 0, U, half)) <= 2 * TOL[prec]
        x, iters, res = g.cg_schur(fh, lib.EVEN, M5, MASS, 1e-30, 2)     # two iterations, every solver kernel once
        assert iters == 2 and 0.0 < res < 1.0
