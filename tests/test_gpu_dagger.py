"""GPU parity of Dhop^dagger: dwf_dhop_dag / dwf_dhop_oe_dag / dwf_dhop_eo_dag against
the oracle's adjoint (pinned in tests/test_oracle_pins.py by the conjugate transpose of the dense
matrix), on the direct kernel (fp64, shapes without a staged variant) and on the staged fp32 kernel
with several tiles per CTA; plus the adjoint relation <phi, D psi> = <D^dag phi, psi> evaluated
entirely on the GPU.  Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64)."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}

CASES = [
    # dims, Ls, prec, bc, staged kernel expected
    ((4, 4, 4, 4), 4, 8, 0, False), ((8, 8, 8, 8), 8, 8, 1, False), ((6, 4, 10, 2), 3, 8, 1, False),
    ((24, 4, 4, 4), 5, 4, 1, False), ((2, 2, 2, 2), 1, 4, 0, False),
    ((32, 16, 16, 16), 4, 4, 1, True), ((48, 12, 12, 12), 3, 4, 0, True), ((16, 8, 8, 12), 6, 4, 1, True),
]


@pytest.mark.parametrize("dims,Ls,prec,bc,staged", CASES)
def test_dagger_full_and_checkerboarded(lib, dims, Ls, prec, bc, staged):
    V = gen.volume(dims)
    U = gen.gauge_random(dims, 61, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, 61, prec=prec)
    want = oracle.dhop(dims, Ls, bc, U, psi, dagger=True)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        if staged:
            g.set_option("kernel", 2)
        got = g.export_spinor(g.dhop_dag(g.import_spinor(psi, lib.FULL)), lib.FULL)
        assert rel_err(got, want) <= TOL[prec]
        for p_out in (1, 0):
            half = gen.split_parity(psi, dims, 1 - p_out)
            fin = g.import_spinor(half, 1 - p_out)
            fo = g.dhop_oe_dag(fin) if p_out == 1 else g.dhop_eo_dag(fin)
            got_h = g.export_spinor(fo, p_out)
            assert rel_err(got_h, oracle.dhop_cb(dims, Ls, bc, p_out, U, half, dagger=True)) <= TOL[prec]
            assert rel_err(got_h, gen.split_parity(want, dims, p_out)) <= TOL[prec]
        # it is not the plain operator
        plain = g.export_spinor(g.dhop(g.import_spinor(psi, lib.FULL)), lib.FULL)
        assert rel_err(plain, want) > 0.1


@pytest.mark.parametrize("dims,Ls,prec", [((32, 16, 16, 16), 8, 4), ((8, 8, 8, 16), 6, 8)])
def test_adjoint_relation_on_the_gpu(lib, dims, Ls, prec):
    """<phi, D psi> = <D^dag phi, psi> with random SU(3) links, antiperiodic time; both sides from
    the CUDA path (fp64-accumulating inner product)."""
    V = gen.volume(dims)
    U = gen.gauge_random(dims, 62, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, 62, gen.STREAM_SPINOR, prec)
    phi = gen.spinor_gaussian(V, Ls, 62, gen.STREAM_SPINOR2, prec)
    with lib.Geometry(dims, Ls, prec, lib.ANTIPERIODIC_T) as g:
        g.load_gauge(U)
        fpsi, fphi = g.import_spinor(psi), g.import_spinor(phi)
        lhs = g.inner_product(fphi, g.dhop(fpsi))
        rhs = g.inner_product(g.dhop_dag(fphi), fpsi)
        scale = np.sqrt(g.norm2(fphi) * g.norm2(fpsi)) * 8
        assert abs(lhs - rhs) <= (1e-6 if prec == 4 else 1e-13) * scale


def test_dagger_argument_errors(lib):
    dims, Ls = (4, 4, 4, 4), 2
    with lib.Geometry(dims, Ls, 4) as g:
        f = g.new_field()
        with pytest.raises(lib.DwfError) as e:
            g.dhop_dag(f)
        assert e.value.code == lib.ERR_NO_GAUGE
        g.load_gauge(gen.gauge_unit(dims, 4))
        with pytest.raises(lib.DwfError) as e:
            lib.dwf_dhop_dag(g.handle, f, f)
        assert e.value.code == lib.ERR_INVALID_ARG
