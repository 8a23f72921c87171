"""GPU parity of the Wilson-matrix fusion: dwf_dhop_oe_axpy / dwf_dhop_eo_axpy,
out = a x + b Dhop in, against a x + b (oracle Dhop) evaluated in fp64 -- on the staged fp32 kernel
(x staged by TMA, combined in the store epilogue; several tiles per CTA) and on the fp64 staged and the
direct kernels (x read at the thread's own site in the epilogue).  Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64)."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}

CASES = [
    # dims, Ls, prec, bc, staged fp32 kernel expected (forced with kernel = 2)
    ((32, 16, 16, 16), 4, 4, 1, True), ((48, 12, 12, 12), 3, 4, 0, True), ((16, 8, 8, 12), 6, 4, 1, True),
    ((8, 8, 12, 8), 5, 4, 0, True), ((8, 8, 8, 8), 8, 8, 1, False), ((24, 4, 4, 4), 5, 4, 1, False),
    ((4, 4, 4, 4), 4, 8, 0, False),
]


@pytest.mark.parametrize("dims,Ls,prec,bc,fused", CASES)
def test_dhop_axpy_matches_oracle(lib, dims, Ls, prec, bc, fused):
    import torch
    a, b = 4.0 + 0.3, -0.5                       # (4 + m) psi - Dhop psi / 2
    V = gen.volume(dims)
    U = gen.gauge_random(dims, 71, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, 71, gen.STREAM_SPINOR, prec)
    xf = gen.spinor_gaussian(V, Ls, 71, gen.STREAM_SPINOR2, prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        if fused:
            g.set_option("kernel", 2)            # the fused kernel or an error
        for p_out in (1, 0):
            half = gen.split_parity(psi, dims, 1 - p_out)
            x = gen.split_parity(xf, dims, p_out)
            fin, fx = g.import_spinor(half, 1 - p_out), g.import_spinor(x, p_out)
            call = g.dhop_oe_axpy if p_out == 1 else g.dhop_eo_axpy
            out = call(fin, fx, a, b)
            want = a * x.astype(np.float64) + b * oracle.dhop_cb(dims, Ls, bc, p_out, U, half)
            assert rel_err(g.export_spinor(out, p_out), want) <= TOL[prec]
            # a = 0, b = 1 is the plain operator, bit for bit (every kernel combines in its store epilogue)
            plain = g.dhop_oe(fin) if p_out == 1 else g.dhop_eo(fin)
            assert torch.equal(call(fin, fx, 0.0, 1.0), plain)
            inplace = fx.clone()                 # x may be the output buffer
            call(fin, inplace, a, b, out=inplace)
            assert torch.equal(inplace, out)
            with pytest.raises(lib.DwfError) as e:
                call(fin, fin, a, b)
            assert e.value.code == lib.ERR_INVALID_ARG


def test_c4_full_size_wilson_schur_step_sampled(lib):
    """32^4 x 16 fp32 (BASELINE.json configs[3] shape): chi_o = DhopOE psi_e, then
    phi_e = psi_e - 1/(4 (4+m)^2) DhopEO chi_o -- the even/odd Schur complement of the Wilson matrix
    up to its overall factor -- on sampled sites."""
    dims, Ls, prec, bc, seed = (32, 32, 32, 32), 16, 4, lib.PERIODIC, 1004
    a, b = 1.0, -0.25 / (4.3 * 4.3)
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec)
    psi_e = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, seed, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        f_e = g.import_spinor(psi_e, lib.EVEN)
        f_o = g.dhop_oe(f_e)
        f_out = g.dhop_eo_axpy(f_o, f_e, a, b)
        chi_o = g.export_spinor(f_o, lib.ODD)
        phi_e = g.export_spinor(f_out, lib.EVEN)
    rng = np.random.default_rng(5)
    even = np.unique(rng.integers(0, gen.volume(dims) // 2, 500)) * 2
    par = gen.site_parity(dims)
    even = even + (par[even] != 0)               # x>>1 is the row; pick the even site of each pair
    rows = even >> 1
    want = a * psi_e[rows].astype(np.float64) + b * oracle.dhop_sites(dims, Ls, bc, U, chi_o, True, even)
    assert rel_err(phi_e[rows], want) <= TOL[prec]
