"""fp16 STORAGE of spinor fields with fp32 arithmetic (third variant; include/dwf.h dwf_*_f16).

The inputs are fp16-representable numbers (the seeded Gaussian field rounded once with numpy), so both sides start from
the same values: the oracle applies Dhop to them in fp64, the kernel widens them to fp32, accumulates in fp32 and rounds
the result once to fp16.  Bar: per element |got - want| <= 2^-11 |want| (half an fp16 ulp of a normal
number, relative) + 1e-5 max|want| (fp32 accumulation of eight legs, fp16 subnormals); relative L2 error <= 4e-4."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle

pytestmark = pytest.mark.gpu


def _quantise(a):
    return a.astype(np.float16).astype(np.float32)


def _check(got, want):
    want = np.asarray(want, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    scale = np.abs(want).max()
    bound = 2.0 ** -11 * np.abs(want) * 1.001 + 1e-5 * scale
    worst = (np.abs(got - want) - bound).max()
    assert worst <= 0.0, f"element beyond half an fp16 ulp by {worst:.3e}"
    rel = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
    assert rel <= 4e-4, rel
    assert rel >= 1e-5          # the output really is fp16 (an fp32 result would sit at 1e-7)


def test_conversion_is_round_to_nearest_even_and_exact_back(lib):
    import torch
    dims, Ls = (16, 4, 4, 4), 3
    psi = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 401, prec=4)
    psi.reshape(-1)[:7] = [65504.0, -65504.0, 1e-7, -3e-8, 0.0, 1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11]      # max, subnormals, ties
    with lib.Geometry(dims, Ls, 4, lib.PERIODIC) as g:
        f = g.import_spinor(psi, lib.EVEN)
        fh = g.to_f16(f, lib.EVEN)
        assert fh.dtype == torch.float16 and fh.numel() == f.numel()
        assert torch.equal(fh, f.to(torch.float16))                         # the same rounding as the library's own cast
        back = g.export_spinor(g.from_f16(fh, lib.EVEN), lib.EVEN)
        assert np.array_equal(back, _quantise(psi))                         # numpy's round-to-nearest-even, through the layout permutation


@pytest.mark.parametrize("dims,Ls,bc,max_ctas,opts", [((32, 8, 8, 8), 3, 1, 0, {}),     # <16,4,2,2>, the C4 tile
                                                      ((32, 8, 8, 8), 2, 0, 3, {}),     # many tiles per CTA: link refill, zigzag
                                                      ((16, 8, 8, 8), 4, 1, 0, {}),     # <8,4,4,2>
                                                      ((48, 4, 6, 4), 2, 1, 0, {}),     # Lh = 24
                                                      ((64, 4, 4, 6), 2, 0, 0, {}),     # Lh = 32
                                                      ((32, 8, 8, 8), 4, 1, 6, {"ssplit": 2}),
                                                      ((32, 8, 8, 8), 1, 1, 2, {"layered": 0, "zigzag": 0})])
def test_dhop_f16_against_oracle(lib, dims, Ls, bc, max_ctas, opts):
    import torch
    U = gen.gauge_random(dims, 402, prec=4)
    he = _quantise(gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 402, prec=4))
    ho = _quantise(gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 403, prec=4))
    with lib.Geometry(dims, Ls, 4, bc) as g:
        g.load_gauge(U)
        if max_ctas:
            g.set_option("max_ctas", max_ctas)
        for k, v in opts.items():
            g.set_option(k, v)
        fe = g.to_f16(g.import_spinor(he, lib.EVEN), lib.EVEN)
        fo = g.to_f16(g.import_spinor(ho, lib.ODD), lib.ODD)
        out_o = g.dhop_oe_f16(fe)
        out_e = g.dhop_eo_f16(fo)
        assert out_o.dtype == torch.float16
        _check(g.export_spinor(g.from_f16(out_o, lib.ODD), lib.ODD), oracle.dhop_cb(dims, Ls, bc, 1, U, he))
        _check(g.export_spinor(g.from_f16(out_e, lib.EVEN), lib.EVEN), oracle.dhop_cb(dims, Ls, bc, 0, U, ho))
        assert torch.equal(g.dhop_oe_f16(fe), out_o)                        # deterministic
        # against the fp32 path on the same (fp16-representable) input: the only difference is the final rounding
        ref = g.dhop_oe(g.from_f16(fe, lib.EVEN))
        assert torch.equal(out_o, ref.to(torch.float16))


def test_dhop_f16_unsupported_shapes(lib):
    import torch
    with lib.Geometry((24, 8, 6, 8), 2, 4, lib.PERIODIC) as g:             # Lh = 12: fp16 rows of 576 bytes
        g.load_gauge(gen.gauge_random((24, 8, 6, 8), 404, prec=4))
        a, b = g.new_field_f16(lib.EVEN), g.new_field_f16(lib.ODD)
        a.zero_()
        with pytest.raises(lib.DwfError) as e:
            g.dhop_oe_f16(a, b)
        assert e.value.code == lib.ERR_UNSUPPORTED
    with lib.Geometry((16, 4, 4, 4), 2, 8, lib.PERIODIC) as g:             # fp64 geometry
        with pytest.raises(lib.DwfError):
            lib.dwf_to_f16(g.handle, g.new_field(lib.EVEN), lib.EVEN, torch.empty(g.new_field(lib.EVEN).numel(), dtype=torch.float16, device="cuda"))
