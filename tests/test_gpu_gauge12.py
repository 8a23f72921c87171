"""Dhop with 12-real link storage (option "gauge12"): the staged fp32 kernel reads rows 0, 1 of
every link and rebuilds row 2 = conj(row0 x row1) once per tile.  Oracle: the plain Dhop oracle applied to the
links of oracle.reconstruct12 (rows 0, 1 as given, third row rebuilt in fp64) -- both sides work with the same
mathematical links, the bar is the fp32 bar of north_star (relative L2 error <= 2e-6).  With antiperiodic time the
library folds the boundary sign into the stored rows, so the rebuilt row of a wrapping link must get it back."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,Ls,bc", [((32, 8, 8, 8), 4, 1),       # <16,4,2,2>: 64 tiles
                                        ((32, 16, 16, 16), 3, 1),    # 256 tiles on 148 CTAs: tile switches, refill of rows 0, 1
                                        ((16, 8, 4, 6), 5, 0), ((24, 8, 6, 4), 2, 1), ((8, 8, 8, 2), 6, 1)])   # L3 = 2: both time hops wrap
def test_gauge12_matches_oracle_with_rebuilt_links(lib, dims, Ls, bc):
    import torch
    U = gen.gauge_random(dims, 95, prec=4)
    U12 = oracle.reconstruct12(U)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 95, prec=4)
    with lib.Geometry(dims, Ls, 4, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        ref = {p: (g.dhop_oe if p else g.dhop_eo)(g.import_spinor(half, 1 - p)).clone() for p in (1, 0)}
        g.set_option("gauge12", 1)
        with pytest.raises(lib.DwfError) as e:                    # the compressed copy is built by the next load_gauge
            g.dhop_oe(g.import_spinor(half, lib.EVEN))
        assert e.value.code == lib.ERR_NO_GAUGE
        g.load_gauge(U)
        for p_out in (1, 0):
            fin = g.import_spinor(half, 1 - p_out)
            out = (g.dhop_oe if p_out else g.dhop_eo)(fin)
            got = g.export_spinor(out, p_out)
            assert rel_err(got, oracle.dhop_cb(dims, Ls, bc, p_out, U12, half)) <= 2e-6
            # close to, but not the same bits as, the 18-real path (the third rows differ by fp32 roundings)
            assert rel_err(got, g.export_spinor(ref[p_out], p_out)) <= 2e-6
            assert torch.equal((g.dhop_oe if p_out else g.dhop_eo)(fin), out)          # deterministic
            # the other entry points keep using the full links
            d = (g.dhop_oe_dag if p_out else g.dhop_eo_dag)(fin)
            assert rel_err(g.export_spinor(d, p_out), oracle.dhop_cb(dims, Ls, bc, p_out, U, half, dagger=True)) <= 2e-6
        g.set_option("gauge12", 0)
        assert torch.equal(g.dhop_eo(g.import_spinor(half, lib.ODD)), ref[0])


def test_gauge12_rejected_for_fp64(lib):
    with lib.Geometry((8, 8, 8, 8), 4, 8) as g:
        with pytest.raises(lib.DwfError) as e:
            g.set_option("gauge12", 1)
        assert e.value.code == lib.ERR_UNSUPPORTED
