"""multiple right-hand sides sharing one gauge load (dwf_dhop_oe_mrhs / dwf_dhop_eo_mrhs).
Each right-hand side against the oracle's half-Dhop (the multi-RHS operation IS nrhs independent
Dhops, so the pinned oracle of Dhop is its oracle), and bit-identical to nrhs separate calls.
Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64)."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("dims,Ls,bc,nrhs", [((32, 8, 8, 8), 4, 1, 3),      # staged kernels, Ls * nrhs = 12 slices per tile
                                             ((16, 8, 4, 6), 5, 0, 2),      # odd Ls
                                             ((24, 6, 6, 4), 2, 1, 5),
                                             ((12, 6, 4, 6), 3, 1, 2),      # direct kernel: one launch per right-hand side
                                             ((8, 8, 8, 8), 8, 1, 1)])      # nrhs = 1 is the plain call
def test_multi_rhs_matches_oracle_and_separate_calls(lib, dims, Ls, bc, nrhs, prec):
    import torch
    U = gen.gauge_random(dims, 91, prec=prec)
    halves = [gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 91 + r, prec=prec) for r in range(nrhs)]
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        for p_out in (1, 0):
            fins = [g.import_spinor(h, 1 - p_out) for h in halves]
            batch = torch.cat(fins)
            for dag in (False, True):
                out = (g.dhop_oe_mrhs if p_out else g.dhop_eo_mrhs)(batch, nrhs, dagger=dag)
                outs = out.view(nrhs, -1)
                for r in range(nrhs):
                    want = oracle.dhop_cb(dims, Ls, bc, p_out, U, halves[r], dagger=dag)
                    assert rel_err(g.export_spinor(outs[r].contiguous(), p_out), want) <= TOL[prec], (p_out, dag, r)
                    single = ((g.dhop_oe_dag if dag else g.dhop_oe) if p_out else (g.dhop_eo_dag if dag else g.dhop_eo))(fins[r])
                    assert torch.equal(single, outs[r]), (p_out, dag, r)
        with pytest.raises(lib.DwfError):
            lib.dwf_dhop_oe_mrhs(g.handle, batch, batch, nrhs)                 # in == out
        with pytest.raises(lib.DwfError):
            lib.dwf_dhop_oe_mrhs(g.handle, batch, torch.empty_like(batch), nrhs + 1)   # size mismatch caught by the binding
