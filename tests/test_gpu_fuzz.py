"""Seeded sweep over random geometries (L0 in {8,16,24,32,40,48,56,64} so that most hit the staged fp32 kernel,
the other extents even and ragged, Ls 1..12, both boundary conditions): every half-Dhop entry point
-- plain, dagger, fused norm2, fused axpy -- against the oracle.  Bar: relative L2 error <= 2e-6."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu


def _cases(n=24, seed=12345):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        L0 = int(rng.choice([8, 16, 32, 48, 24, 40, 56, 64]))
        dims = (L0,) + tuple(int(2 * rng.integers(1, 9)) for _ in range(3))
        Ls, bc = int(rng.integers(1, 13)), int(rng.integers(0, 2))
        if gen.volume(dims) * Ls <= 1_500_000:
            out.append((dims, Ls, bc))
    return out


@pytest.mark.parametrize("dims,Ls,bc", _cases())
def test_random_geometry_all_entry_points(lib, dims, Ls, bc):
    V, seed = gen.volume(dims), 100 + Ls
    U = gen.gauge_random(dims, seed, prec=4)
    psi = gen.spinor_gaussian(V, Ls, seed, prec=4)
    xf = gen.spinor_gaussian(V, Ls, seed, gen.STREAM_SPINOR2, 4)
    with lib.Geometry(dims, Ls, 4, bc) as g:
        g.load_gauge(U)
        for p_out in (1, 0):
            half, x = gen.split_parity(psi, dims, 1 - p_out), gen.split_parity(xf, dims, p_out)
            fin, fx = g.import_spinor(half, 1 - p_out), g.import_spinor(x, p_out)
            want = oracle.dhop_cb(dims, Ls, bc, p_out, U, half)
            want_dag = oracle.dhop_cb(dims, Ls, bc, p_out, U, half, dagger=True)
            plain, dag, fused, axpy = ((g.dhop_oe, g.dhop_oe_dag, g.dhop_oe_norm2, g.dhop_oe_axpy) if p_out else
                                       (g.dhop_eo, g.dhop_eo_dag, g.dhop_eo_norm2, g.dhop_eo_axpy))
            assert rel_err(g.export_spinor(plain(fin), p_out), want) <= 2e-6
            assert rel_err(g.export_spinor(dag(fin), p_out), want_dag) <= 2e-6
            out, n = fused(fin)
            got = g.export_spinor(out, p_out)
            assert rel_err(got, want) <= 2e-6
            assert abs(n - oracle.norm2(got)) <= 1e-12 * n
            assert rel_err(g.export_spinor(axpy(fin, fx, 1.7, -0.4), p_out), 1.7 * x.astype(np.float64) - 0.4 * want) <= 2e-6
