"""SURVEY.md 8(f3) on one GPU: the time-decomposed half-Dhop (open-boundary bulk kernel + dwf_face_pack_t +
dwf_face_apply_t, driven by paper_2203_06777_b200/dist.py) against the oracle's Dhop of the WHOLE lattice.
Several ranks are emulated in one process: every virtual rank has its own slab geometry and fields, the phases
(pack, exchange, bulk + faces) run for all ranks in turn and the transport is a device copy between their
buffers -- no kernel ever waits for another rank.  world = 1 is a real configuration (a rank that is its own
neighbour).  Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64)."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}


def run_decomposed(lib, gdims, Ls, prec, bc, world, p_out, dagger, U, half):
    from paper_2203_06777_b200.dist import SlabDhop
    nl = gdims[0] * gdims[1] * gdims[2]
    ops = []

    def transport(me):                       # recv_lo <- lower neighbour's send_up, recv_hi <- upper neighbour's send_down
        me.recv_lo.copy_(ops[me.plan["lower"]].send_up)
        me.recv_hi.copy_(ops[me.plan["upper"]].send_down)

    for r in range(world):
        ops.append(SlabDhop(gdims, Ls, prec, bc, r, world, exchange=transport))
    try:
        fins = []
        for op in ops:
            t0, t1 = op.plan["t0"], op.plan["t1"]
            op.load_gauge(np.ascontiguousarray(U.reshape(-1, 4, 3, 3, 2)[t0 * nl:t1 * nl]))
            fins.append(op.geometry.import_spinor(np.ascontiguousarray(half[t0 * nl // 2:t1 * nl // 2]), 1 - p_out))
        for op, f in zip(ops, fins):
            op.pack(f, p_out, dagger)
        for op in ops:
            op.communicate()
        outs = [op.bulk_and_faces(f, p_out, dagger) for op, f in zip(ops, fins)]
        return np.concatenate([op.geometry.export_spinor(o, p_out) for op, o in zip(ops, outs)])
    finally:
        for op in ops:
            op.close()


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("gdims,Ls,bc,world", [((8, 4, 4, 8), 3, 1, 1), ((8, 4, 4, 8), 3, 0, 2), ((8, 4, 6, 16), 2, 1, 4),
                                               ((32, 8, 8, 16), 4, 1, 2),      # staged kernels, several tiles per slab
                                               ((4, 4, 2, 4), 5, 1, 2)])       # two-layer slabs: every site is a face site
def test_time_decomposed_dhop_matches_global_oracle(lib, gdims, Ls, bc, world, prec):
    U = gen.gauge_random(gdims, 97, prec=prec)
    psi = gen.spinor_gaussian(gen.volume(gdims), Ls, 97, prec=prec)
    for p_out in (1, 0):
        half = gen.split_parity(psi, gdims, 1 - p_out)
        for dagger in (False, True):
            got = run_decomposed(lib, gdims, Ls, prec, bc, world, p_out, dagger, U, half)
            want = oracle.dhop_cb(gdims, Ls, bc, p_out, U, half, dagger=dagger)
            assert rel_err(got, want) <= TOL[prec], (p_out, dagger)


@pytest.mark.parametrize("prec", [4, 8])
def test_open_boundary_bulk_kernel_matches_open_oracle(lib, prec):
    """The slab operator on its own: bc_time = OPEN_T on every kernel family (staged, direct, full field)."""
    for dims, Ls in (((32, 8, 8, 8), 3), ((12, 6, 4, 6), 4), ((8, 8, 8, 2), 2)):
        U = gen.gauge_random(dims, 98, prec=prec)
        psi = gen.spinor_gaussian(gen.volume(dims), Ls, 98, prec=prec)
        with lib.Geometry(dims, Ls, prec, lib.OPEN_T) as g:
            g.load_gauge(U)
            got = g.export_spinor(g.dhop(g.import_spinor(psi, lib.FULL)), lib.FULL)
            assert rel_err(got, oracle.dhop(dims, Ls, oracle.OPEN_T, U, psi)) <= TOL[prec]


def test_one_rank_slab_driver_end_to_end(lib):
    """SlabDhop as a user calls it (world = 1, default transport = copies on the side stream), both parities."""
    from paper_2203_06777_b200.dist import SlabDhop
    gdims, Ls, prec, bc = (16, 8, 8, 8), 4, 4, 1
    U = gen.gauge_random(gdims, 99, prec=prec)
    half = gen.spinor_gaussian(gen.volume(gdims) // 2, Ls, 99, prec=prec)
    op = SlabDhop(gdims, Ls, prec, bc, 0, 1)
    try:
        op.load_gauge(U)
        f_e = op.geometry.import_spinor(half, lib.EVEN)
        f_o = op.dhop_oe(f_e)
        assert rel_err(op.geometry.export_spinor(f_o, lib.ODD), oracle.dhop_cb(gdims, Ls, bc, 1, U, half)) <= TOL[prec]
        f_e2 = op.dhop_eo(f_o)
        want = oracle.dhop_cb(gdims, Ls, bc, 0, U, op.geometry.export_spinor(f_o, lib.ODD))
        assert rel_err(op.geometry.export_spinor(f_e2, lib.EVEN), want) <= TOL[prec]
    finally:
        op.close()
