"""SURVEY.md 8(f3) on CPU: the host-side logic of the time decomposition (paper_2203_06777_b200/dist.py).

* slab_plan: neighbours, layer ranges, boundary signs, rejected splits.
* two gloo ranks run the WHOLE decomposed half-Dhop on CPU -- the oracle's open-boundary Dhop as the slab
  operator, the face terms restated here in numpy from DESIGN.md reading #26, dist.exchange_faces as the
  transport -- and together reproduce the oracle's Dhop of the whole lattice: the exchange pattern (who gets
  which buffer, also when both neighbours are the same peer), the slab slicing and the antiperiodic signs."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_slab_plan():
    from paper_2203_06777_b200.dist import slab_plan
    p = slab_plan(0, 4, 32, 1)
    assert (p["lower"], p["upper"], p["t0"], p["t1"], p["local_L3"]) == (3, 1, 0, 8, 8)
    assert (p["sign_lo"], p["sign_hi"]) == (-1.0, 1.0)
    p = slab_plan(3, 4, 32, 1)
    assert (p["lower"], p["upper"], p["sign_lo"], p["sign_hi"]) == (2, 0, 1.0, -1.0)
    p = slab_plan(0, 1, 8, 1)
    assert (p["lower"], p["upper"], p["sign_lo"], p["sign_hi"]) == (0, 0, -1.0, -1.0)
    assert slab_plan(1, 2, 8, 0)["sign_lo"] == 1.0
    for bad in ((0, 3, 32), (0, 4, 12), (0, 8, 8), (2, 2, 8)):       # not divisible, odd slabs, one-layer slabs, bad rank
        with pytest.raises(ValueError):
            slab_plan(bad[0], bad[1], bad[2], 0)


# ---- numpy restatement of the face terms (test-side; complex arrays (site, s, spin, colour)) ----
def _cplx(a):
    return a[..., 0] + 1j * a[..., 1]


def _layer_sites(dims, x3, parity):
    """lexicographic indices of the sites of `parity` in time layer x3, increasing"""
    nl = dims[0] * dims[1] * dims[2]
    x = np.arange(nl)
    s = x % dims[0] + (x // dims[0]) % dims[1] + x // (dims[0] * dims[1]) + x3
    return x[(s & 1) == parity] + nl * x3


def face_pack(dims, U, psi_half, q, dagger):
    """(send_down, send_up) of a slab: half spinors (site, s, 2, 3)"""
    nlh = dims[0] * dims[1] * dims[2] // 2
    z = _cplx(psi_half.astype(np.float64))
    sg = 1.0 if dagger else -1.0
    first, last = z[:nlh], z[-nlh:]
    send_down = first[:, :, 0:2] + sg * first[:, :, 2:4]                  # (1 - gamma_t) psi  (dagger: 1 + gamma_t)
    h = last[:, :, 0:2] - sg * last[:, :, 2:4]                            # (1 + gamma_t) psi  (dagger: 1 - gamma_t)
    Ut = _cplx(U.astype(np.float64)).reshape(-1, 4, 3, 3)[_layer_sites(dims, dims[3] - 1, q), 3]
    send_up = np.einsum("xba,xsgb->xsga", Ut.conj(), h)                   # U_t^dag(y) h
    return send_down, send_up


def face_apply(dims, U, out_half, recv_lo, recv_hi, p, dagger, sign_lo, sign_hi):
    nlh = dims[0] * dims[1] * dims[2] // 2
    sg = -1.0 if dagger else 1.0
    out = out_half.copy()
    out[:nlh, :, 0:2] += sign_lo * recv_lo                                # backward hop: (1 + gamma_t): r2 = +h0, r3 = +h1
    out[:nlh, :, 2:4] += sign_lo * sg * recv_lo
    Ut = _cplx(U.astype(np.float64)).reshape(-1, 4, 3, 3)[_layer_sites(dims, dims[3] - 1, p), 3]
    chi = np.einsum("xab,xsgb->xsga", Ut, recv_hi)                        # forward hop: U_t(x) h, (1 - gamma_t): r2 = -chi0
    out[-nlh:, :, 0:2] += sign_hi * chi
    out[-nlh:, :, 2:4] -= sign_hi * sg * chi
    return out


def _worker(rank, world, port, bc, dagger, out_path):
    sys.path.insert(0, ROOT)
    import dwf_inputs as gen
    import oracle
    from paper_2203_06777_b200.dist import exchange_faces, slab_plan
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    gdims, Ls = (4, 2, 2, 4 * world), 2
    U = gen.gauge_random(gdims, 21, prec=8)
    p_out = 1
    half = gen.spinor_gaussian(gen.volume(gdims) // 2, Ls, 21, prec=8)           # global even half field
    plan = slab_plan(rank, world, gdims[3], bc)
    ld = gdims[:3] + (plan["local_L3"],)
    nl = gdims[0] * gdims[1] * gdims[2]
    Ul = U.reshape(-1, 4, 3, 3, 2)[plan["t0"] * nl:plan["t1"] * nl]
    hl = half[plan["t0"] * nl // 2:plan["t1"] * nl // 2]
    sd, su = face_pack(ld, Ul, hl, 1 - p_out, dagger)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(np.stack([a.real, a.imag], -1)))
    send_down, send_up = t(sd), t(su)
    recv_lo, recv_hi = torch.empty_like(send_up), torch.empty_like(send_down)
    exchange_faces(send_down, send_up, recv_lo, recv_hi, rank, world)
    bulk = _cplx(oracle.dhop_cb(ld, Ls, oracle.OPEN_T, p_out, Ul, hl, dagger=dagger))
    mine = face_apply(ld, Ul, bulk, _cplx(recv_lo.numpy()), _cplx(recv_hi.numpy()), p_out, dagger, plan["sign_lo"], plan["sign_hi"])
    want = _cplx(oracle.dhop_cb(gdims, Ls, bc, p_out, U, half, dagger=dagger))[plan["t0"] * nl // 2:plan["t1"] * nl // 2]
    err = float(np.abs(mine - want).max() / np.abs(want).max())
    errs = [None] * world
    dist.all_gather_object(errs, err)
    if rank == 0:
        with open(out_path, "w") as f:
            f.write(" ".join(repr(e) for e in errs))
    dist.destroy_process_group()


@pytest.mark.parametrize("world,bc,dagger", [(2, 1, False), (2, 0, True), (3, 1, True)])
def test_decomposed_dhop_over_gloo_matches_the_global_oracle(tmp_path, world, bc, dagger):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = tmp_path / "errs.txt"
    mp.spawn(_worker, args=(world, port, bc, dagger, str(out)), nprocs=world, join=True)
    errs = [float(x) for x in out.read_text().split()]
    assert len(errs) == world and max(errs) <= 1e-13, errs
