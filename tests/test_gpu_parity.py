"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
identical seeded inputs.  Bars (BASELINE.json north_star): relative L2 error <= 1e-13 in fp64
and <= 2e-6 in fp32.  Configs C1-C5 are BASELINE.json's; the extra shapes cover ragged tiles
(extents that are not powers of two), L=2 wraps, odd Ls and Ls=1."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}


def make_inputs(dims, Ls, prec, seed, near_unit=False):
    V = gen.volume(dims)
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec) if near_unit else gen.gauge_random(dims, seed, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, seed, prec=prec)
    return U, psi


def gpu_full(lib, dims, Ls, prec, bc, U, psi):
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fin = g.import_spinor(psi, lib.FULL)
        fout = g.dhop(fin)
        return g.export_spinor(fout, lib.FULL)


def gpu_cb(lib, dims, Ls, prec, bc, U, psi_half, parity_out):
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fin = g.import_spinor(psi_half, 1 - parity_out)
        fout = g.dhop_oe(fin) if parity_out == lib.ODD else g.dhop_eo(fin)
        return g.export_spinor(fout, parity_out)


def test_c1_full_fp64(lib):
    dims, Ls, prec = (4, 4, 4, 4), 4, 8
    U, psi = make_inputs(dims, Ls, prec, 1001)
    got = gpu_full(lib, dims, Ls, prec, lib.PERIODIC, U, psi)
    want = oracle.dhop(dims, Ls, oracle.PERIODIC, U, psi)
    assert rel_err(got, want) <= TOL[prec]


def test_c2_full_and_eo_fp64_antiperiodic(lib):
    dims, Ls, prec, bc = (8, 8, 8, 8), 8, 8, lib.ANTIPERIODIC_T
    U, psi = make_inputs(dims, Ls, prec, 1002)
    want = oracle.dhop(dims, Ls, oracle.ANTIPERIODIC_T, U, psi)
    full = gpu_full(lib, dims, Ls, prec, bc, U, psi)
    assert rel_err(full, want) <= TOL[prec]
    par = gen.site_parity(dims)
    pe, po = gen.split_parity(psi, dims, 0), gen.split_parity(psi, dims, 1)
    out_o = gpu_cb(lib, dims, Ls, prec, bc, U, pe, lib.ODD)      # DhopOE: even in -> odd out
    out_e = gpu_cb(lib, dims, Ls, prec, bc, U, po, lib.EVEN)     # DhopEO: odd in -> even out
    assert rel_err(out_o, oracle.dhop_oe(dims, Ls, bc, U, pe)) <= TOL[prec]
    assert rel_err(out_e, oracle.dhop_eo(dims, Ls, bc, U, po)) <= TOL[prec]
    # the even/odd pair reassembles to the full operator
    re = np.empty_like(full)
    re[par == 0], re[par == 1] = out_e, out_o
    assert rel_err(re, want) <= TOL[prec]
    assert rel_err(re, full) <= TOL[prec]


def test_c3_full_fp32(lib):
    dims, Ls, prec = (16, 16, 16, 16), 16, 4
    U, psi = make_inputs(dims, Ls, prec, 1003)
    got = gpu_full(lib, dims, Ls, prec, lib.PERIODIC, U, psi)
    want = oracle.dhop(dims, Ls, oracle.PERIODIC, U, psi)
    assert rel_err(got, want) <= TOL[prec]


RAGGED = [
    # dims, Ls: tiles that do not fill a CTA, non power-of-two extents, L=2 wraps, odd Ls
    ((2, 2, 2, 2), 1), ((2, 2, 2, 2), 4), ((6, 4, 10, 2), 3), ((12, 6, 2, 4), 12), ((4, 2, 6, 14), 5),
    ((10, 10, 6, 4), 2), ((24, 4, 4, 4), 16), ((4, 4, 4, 24), 8), ((8, 12, 4, 6), 6),
]


@pytest.mark.parametrize("prec", [4, 8])
@pytest.mark.parametrize("bc", [0, 1])
@pytest.mark.parametrize("dims,Ls", RAGGED)
def test_ragged_shapes_full_and_cb(lib, dims, Ls, bc, prec):
    U, psi = make_inputs(dims, Ls, prec, 77)
    want = oracle.dhop(dims, Ls, bc, U, psi)
    assert rel_err(gpu_full(lib, dims, Ls, prec, bc, U, psi), want) <= TOL[prec]
    for p_out in (0, 1):
        half = gen.split_parity(psi, dims, 1 - p_out)
        got = gpu_cb(lib, dims, Ls, prec, bc, U, half, p_out)
        assert rel_err(got, oracle.dhop_cb(dims, Ls, bc, p_out, U, half)) <= TOL[prec]
        assert rel_err(got, gen.split_parity(want, dims, p_out)) <= TOL[prec]


@pytest.mark.parametrize("prec", [4, 8])
def test_import_export_roundtrip_is_exact(lib, prec):
    dims, Ls = (6, 4, 4, 8), 6
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 5, prec=prec)
    with lib.Geometry(dims, Ls, prec) as g:
        assert np.array_equal(g.export_spinor(g.import_spinor(psi, lib.FULL), lib.FULL), psi)
        half = gen.split_parity(psi, dims, 1)
        assert np.array_equal(g.export_spinor(g.import_spinor(half, lib.ODD), lib.ODD), half)
        # device-resident canonical source / destination
        import torch
        t = torch.from_numpy(psi).cuda()
        f = g.import_spinor(t, lib.FULL)
        back = torch.empty_like(t)
        lib.dwf_export_spinor(g.handle, f, lib.FULL, back)
        assert torch.equal(back, t)


@pytest.mark.parametrize("prec", [4, 8])
def test_chunked_host_transfers_roundtrip_and_async(lib, prec):
    """Host arrays larger than one ring buffer (32 MB): several chunks per call with a ragged last chunk,
    full and half fields, pinned and pageable memory; with "async_host" the calls return early and
    dwf_host_wait completes them (an export followed at once by an import of another array)."""
    import torch
    dims, Ls = (32, 6, 10, 14), 9                # full field: 26880 sites * 9 * 24 reals = 23 / 46 MB ... x2 parities
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 6, prec=prec)
    psi = np.concatenate([psi, psi[::-1]], axis=1)[:, :Ls * 2]     # Ls = 18: 93 MB (fp32) / 186 MB (fp64)
    Ls2 = psi.shape[1]
    psi = np.ascontiguousarray(psi)
    with lib.Geometry(dims, Ls2, prec) as g:
        f = g.import_spinor(psi, lib.FULL)
        assert np.array_equal(g.export_spinor(f, lib.FULL), psi)
        # the device-source path produces the same device field as the chunked host path
        assert torch.equal(g.import_spinor(torch.from_numpy(psi).cuda(), lib.FULL), f)
        half = gen.split_parity(psi, dims, 0)
        fh = g.import_spinor(half, lib.EVEN)
        assert np.array_equal(g.export_spinor(fh, lib.EVEN), half)
        # pinned host memory, asynchronous mode
        pin_in = torch.from_numpy(half).pin_memory()
        pin_out = torch.empty_like(pin_in).pin_memory()
        other = torch.from_numpy(np.ascontiguousarray(half[::-1])).pin_memory()
        g.set_option("async_host", 1)
        f1 = g.import_spinor(pin_in.numpy(), lib.EVEN)
        g.export_spinor(f1, lib.EVEN, out=pin_out.numpy())
        f2 = g.import_spinor(other.numpy(), lib.EVEN)            # H2D of this one overlaps the D2H of the export
        g.host_wait()
        torch.cuda.synchronize()
        g.set_option("async_host", 0)
        assert torch.equal(pin_out, pin_in)
        assert np.array_equal(g.export_spinor(f2, lib.EVEN), other.numpy())


@pytest.mark.parametrize("prec", [4, 8])
def test_norm2_and_inner_product(lib, prec):
    dims, Ls = (8, 4, 6, 4), 5
    V = gen.volume(dims)
    a = gen.spinor_gaussian(V, Ls, 9, gen.STREAM_SPINOR, prec)
    b = gen.spinor_gaussian(V, Ls, 9, gen.STREAM_SPINOR2, prec)
    with lib.Geometry(dims, Ls, prec) as g:
        fa, fb = g.import_spinor(a), g.import_spinor(b)
        n = g.norm2(fa)
        assert abs(n - oracle.norm2(a)) <= 1e-12 * oracle.norm2(a)
        assert g.norm2(fa) == n                                   # deterministic
        ip = g.inner_product(fa, fb)
        want = oracle.inner(a, b)
        assert abs(ip - want) <= 1e-12 * np.sqrt(oracle.norm2(a) * oracle.norm2(b))
        ha = gen.split_parity(a, dims, 0)
        assert abs(g.norm2(g.import_spinor(ha, lib.EVEN), lib.EVEN) - oracle.norm2(ha)) <= 1e-12 * oracle.norm2(ha)
        # closed form: constant field c -> N |c|^2
        c = np.full_like(a, 0.5)
        assert g.norm2(g.import_spinor(c)) == pytest.approx(0.25 * c.size, rel=1e-14)


def test_runtime_errors(lib):
    import torch
    dims, Ls = (4, 4, 4, 4), 4
    with lib.Geometry(dims, Ls, 8) as g:
        f, o = g.new_field(), g.new_field()
        with pytest.raises(lib.DwfError) as e:
            g.dhop(f, o)
        assert e.value.code == lib.ERR_NO_GAUGE
        g.load_gauge(gen.gauge_unit(dims))
        with pytest.raises(lib.DwfError) as e:
            g.dhop(f, f)
        assert e.value.code == lib.ERR_INVALID_ARG
        with pytest.raises(lib.DwfError) as e:
            lib.dwf_dhop(g.handle, f[1:], o)                     # 8-byte aligned only
        assert e.value.code == lib.ERR_INVALID_ARG
        with pytest.raises(lib.DwfError) as e:
            g.norm2(f, 7)
        assert e.value.code == lib.ERR_INVALID_ARG
    assert torch.cuda.is_available()


def test_free_field_constant_gives_8psi(lib):
    """P2 at p=0 run on the GPU output directly: unit gauge, constant-in-x field -> 8 psi."""
    dims, Ls, prec = (8, 6, 4, 10), 4, 8
    V = gen.volume(dims)
    chi = gen.spinor_gaussian(1, Ls, 3, prec=prec)
    psi = np.ascontiguousarray(np.broadcast_to(chi, (V, Ls, 4, 3, 2)))
    got = gpu_full(lib, dims, Ls, prec, lib.PERIODIC, gen.gauge_unit(dims, prec), psi)
    assert rel_err(got, 8.0 * psi) <= 1e-14


def test_launch_counter_moves(lib):
    dims, Ls = (4, 4, 4, 4), 2
    n0 = lib.dwf_launch_count()
    U, psi = make_inputs(dims, Ls, 4, 1)
    gpu_full(lib, dims, Ls, 4, 0, U, psi)
    assert lib.dwf_launch_count() >= n0 + 4          # pack gauge, import, dhop, export
