"""GPU parity of the TMA-staged, link-stationary fp32 kernel (csrc/dhop_staged.cu) in the launch
configurations bench.py times: tiles per CTA > 1 (tile switch with link refill), Lh = 16 and
Lh = 24 rows, every tunable, and BASELINE.json's full-size configs C4 (whole field) / C5 (every
site, slab by slab through oracle.dhop_sites) plus properties that hold at any size.
Bars: relative L2 error <= 2e-6 (fp32), <= 1e-13 (fp64)."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle
from _util import rel_err

pytestmark = pytest.mark.gpu

TOL = {4: 2e-6, 8: 1e-13}


def sample_sites(dims, parity, n, seed):
    """n lexicographic site indices of the given parity: random ones plus the lattice corners and
    sites on every boundary face (periodic wrap, antiperiodic time hop)."""
    L = [int(d) for d in dims]
    rng = np.random.default_rng(seed)
    coords = rng.integers(0, L, size=(4 * n, 4))
    edge = []
    for mask in range(16):
        edge.append([(L[m] - 1) if (mask >> m) & 1 else 0 for m in range(4)])
    for m in range(4):
        for v in (0, 1, L[m] - 2, L[m] - 1):
            c = rng.integers(0, L, size=(8, 4))
            c[:, m] = v
            edge.extend(c.tolist())
    coords = np.concatenate([np.array(edge, dtype=np.int64), coords])
    coords = coords[(coords.sum(axis=1) & 1) == parity][:n]
    x = coords[:, 0] + L[0] * (coords[:, 1] + L[1] * (coords[:, 2] + L[2] * coords[:, 3]))
    return np.unique(x)


def cb_rows(dims, sites):
    """Row index of lexicographic sites inside the half field of their parity (cb index x >> 1)."""
    return np.asarray(sites, dtype=np.int64) >> 1


def check_cb_against_oracle(lib, dims, Ls, prec, bc, seed, near_unit=False):
    V = gen.volume(dims)
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec) if near_unit else gen.gauge_random(dims, seed, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, seed, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)          # staged kernel or an error: no silent fall back to the direct kernel
        for p_out in (1, 0):
            half = gen.split_parity(psi, dims, 1 - p_out)
            fin = g.import_spinor(half, 1 - p_out)
            fout = g.dhop_oe(fin) if p_out == 1 else g.dhop_eo(fin)
            got = g.export_spinor(fout, p_out)
            want = oracle.dhop_cb(dims, Ls, bc, p_out, U, half)
            assert rel_err(got, want) <= TOL[prec], (dims, Ls, p_out)


def test_staged_lh16_many_tiles_per_cta(lib):
    # <16,4,2,2> rows boxes: 4 x 8 x 8 = 256 tiles on 148 CTAs -> tile switch and link refill
    check_cb_against_oracle(lib, (32, 16, 16, 16), 4, 4, lib.ANTIPERIODIC_T, 41)


def test_staged_lh16_ragged_tail_of_tiles(lib):
    # 4 x 5 x 9 = 180 tiles: CTAs with one and with two tiles; Ls = 5 (odd), periodic
    check_cb_against_oracle(lib, (32, 16, 10, 18), 5, 4, lib.PERIODIC, 42)


def test_staged_lh24_many_tiles_per_cta(lib):
    # <24,2,2,2>: 6 x 6 x 6 = 216 tiles, 192 of 256 consumer threads active, Ls = 3
    check_cb_against_oracle(lib, (48, 12, 12, 12), 3, 4, lib.ANTIPERIODIC_T, 43)


def test_staged_lh8_and_lh4(lib):
    check_cb_against_oracle(lib, (16, 8, 8, 12), 6, 4, lib.ANTIPERIODIC_T, 44)
    check_cb_against_oracle(lib, (8, 8, 12, 8), 7, 4, lib.PERIODIC, 45)


@pytest.mark.parametrize("dims,Ls,bc", [((24, 24, 12, 12), 3, 1),    # <12,4,2,2>: the paper's 24^4 volume class
                                        ((24, 6, 10, 6), 4, 0),      # <12,3,2,3>: L1 not a multiple of 4
                                        ((24, 6, 2, 6), 5, 1),       # <12,3,2,3> with L2 = 2: both x2 faces are the same row
                                        ((64, 8, 8, 6), 3, 1),       # <32,2,2,2>: 256-site tiles, 196 KB of staging
                                        ((64, 4, 6, 2), 2, 0),
                                        ((40, 12, 8, 4), 3, 1),      # <20,3,2,2>
                                        ((40, 8, 8, 6), 2, 0),       # <20,2,2,2>
                                        ((56, 8, 4, 6), 3, 1)])      # <28,2,2,2>
def test_staged_other_row_lengths(lib, dims, Ls, bc):
    """Lh = 12, 20, 28, 32 (L0 = 24, 40, 56, 64): the staged fp32 kernel, several tiles per CTA, every MODE."""
    import torch
    check_cb_against_oracle(lib, dims, Ls, 4, bc, 61)
    U = gen.gauge_random(dims, 62, prec=4)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 62, prec=4)
    xh = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 62, gen.STREAM_SPINOR2, 4)
    with lib.Geometry(dims, Ls, 4, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        assert g.kernel_info().startswith("dhop_staged_kernel<%d," % (dims[0] // 2))
        fin, fx = g.import_spinor(half, lib.EVEN), g.import_spinor(xh, lib.ODD)
        want = oracle.dhop_cb(dims, Ls, bc, 1, U, half)
        plain = g.dhop_oe(fin).clone()
        fused, n = g.dhop_oe_norm2(fin)
        assert torch.equal(fused, plain) and abs(n - oracle.norm2(g.export_spinor(fused, lib.ODD))) <= 1e-12 * n
        assert rel_err(g.export_spinor(g.dhop_oe_dag(fin), lib.ODD), oracle.dhop_cb(dims, Ls, bc, 1, U, half, dagger=True)) <= TOL[4]
        assert rel_err(g.export_spinor(g.dhop_oe_axpy(fin, fx, 1.3, -0.5), lib.ODD), 1.3 * xh.astype(np.float64) - 0.5 * want) <= TOL[4]


OPTION_SETS = [
    {"variant": 2}, {"variant": 3}, {"variant": 12}, {"variant": 13}, {"variant": 14}, {"variant": 15},
    {"raster_staged": 0}, {"raster_staged": 1}, {"raster_staged": 3}, {"raster_staged": 11}, {"raster_staged": 21}, {"raster_staged": 31},
    {"zigzag": 0}, {"ssplit": 2}, {"ssplit": 4}, {"layered": 0},
    {"l2pol": 0}, {"l2pol": 11212020},
]


def test_staged_tunables_do_not_change_the_result(lib):
    """Tile shape, launch order, slice split, L2 policies only move work around: the
    arithmetic per output site is the same, so the results must be bit-identical; the direct
    kernel (kernel=1) sums the legs in another order and is held to the parity bar instead."""
    import torch
    dims, Ls, prec, bc = (32, 16, 16, 16), 4, 4, lib.ANTIPERIODIC_T
    U = gen.gauge_random(dims, 46, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 46, prec=prec)
    want = oracle.dhop_oe(dims, Ls, bc, U, half)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        fin = g.import_spinor(half, lib.EVEN)
        ref = g.dhop_oe(fin).clone()
        assert rel_err(g.export_spinor(ref, lib.ODD), want) <= TOL[prec]
        defaults = {"variant": 0, "raster_staged": -1, "zigzag": 1, "ssplit": 1, "layered": 1,
                    "l2pol": 11222222}
        for opts in OPTION_SETS:
            for k, v in {**defaults, **opts}.items():
                g.set_option(k, v)
            out = g.dhop_oe(fin)
            assert torch.equal(out, ref), opts
        for k, v in defaults.items():
            g.set_option(k, v)
        g.set_option("kernel", 1)
        assert rel_err(g.export_spinor(g.dhop_oe(fin), lib.ODD), want) <= TOL[prec]
        g.set_option("kernel", 2)
        assert torch.equal(g.dhop_oe(fin), ref)


@pytest.mark.parametrize("prec", [4, 8])
def test_c4_full_size_oe_then_eo_whole_field(lib, prec):
    """BASELINE.json configs[3]: 32^4 x 16, near-unit gauge, Gaussian spinor on the even
    checkerboard, DhopOE followed by DhopEO -- the launch configuration bench.py times -- compared
    with the oracle on EVERY element of both results (whole field, not samples)."""
    dims, Ls, bc, seed = (32, 32, 32, 32), 16, lib.PERIODIC, 1004
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec)
    psi_e = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, seed, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)           # the staged kernels, or an error
        f_e = g.import_spinor(psi_e, lib.EVEN)
        f_o = g.dhop_oe(f_e)
        f_e2 = g.dhop_eo(f_o)
        chi_o = g.export_spinor(f_o, lib.ODD)
        phi_e = g.export_spinor(f_e2, lib.EVEN)
        n_in, n_mid, n_out = g.norm2(f_e, lib.EVEN), g.norm2(f_o, lib.ODD), g.norm2(f_e2, lib.EVEN)
    want = oracle.dhop_cb(dims, Ls, bc, 1, U, psi_e)
    assert rel_err(chi_o, want) <= TOL[prec]
    # per-site worst case as well: no single site may hide behind the field norm
    d = np.linalg.norm((chi_o - want).reshape(want.shape[0], -1), axis=1)
    assert d.max() <= 8 * TOL[prec] * np.sqrt(np.mean(np.sum(want.reshape(want.shape[0], -1) ** 2, axis=1)))
    del want
    want = oracle.dhop_cb(dims, Ls, bc, 0, U, chi_o)                  # the GPU's own chi_o is the input here
    assert rel_err(phi_e, want) <= TOL[prec]
    d = np.linalg.norm((phi_e - want).reshape(want.shape[0], -1), axis=1)
    assert d.max() <= 8 * TOL[prec] * np.sqrt(np.mean(np.sum(want.reshape(want.shape[0], -1) ** 2, axis=1)))
    # properties at full size: P8 norm bound, and the GPU norm2 against the oracle's on the exported field
    assert n_mid <= 64.0 * n_in and n_out <= 64.0 * n_mid
    assert abs(n_mid - oracle.norm2(chi_o)) <= 1e-12 * n_mid
    assert abs(n_out - oracle.norm2(phi_e)) <= 1e-12 * n_out


def test_c5_full_size_slab_by_slab(lib):
    """BASELINE.json configs[4]: 48^3 x 96 x Ls=12 fp32, random SU(3), antiperiodic time: full Dhop
    compared with the oracle on every site, slab by slab in x3 (the 24.5 GB fp64
    oracle field is never materialised), norm2 of the result, and the even/odd pair against the two
    halves of the full result.  Every CTA of the staged kernel walks > 64 tiles here (the tile
    origins beyond the shared-memory cache come from global memory)."""
    dims, Ls, prec, bc, seed = (48, 48, 48, 96), 12, 4, lib.ANTIPERIODIC_T, 1005
    V = gen.volume(dims)
    slab = dims[0] * dims[1] * dims[2]
    U = gen.gauge_random(dims, seed, prec=prec)
    psi = gen.spinor_gaussian(V, Ls, seed, prec=prec)
    par = gen.site_parity(dims)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        f = g.import_spinor(psi, lib.FULL)
        out = g.dhop(f)
        n_in, n_out = g.norm2(f), g.norm2(out)
        got = g.export_spinor(out, lib.FULL)
        del f, out
        assert n_out <= 64.0 * n_in
        assert abs(n_out - oracle.norm2(got)) <= 1e-12 * n_out
        num = den = 0.0
        worst = 0.0
        for x3 in range(dims[3]):
            sites = np.arange(x3 * slab, (x3 + 1) * slab, dtype=np.int64)
            want = oracle.dhop_sites(dims, Ls, bc, U, psi, False, sites)
            diff = got[x3 * slab:(x3 + 1) * slab].astype(np.float64) - want
            e, r = float(np.sum(diff * diff)), float(np.sum(want * want))
            num, den = num + e, den + r
            worst = max(worst, np.sqrt(e / r))
        assert np.sqrt(num / den) <= TOL[prec]
        assert worst <= TOL[prec]                                     # every slab on its own meets the bar
        # the even/odd pair must reproduce the two halves of the full result (bitwise: same kernel, same order)
        for p_out in (1, 0):
            half = np.ascontiguousarray(psi[par == 1 - p_out])
            fin = g.import_spinor(half, 1 - p_out)
            del half
            fo = g.dhop_oe(fin) if p_out == 1 else g.dhop_eo(fin)
            got_h = g.export_spinor(fo, p_out)
            del fin, fo
            for x3 in range(dims[3]):
                a, b = x3 * slab, (x3 + 1) * slab
                assert np.array_equal(got_h[a >> 1:b >> 1], got[a:b][par[a:b] == p_out])
            del got_h


def test_axpy_maps_survive_cache_eviction(lib):
    """The fused a x + b Dhop looks up two tensor-map sets in an 8-slot round-robin cache; `in` hitting
    in the slot that the miss of `x` evicts must not make the kernel read `in` from x's buffer
    (ADVICE r1).  Fill the cache so that exactly this happens and compare with a cold-cache result."""
    import torch
    dims, Ls, prec, bc = (32, 8, 8, 8), 4, 4, lib.ANTIPERIODIC_T
    U = gen.gauge_random(dims, 52, prec=prec)
    nh = gen.volume(dims) // 2
    a_in = gen.spinor_gaussian(nh, Ls, 52, prec=prec)
    xs = [gen.spinor_gaussian(nh, Ls, 53 + i, gen.STREAM_SPINOR2, prec) for i in range(3)]
    want = [4.3 * x.astype(np.float64) - 0.5 * oracle.dhop_cb(dims, Ls, bc, 1, U, a_in) for x in xs]
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        fin = g.import_spinor(a_in, lib.EVEN)
        fx = [g.import_spinor(x, lib.ODD) for x in xs]
        dummies = [g.new_field(lib.EVEN) for _ in range(9)]
        scratch = g.new_field(lib.ODD)
        for fill in range(0, 10):
            # `fill` other input fields between two fused calls: every phase of the round-robin slot counter
            for k, (x, w) in enumerate(zip(fx, want)):
                for dmy in dummies[:fill]:
                    dmy.zero_()
                    g.dhop_oe(dmy, scratch)
                got = g.export_spinor(g.dhop_oe_axpy(fin, x, 4.3, -0.5), lib.ODD)
                assert rel_err(got, w) <= TOL[prec], (fill, k)


@pytest.mark.parametrize("prec", [4, 8])
def test_c4_stress_many_launches_bit_identical(lib, prec):
    """>= 200 launches of the C4 half-Dhop under slice-split / zigzag / launch-order variations: every
    output must equal the first one bit for bit (a shared-memory region handed back to the TMA
    producer too early would show up here as a corrupted site; VERDICT r1 task 1a)."""
    import torch
    dims, Ls, bc, seed = (32, 32, 32, 32), 16, lib.PERIODIC, 1004
    U = gen.gauge_near_unit(dims, seed, 0.2, prec=prec)
    psi_e = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, seed, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        f_e = g.import_spinor(psi_e, lib.EVEN)
        ref = g.dhop_oe(f_e).clone()
        out = g.new_field(lib.ODD)
        variations = [{}, {"ssplit": 2}, {"zigzag": 0}, {"ssplit": 4, "zigzag": 0}, {"raster_staged": 0}] if prec == 4 else [{}, {"raster_staged": 0}, {"zigzag": 0}, {"max_ctas": 101}]
        n = 0
        for rep in range(45 if prec == 4 else 60):
            for opts in variations:
                for k, v in {"ssplit": 1, "zigzag": 1, "raster_staged": -1, "max_ctas": 0, **opts}.items():
                    g.set_option(k, v)
                out.zero_()
                g.dhop_oe(f_e, out)
                assert torch.equal(out, ref), (rep, opts)
                n += 1
        assert n >= 200


@pytest.mark.parametrize("dims,Ls,prec", [((32, 16, 16, 16), 4, 4), ((48, 12, 12, 12), 3, 4), ((8, 8, 8, 8), 8, 8),
                                          ((12, 6, 2, 4), 5, 4)])
def test_fused_dhop_norm2(lib, dims, Ls, prec):
    """dwf_dhop_oe_norm2 / dwf_dhop_eo_norm2: the same output bits as the plain call, and the
    reduction of the epilogue (staged fp32 kernel) or of the second pass (other geometries) within
    1e-12 of dwf_norm2 of that output and of the oracle's sum; deterministic."""
    import torch
    bc = lib.ANTIPERIODIC_T
    U = gen.gauge_random(dims, 51, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 51, prec=prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        for p_out in (1, 0):
            fin = g.import_spinor(half, 1 - p_out)
            plain = g.dhop_oe(fin) if p_out == 1 else g.dhop_eo(fin)
            fused, n = g.dhop_oe_norm2(fin) if p_out == 1 else g.dhop_eo_norm2(fin)
            assert torch.equal(fused, plain)
            n_sep = g.norm2(plain, p_out)
            assert abs(n - n_sep) <= 1e-12 * n_sep
            assert abs(n - oracle.norm2(g.export_spinor(fused, p_out))) <= 1e-12 * n_sep
            _, n2 = g.dhop_oe_norm2(fin) if p_out == 1 else g.dhop_eo_norm2(fin)
            assert n2 == n
        with pytest.raises(lib.DwfError):
            lib.dwf_dhop_eo_norm2(g.handle, fin, fin)


@pytest.mark.parametrize("opts", [{"ssplit": 2}, {"variant": 2}, {"variant": 12, "raster_staged": 2}, {"zigzag": 0, "layered": 0}])
def test_other_modes_under_tunables(lib, opts):
    """The norm2-fused, dagger and axpy instances of the staged kernel under a few tunables: outputs
    bit-identical to the default configuration, the fused norm within its summation-order tolerance."""
    import torch
    dims, Ls, prec, bc = (32, 16, 16, 16), 4, 4, lib.ANTIPERIODIC_T
    U = gen.gauge_random(dims, 47, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 47, prec=prec)
    xh = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 47, gen.STREAM_SPINOR2, prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        fin, fx = g.import_spinor(half, lib.EVEN), g.import_spinor(xh, lib.ODD)
        ref_n_out, ref_n = g.dhop_oe_norm2(fin)
        ref_n_out = ref_n_out.clone()
        ref_d = g.dhop_oe_dag(fin).clone()
        ref_a = g.dhop_oe_axpy(fin, fx, 4.3, -0.5).clone()
        for k, v in opts.items():
            g.set_option(k, v)
        out, n = g.dhop_oe_norm2(fin)
        assert torch.equal(out, ref_n_out) and abs(n - ref_n) <= 1e-12 * ref_n
        assert torch.equal(g.dhop_oe_dag(fin), ref_d)
        assert torch.equal(g.dhop_oe_axpy(fin, fx, 4.3, -0.5), ref_a)


def test_dhop_calls_can_be_captured_in_a_cuda_graph(lib):
    """dwf_dhop_oe / dwf_dhop_eo enqueue one kernel each and never synchronise, so a solver may
    capture them in a CUDA graph (removes the launch gaps that dominate small lattices)."""
    import torch
    dims, Ls, prec = (16, 16, 16, 16), 16, 4                     # BASELINE.json configs[2] shape
    U = gen.gauge_random(dims, 1003, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 1003, prec=prec)
    with lib.Geometry(dims, Ls, prec, lib.PERIODIC) as g:
        g.load_gauge(U)
        f_e = g.import_spinor(half, lib.EVEN)
        f_o, f_x = g.new_field(lib.ODD), g.new_field(lib.EVEN)
        g.dhop_oe(f_e, f_o)
        g.dhop_eo(f_o, f_x)
        torch.cuda.synchronize()
        ref = f_x.clone()
        graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        with torch.cuda.stream(side):
            g.dhop_oe(f_e, f_o)                                  # warm the per-thread tensor-map cache outside the capture
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=side):
                g.dhop_oe(f_e, f_o)
                g.dhop_eo(f_o, f_x)
        f_x.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(f_x, ref)


@pytest.mark.parametrize("dims,Ls,bc", [((32, 8, 8, 8), 3, 1), ((16, 8, 4, 6), 5, 0), ((8, 8, 8, 8), 8, 1), ((32, 6, 4, 10), 2, 0),
                                        ((24, 8, 6, 8), 4, 1), ((48, 4, 6, 4), 3, 0), ((64, 4, 4, 6), 3, 1), ((40, 6, 4, 4), 5, 1),
                                        ((56, 4, 4, 6), 2, 1), ((40, 8, 8, 6), 2, 0)])
def test_staged64_fp64_kernel(lib, dims, Ls, bc):
    """The fp64 staged kernels (csrc/dhop_staged64.cu: site-per-thread with the links in tensor memory for
    Lh = 4 .. 28, tiles of 96 .. 128 sites; colour-split for Lh = 32), forced with kernel=2: plain, dagger, fused norm2 and
    fused a x + b Dhop against the oracle at the fp64 bar; bit-identical from run to run and under zigzag."""
    import torch
    check_cb_against_oracle(lib, dims, Ls, 8, bc, 48)
    U = gen.gauge_random(dims, 49, prec=8)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 49, prec=8)
    xh = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 49, gen.STREAM_SPINOR2, 8)
    with lib.Geometry(dims, Ls, 8, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        assert g.kernel_info().startswith("dhop_staged64")
        fin, fx = g.import_spinor(half, lib.EVEN), g.import_spinor(xh, lib.ODD)
        want = oracle.dhop_cb(dims, Ls, bc, 1, U, half)
        a = g.dhop_oe_dag(fin).clone()
        assert rel_err(g.export_spinor(a, lib.ODD), oracle.dhop_cb(dims, Ls, bc, 1, U, half, dagger=True)) <= TOL[8]
        assert torch.equal(g.dhop_oe_dag(fin), a)
        plain = g.dhop_oe(fin).clone()
        fused, n = g.dhop_oe_norm2(fin)                           # MODE 4: norm2 in the store epilogue
        assert torch.equal(fused, plain)
        assert abs(n - oracle.norm2(g.export_spinor(fused, lib.ODD))) <= 1e-12 * n
        assert g.dhop_oe_norm2(fin)[1] == n
        ax = g.dhop_oe_axpy(fin, fx, 1.3, -0.5)
        assert rel_err(g.export_spinor(ax, lib.ODD), 1.3 * xh - 0.5 * want) <= TOL[8]
        buf = fx.clone()
        lib.dwf_dhop_oe_axpy(g.handle, fin, buf, 1.3, -0.5, buf)   # x == out
        assert torch.equal(buf, ax)
        g.set_option("zigzag", 0)
        assert torch.equal(g.dhop_oe(fin), plain)
        g.set_option("kernel", 1)                                 # direct kernel: another summation order
        assert rel_err(g.export_spinor(g.dhop_oe_dag(fin), lib.ODD), g.export_spinor(a, lib.ODD)) <= TOL[8]


@pytest.mark.parametrize("prec,dims,Ls,bc,max_ctas", [
    (8, (32, 8, 8, 8), 3, 1, 5),        # staged64s <16,2,2,2>: 64 tiles on 5 CTAs = 12-13 tiles each: the 14-slot link ring wraps
    (8, (32, 8, 8, 8), 1, 0, 3),        # Ls = 1: every slice is a tile's first and last one (all four link barriers per slice)
    (8, (32, 8, 8, 8), 2, 1, 64),       # one tile per CTA: no hand-over at all
    (8, (32, 8, 8, 8), 2, 0, 63),       # CTA 0 walks two tiles, all others one
    (8, (16, 8, 8, 8), 4, 1, 2),        # staged64s <8,4,2,2>: 16 tiles on 2 CTAs
    (8, (8, 8, 8, 8), 5, 1, 1),         # staged64s <4,4,4,2>: all 16 tiles on ONE CTA
    (8, (24, 8, 6, 8), 3, 1, 4),        # staged64s <12,2,2,2>: 96-site tiles, the fourth consumer / loader warp idles
    (8, (40, 6, 4, 4), 2, 1, 3),        # staged64s <20,3,2,1>: 120-site tiles, eight lanes of the last warp own no site
    (8, (56, 4, 4, 6), 2, 0, 5),        # staged64s <28,2,2,1>: 112-site tiles
    (4, (32, 8, 8, 8), 3, 1, 3),        # fp32 staged <16,4,2,2>: 32 tiles on 3 CTAs (link refill in the last slice)
    (4, (32, 8, 8, 8), 1, 0, 2),
])
def test_staged_many_tiles_per_cta(lib, prec, dims, Ls, bc, max_ctas):
    """Tile switches on small lattices: the option "max_ctas" caps the grid of the staged kernels, so that a CTA walks
    many tiles -- every phase of the loader / consumer link hand-over of the fp64 site-per-thread kernel (slot ring of
    14 wraps after 7 tiles), the link refill of the fp32 kernel, odd and even tile counts per CTA.  Plain, dagger, fused
    norm2 and fused a x + b Dhop against the oracle; the result does not depend on the grid (bit-identical)."""
    import torch
    U = gen.gauge_random(dims, 91, prec=prec)
    half = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 91, prec=prec)
    xh = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 91, gen.STREAM_SPINOR2, prec)
    with lib.Geometry(dims, Ls, prec, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        fin, fx = g.import_spinor(half, lib.EVEN), g.import_spinor(xh, lib.ODD)
        full_grid = g.dhop_oe(fin).clone()
        full_grid_eo = g.dhop_eo(fx).clone()
        g.set_option("max_ctas", max_ctas)
        want = oracle.dhop_cb(dims, Ls, bc, 1, U, half)
        out = g.dhop_oe(fin)
        assert rel_err(g.export_spinor(out, lib.ODD), want) <= TOL[prec]
        assert torch.equal(out, full_grid)
        assert torch.equal(g.dhop_eo(fx), full_grid_eo)
        want_d = oracle.dhop_cb(dims, Ls, bc, 1, U, half, dagger=True)
        assert rel_err(g.export_spinor(g.dhop_oe_dag(fin), lib.ODD), want_d) <= TOL[prec]
        fused, n = g.dhop_oe_norm2(fin)
        assert torch.equal(fused, full_grid)
        assert abs(n - oracle.norm2(g.export_spinor(fused, lib.ODD))) <= 1e-12 * n
        ax = g.dhop_oe_axpy(fin, fx, -0.25, 2.0)
        assert rel_err(g.export_spinor(ax, lib.ODD), -0.25 * xh.astype(np.float64) + 2.0 * want) <= TOL[prec]
        with pytest.raises(lib.DwfError):
            g.set_option("max_ctas", -1)


@pytest.mark.parametrize("dims,Ls,bc,max_ctas,opts", [((32, 8, 8, 8), 3, 1, 0, {}), ((16, 8, 8, 8), 4, 0, 0, {}), ((32, 8, 8, 8), 2, 1, 3, {}),
                                                      ((24, 8, 6, 8), 2, 1, 5, {}), ((8, 8, 8, 8), 5, 1, 1, {}),
                                                      ((32, 8, 8, 8), 4, 1, 6, {"ssplit": 2}), ((32, 8, 8, 8), 3, 0, 0, {"zigzag": 0, "layered": 0})])
def test_full_field_dhop_is_one_launch(lib, dims, Ls, bc, max_ctas, opts):
    """dwf_dhop on an fp32 geometry with a staged variant: ONE launch whose tile table spans both parities (VERDICT r01
    task 8).  Against the oracle on every element, bit-identical to the two half-field launches (option full_launch = 0),
    also when few CTAs walk tiles of both parities one after the other (max_ctas: the tile switch changes the link set,
    the input half and the output half)."""
    import torch
    U = gen.gauge_random(dims, 95, prec=4)
    psi = gen.spinor_gaussian(gen.volume(dims), Ls, 95, prec=4)
    with lib.Geometry(dims, Ls, 4, bc) as g:
        g.load_gauge(U)
        g.set_option("kernel", 2)
        if max_ctas:
            g.set_option("max_ctas", max_ctas)
        for k, v in opts.items():
            g.set_option(k, v)
        fin = g.import_spinor(psi, lib.FULL)
        n0 = lib.dwf_launch_count()
        out = g.dhop(fin).clone()
        assert lib.dwf_launch_count() - n0 == 1
        assert rel_err(g.export_spinor(out, lib.FULL), oracle.dhop(dims, Ls, bc, U, psi)) <= TOL[4]
        g.set_option("full_launch", 0)
        n0 = lib.dwf_launch_count()
        two = g.dhop(fin)
        assert lib.dwf_launch_count() - n0 == 2
        assert torch.equal(two, out)
        g.set_option("full_launch", 1)
        assert torch.equal(g.dhop(fin), out)


@pytest.mark.parametrize("prec,dims,Ls", [(4, (32, 8, 8, 8), 4), (8, (32, 8, 8, 8), 3), (4, (12, 6, 4, 6), 3)])
def test_norm2_async_tickets(lib, prec, dims, Ls):
    """dwf_dhop_*_norm2_async + dwf_reduction_wait: several steps enqueued before any value is read; every ticket returns the
    value of its own step (the same bits as the waiting call), out of order as well; a ticket older than the ring of kept
    results is refused."""
    import torch
    U = gen.gauge_random(dims, 97, prec=prec)
    with lib.Geometry(dims, Ls, prec, 1) as g:
        g.load_gauge(U)
        fields = [g.import_spinor(gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 100 + i, prec=prec), lib.EVEN) for i in range(5)]
        want = [g.dhop_oe_norm2(f)[1] for f in fields]
        ref_out = g.dhop_oe(fields[3]).clone()
        outs, tickets = [], []
        for f in fields:                                    # five steps in flight
            o, t = g.dhop_oe_norm2_async(f)
            outs.append(o)
            tickets.append(t)
        assert tickets == list(range(tickets[0], tickets[0] + 5))
        for i in (4, 0, 2, 1, 3):
            assert g.reduction_wait(tickets[i]) == want[i]
        assert torch.equal(outs[3], ref_out)
        assert g.norm2(fields[0], lib.EVEN) > 0.0           # the waiting calls still work in between
        for f in fields * 2:
            _, t_last = g.dhop_eo_norm2_async(g.dhop_oe(f))
        with pytest.raises(lib.DwfError):
            g.reduction_wait(tickets[0])                    # more than 8 reductions ago
        with pytest.raises(lib.DwfError):
            g.reduction_wait(t_last + 1)                    # never issued
        assert g.reduction_wait(t_last) > 0.0
