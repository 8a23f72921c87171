"""dwf_norm2_static: the norm2 that allocates nothing (scratch in a file-scope __device__ array of libdwf.so,
csrc/norm2_static.cu) against the existing path dwf_norm2 (scratch allocated by the geometry), at the bar the other
reduction tests use (relative 1e-12: the two differ only in summation order), and against the oracle.

This file is collected last on purpose (pytest -x: a failure here hides nothing behind it); it
passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import dwf_inputs as gen
import oracle

pytestmark = pytest.mark.gpu

RTOL = 1e-12


@pytest.mark.parametrize("prec", [4, 8])
def test_norm2_static_matches_existing_path_twice_in_a_row(lib, prec):
    import torch
    dims, Ls = (16, 8, 8, 8), 6                 # half field: 4096 * 6 * 24 reals = 590k reals: 72 / 144 CTAs of the static kernel
    psi_a = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 301, prec=prec)
    psi_b = gen.spinor_gaussian(gen.volume(dims) // 2, Ls, 302, prec=prec)
    result = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    with lib.Geometry(dims, Ls, prec, lib.PERIODIC) as g:
        fa, fb = g.import_spinor(psi_a, lib.EVEN), g.import_spinor(psi_b, lib.ODD)
        want_a, want_b = g.norm2(fa, lib.EVEN), g.norm2(fb, lib.ODD)        # the existing path
        assert abs(want_a - oracle.norm2(psi_a)) <= RTOL * want_a
        # two calls in a row, the second on another buffer: the shared scratch keeps the first call's partials
        lib.dwf_norm2_static(fa, result)
        got_a = float(result.item())
        lib.dwf_norm2_static(fb, result)
        got_b = float(result.item())
        assert abs(got_a - want_a) <= RTOL * want_a
        assert abs(got_b - want_b) <= RTOL * want_b
        assert got_a != got_b
        # back to back without a host read in between, then a shorter buffer (fewer CTAs than the call before,
        # a ragged last chunk and reals behind the last whole 128-bit vector): stale partials are not read
        lib.dwf_norm2_static(fb, result)
        lib.dwf_norm2_static(fa, result)
        assert float(result.item()) == got_a                                # deterministic: the same bits
        n_short = 2048 * (16 // prec) * 3 + 7 * (16 // prec) + 1
        flat = fa.reshape(-1)
        lib.dwf_norm2_static(flat, result, n_reals=n_short)
        want_short = float((flat[:n_short].double() ** 2).sum().item())
        assert abs(float(result.item()) - want_short) <= RTOL * want_short
        lib.dwf_norm2_static(flat, result, n_reals=0)
        assert float(result.item()) == 0.0
        # the existing path is untouched by the new one
        assert g.norm2(fa, lib.EVEN) == want_a


def test_norm2_static_rejects_oversize_and_bad_arguments(lib):
    import torch
    x = torch.ones(1024, dtype=torch.float32, device="cuda")
    result = torch.zeros(1, dtype=torch.float64, device="cuda")
    too_many = lib.NORM2_STATIC_MAX_BYTES // 4 + 1          # checked before anything is read
    with pytest.raises(lib.DwfError) as e:
        lib.dwf_norm2_static(x, result, n_reals=too_many)
    assert e.value.code == lib.ERR_INVALID_ARG and "DWF_NORM2_STATIC_MAX_BYTES" in str(e.value)
    with pytest.raises(lib.DwfError):
        lib.dwf_norm2_static(x[1:], result)                 # not 16-byte aligned
    with pytest.raises(lib.DwfError):
        lib.dwf_norm2_static(x, torch.zeros(1, dtype=torch.float32, device="cuda"))
    lib.dwf_norm2_static(x, result)                         # and a good call still works afterwards
    assert float(result.item()) == 1024.0
