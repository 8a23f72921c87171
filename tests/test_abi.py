"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/dwf.h declares, and validates arguments before touching CUDA.  No compute calls."""
import ctypes
import os
import re

import pytest

import paper_2203_06777_b200 as dwf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dwf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dwf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported():
    lib = dwf.load()
    declared = _declared_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), f"libdwf.so does not export {name}"
    assert sorted(dwf.SYMBOLS) == declared, "binding's symbol list differs from include/dwf.h"
    for name in declared:          # the Python binding carries the same names
        if name not in ("dwf_error_string", "dwf_last_error"):
            assert callable(getattr(dwf, name))


def test_no_cpp_symbols_leak():
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", dwf.LIB_PATH], capture_output=True, text=True).stdout
    names = [l.split()[-1] for l in out.splitlines() if " T " in l]
    assert names and all(n.startswith("dwf_") for n in names), names


def test_error_strings():
    lib = dwf.load()
    assert lib.dwf_error_string(0) == b"success"
    for code in range(1, 7):
        assert lib.dwf_error_string(code) not in (b"", b"success")


@pytest.mark.parametrize("dims,Ls,prec,code", [
    ((4, 4, 4, 3), 4, 8, dwf.ERR_BAD_GEOMETRY),      # odd extent
    ((4, 4, 0, 4), 4, 8, dwf.ERR_BAD_GEOMETRY),
    ((4, 4, 4, 4), 0, 8, dwf.ERR_BAD_GEOMETRY),
    ((4, 4, 4, 4), 4, 2, dwf.ERR_UNSUPPORTED),       # fp16 is not a precision of this library
    ((4096, 4096, 4096, 4096), 4, 4, dwf.ERR_BAD_GEOMETRY),
])
def test_create_geometry_rejects_bad_arguments(dims, Ls, prec, code):
    with pytest.raises(dwf.DwfError) as e:
        dwf.dwf_create_geometry(dims, Ls, prec)
    assert e.value.code == code


def test_null_arguments():
    lib = dwf.load()
    assert lib.dwf_create_geometry(None, 4, 8, 0, 0, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_dhop(None, None, None, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_load_gauge(None, None, 0, None) == dwf.ERR_INVALID_ARG
    r = ctypes.c_double(-1.0)
    assert lib.dwf_norm2(None, None, 0, ctypes.byref(r), None) == dwf.ERR_INVALID_ARG
    assert r.value == -1.0                                  # outputs untouched on error
    for f in (lib.dwf_dhop_dag, lib.dwf_dhop_oe_dag, lib.dwf_dhop_eo_dag, lib.dwf_dhop_oe, lib.dwf_dhop_eo):
        assert f(None, None, None, None) == dwf.ERR_INVALID_ARG
    for f in (lib.dwf_dhop_oe_norm2, lib.dwf_dhop_eo_norm2):
        assert f(None, None, None, ctypes.byref(r), None) == dwf.ERR_INVALID_ARG
        assert r.value == -1.0
    for f in (lib.dwf_dhop_oe_axpy, lib.dwf_dhop_eo_axpy):
        assert f(None, None, None, 1.0, 1.0, None, None) == dwf.ERR_INVALID_ARG
    for f in (lib.dwf_mooee, lib.dwf_mooee_inv):
        assert f(None, None, None, 0, 1.8, 0.1, 0, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_ddwf(None, None, None, 1.8, 0.1, 0, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_schur(None, None, None, 0, 1.8, 0.1, 0, None, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_axpby(None, 1.0, None, 1.0, None, None, 0, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_cg_schur(None, None, None, 0, 1.8, 0.1, 1e-8, 10, None, None, None, None) == dwf.ERR_INVALID_ARG
    assert lib.dwf_schur_work_bytes(None) == 0 and lib.dwf_cg_work_bytes(None) == 0
    assert lib.dwf_kernel_info(None, None, 0) == dwf.ERR_INVALID_ARG
    assert lib.dwf_set_option(None, b"kernel", 1) == dwf.ERR_INVALID_ARG
    assert lib.dwf_field_bytes(None, 0) == 0
    assert lib.dwf_destroy_geometry(None) == dwf.OK
    assert b"NULL" in lib.dwf_last_error() or lib.dwf_last_error() != b""


def test_product_does_not_import_oracle():
    """The CUDA path never routes through the oracle (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2203_06777_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src
                assert "liboracle" not in src and "dhop_oracle" not in src
