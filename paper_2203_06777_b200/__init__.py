"""paper_2203_06777_b200 -- thin Python binding of libdwf.so (include/dwf.h).

Argument marshalling only: every step of the Dhop path runs in the CUDA kernels of
``csrc/``.  The functions carry the names of the C ABI (``dwf_create_geometry``,
``dwf_load_gauge``, ``dwf_dhop``, ``dwf_dhop_oe``, ``dwf_dhop_eo``, ``dwf_norm2`` ...) and take
numpy arrays (host, canonical layouts) or torch CUDA tensors (device memory).  PyTorch is used
for device memory and streams only.  There is no CPU fallback: ``load()`` raises when
``libdwf.so`` cannot be loaded, and this package never imports ``oracle``.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

OK, ERR_INVALID_ARG, ERR_BAD_GEOMETRY, ERR_NO_GAUGE, ERR_CUDA, ERR_ALLOC, ERR_UNSUPPORTED = range(7)
F32, F64 = 4, 8
PERIODIC, ANTIPERIODIC_T, OPEN_T = 0, 1, 2
FULL, EVEN, ODD = -1, 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdwf.so")

# every symbol include/dwf.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "dwf_create_geometry", "dwf_destroy_geometry", "dwf_load_gauge", "dwf_dhop", "dwf_dhop_oe",
    "dwf_dhop_eo", "dwf_dhop_dag", "dwf_dhop_oe_dag", "dwf_dhop_eo_dag", "dwf_dhop_oe_axpy", "dwf_dhop_eo_axpy", "dwf_dhop_oe_norm2", "dwf_dhop_eo_norm2", "dwf_norm2", "dwf_inner_product", "dwf_field_bytes",
    "dwf_import_spinor", "dwf_export_spinor", "dwf_launch_count", "dwf_kernel_info", "dwf_set_option",
    "dwf_error_string", "dwf_last_error",
    "dwf_dhop_oe_mrhs", "dwf_dhop_eo_mrhs", "dwf_host_wait", "dwf_face_bytes", "dwf_face_pack_t", "dwf_face_apply_t",
    "dwf_mooee", "dwf_mooee_inv", "dwf_ddwf", "dwf_schur_work_bytes", "dwf_schur", "dwf_axpby", "dwf_cg_work_bytes", "dwf_cg_schur",
    "dwf_dhop_oe_norm2_async", "dwf_dhop_eo_norm2_async", "dwf_reduction_wait",
    "dwf_norm2_static", "dwf_to_f16", "dwf_from_f16", "dwf_dhop_oe_f16", "dwf_dhop_eo_f16",
)


class DwfError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str):
        super().__init__(f"{what}: {detail} (code {code})")
        self.code = code


_lib = None


def load(build_if_missing: bool = True):
    """Load libdwf.so (building it in-tree with nvcc if it is absent).  Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise RuntimeError(f"{LIB_PATH} is missing: run python -m paper_2203_06777_b200.build")
        from . import build as _b
        _b.build()
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, cs = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    lib.dwf_create_geometry.argtypes = [ctypes.POINTER(ci), ci, ci, ci, ci, ctypes.POINTER(vp)]
    lib.dwf_destroy_geometry.argtypes = [vp]
    lib.dwf_load_gauge.argtypes = [vp, vp, ci, vp]
    for f in (lib.dwf_dhop, lib.dwf_dhop_oe, lib.dwf_dhop_eo, lib.dwf_dhop_dag, lib.dwf_dhop_oe_dag, lib.dwf_dhop_eo_dag):
        f.argtypes = [vp, vp, vp, vp]
    for f in (lib.dwf_dhop_oe_mrhs, lib.dwf_dhop_eo_mrhs):
        f.argtypes = [vp, vp, vp, ci, ci, vp]
    lib.dwf_norm2.argtypes = [vp, vp, ci, ctypes.POINTER(ctypes.c_double), vp]
    lib.dwf_norm2_static.argtypes = [vp, ctypes.c_size_t, ci, ci, vp, vp]
    for f in (lib.dwf_dhop_oe_norm2_async, lib.dwf_dhop_eo_norm2_async):
        f.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_ulonglong), vp]
    lib.dwf_reduction_wait.argtypes = [vp, ctypes.c_ulonglong, ctypes.POINTER(ctypes.c_double), vp]
    for f in (lib.dwf_to_f16, lib.dwf_from_f16):
        f.argtypes = [vp, vp, ci, vp, vp]
    for f in (lib.dwf_dhop_oe_f16, lib.dwf_dhop_eo_f16):
        f.argtypes = [vp, vp, vp, vp]
    for f in (lib.dwf_dhop_oe_axpy, lib.dwf_dhop_eo_axpy):
        f.argtypes = [vp, vp, vp, ctypes.c_double, ctypes.c_double, vp, vp]
    for f in (lib.dwf_dhop_oe_norm2, lib.dwf_dhop_eo_norm2):
        f.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.dwf_inner_product.argtypes = [vp, vp, vp, ci, ctypes.POINTER(ctypes.c_double), vp]
    lib.dwf_field_bytes.argtypes = [vp, ci]
    lib.dwf_field_bytes.restype = cs
    lib.dwf_import_spinor.argtypes = [vp, vp, ci, ci, vp, vp]
    lib.dwf_export_spinor.argtypes = [vp, vp, ci, vp, ci, vp]
    lib.dwf_host_wait.argtypes = [vp]
    lib.dwf_face_bytes.argtypes = [vp]
    lib.dwf_face_bytes.restype = cs
    lib.dwf_face_pack_t.argtypes = [vp, vp, ci, ci, vp, vp, vp]
    lib.dwf_face_apply_t.argtypes = [vp, vp, vp, ctypes.c_double, ctypes.c_double, vp, ci, ci, vp]
    lib.dwf_launch_count.argtypes = []
    lib.dwf_launch_count.restype = ctypes.c_ulonglong
    lib.dwf_kernel_info.argtypes = [vp, ctypes.c_char_p, cs]
    dbl = ctypes.c_double
    for f in (lib.dwf_mooee, lib.dwf_mooee_inv):
        f.argtypes = [vp, vp, vp, ci, dbl, dbl, ci, vp]
    lib.dwf_ddwf.argtypes = [vp, vp, vp, dbl, dbl, ci, vp]
    lib.dwf_schur.argtypes = [vp, vp, vp, ci, dbl, dbl, ci, vp, vp]
    lib.dwf_axpby.argtypes = [vp, dbl, vp, dbl, vp, vp, ci, vp]
    lib.dwf_cg_schur.argtypes = [vp, vp, vp, ci, dbl, dbl, dbl, ci, vp, ctypes.POINTER(ci), ctypes.POINTER(dbl), vp]
    for f in (lib.dwf_schur_work_bytes, lib.dwf_cg_work_bytes):
        f.argtypes = [vp]
        f.restype = cs
    lib.dwf_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_longlong]
    lib.dwf_error_string.argtypes = [ci]
    lib.dwf_error_string.restype = ctypes.c_char_p
    lib.dwf_last_error.argtypes = []
    lib.dwf_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != OK:
        lib = load()
        raise DwfError(rc, what, (lib.dwf_last_error() or lib.dwf_error_string(rc)).decode())


_geom_info = {}     # handle -> (precision, cuda device, Ls): what the argument checks below need


def _stream(stream, g=None) -> int:
    """cudaStream_t as an integer: None = torch's current stream on the geometry's device."""
    if stream is None:
        import torch
        dev = _geom_info[g][1] if g in _geom_info else None
        return int(torch.cuda.current_stream(dev).cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return int(stream.cuda_stream)
    return int(stream)


def _ptr(a):
    """(address, is_device) of a numpy array or a torch tensor."""
    if isinstance(a, np.ndarray):
        if not a.flags.c_contiguous:
            raise ValueError("host arrays must be C-contiguous")
        return a.ctypes.data, 0
    if not a.is_contiguous():
        raise ValueError("tensors must be contiguous")
    return a.data_ptr(), 1 if a.is_cuda else 0


def _dev_ptr(t, g=None, parity=None) -> int:
    """Address of a device field.  With g and parity: also checks the element type against the
    geometry's precision and the size against dwf_field_bytes (the C ABI carries no sizes)."""
    if not getattr(t, "is_cuda", False) or not t.is_contiguous():
        raise ValueError("device fields must be contiguous torch CUDA tensors")
    if g in _geom_info and parity is not None:
        prec, dev, _ = _geom_info[g]
        if t.element_size() != prec or not t.dtype.is_floating_point:
            raise DwfError(ERR_INVALID_ARG, "binding", f"field dtype {t.dtype} does not match the geometry's precision ({prec} bytes per real)")
        want = dwf_field_bytes(g, parity)
        if t.numel() * t.element_size() != want:
            raise DwfError(ERR_INVALID_ARG, "binding", f"field holds {t.numel() * t.element_size()} bytes, the geometry needs {want} (parity {parity})")
        if t.device.index != dev:
            raise DwfError(ERR_INVALID_ARG, "binding", f"field lives on cuda:{t.device.index}, the geometry on cuda:{dev}")
    return t.data_ptr()


def _canon(a, g, parity):
    """(address, is_device) of a canonical array, size- and dtype-checked against the geometry."""
    p, on_dev = _ptr(a)
    if g in _geom_info:
        prec = _geom_info[g][0]
        nbytes = a.nbytes if isinstance(a, np.ndarray) else a.numel() * a.element_size()
        item = a.itemsize if isinstance(a, np.ndarray) else a.element_size()
        if item != prec or nbytes != dwf_field_bytes(g, parity):
            raise DwfError(ERR_INVALID_ARG, "binding", "canonical array does not match the geometry (dtype or size)")
    return p, on_dev


# ---------------------------------------------------------------------------------------------
# the C ABI, name for name
# ---------------------------------------------------------------------------------------------
def dwf_create_geometry(dims, Ls: int, precision: int, bc_time: int = PERIODIC, cuda_device: int = 0) -> int:
    lib = load()
    d = (ctypes.c_int * 4)(*[int(v) for v in dims])
    h = ctypes.c_void_p()
    _check(lib.dwf_create_geometry(d, int(Ls), int(precision), int(bc_time), int(cuda_device),
                                   ctypes.byref(h)), "dwf_create_geometry")
    _geom_info[h.value] = (int(precision), int(cuda_device), int(Ls))
    return h.value


def dwf_destroy_geometry(g: int) -> None:
    _geom_info.pop(g, None)
    _check(load().dwf_destroy_geometry(g), "dwf_destroy_geometry")


def dwf_load_gauge(g: int, U, stream=None) -> None:
    p, on_dev = _ptr(U)
    if g in _geom_info:
        item = U.itemsize if isinstance(U, np.ndarray) else U.element_size()
        nbytes = U.nbytes if isinstance(U, np.ndarray) else U.numel() * U.element_size()
        if item != _geom_info[g][0] or nbytes != dwf_field_bytes(g, FULL) // _geom_info[g][2] * 3:
            raise DwfError(ERR_INVALID_ARG, "binding", "gauge array does not match the geometry (dtype or size: V4*72 reals)")
    _check(load().dwf_load_gauge(g, p, on_dev, _stream(stream, g)), "dwf_load_gauge")


def dwf_dhop(g: int, in_full, out_full, stream=None) -> None:
    _check(load().dwf_dhop(g, _dev_ptr(in_full, g, FULL), _dev_ptr(out_full, g, FULL), _stream(stream, g)), "dwf_dhop")


def dwf_dhop_oe(g: int, in_even, out_odd, stream=None) -> None:
    _check(load().dwf_dhop_oe(g, _dev_ptr(in_even, g, EVEN), _dev_ptr(out_odd, g, ODD), _stream(stream, g)), "dwf_dhop_oe")


def dwf_dhop_eo(g: int, in_odd, out_even, stream=None) -> None:
    _check(load().dwf_dhop_eo(g, _dev_ptr(in_odd, g, ODD), _dev_ptr(out_even, g, EVEN), _stream(stream, g)), "dwf_dhop_eo")


def dwf_dhop_dag(g: int, in_full, out_full, stream=None) -> None:
    _check(load().dwf_dhop_dag(g, _dev_ptr(in_full, g, FULL), _dev_ptr(out_full, g, FULL), _stream(stream, g)), "dwf_dhop_dag")


def dwf_dhop_oe_dag(g: int, in_even, out_odd, stream=None) -> None:
    _check(load().dwf_dhop_oe_dag(g, _dev_ptr(in_even, g, EVEN), _dev_ptr(out_odd, g, ODD), _stream(stream, g)), "dwf_dhop_oe_dag")


def dwf_dhop_eo_dag(g: int, in_odd, out_even, stream=None) -> None:
    _check(load().dwf_dhop_eo_dag(g, _dev_ptr(in_odd, g, ODD), _dev_ptr(out_even, g, EVEN), _stream(stream, g)), "dwf_dhop_eo_dag")


def _mrhs_ptr(t, g, parity, nrhs):
    """Address of nrhs device fields stored one after the other (size- and dtype-checked)."""
    if not getattr(t, "is_cuda", False) or not t.is_contiguous():
        raise ValueError("device fields must be contiguous torch CUDA tensors")
    if g in _geom_info:
        prec = _geom_info[g][0]
        if t.element_size() != prec or t.numel() * prec != int(nrhs) * dwf_field_bytes(g, parity):
            raise DwfError(ERR_INVALID_ARG, "binding", "multi-RHS buffer does not match nrhs fields of the geometry (dtype or size)")
    return t.data_ptr()


def dwf_dhop_oe_mrhs(g: int, in_even, out_odd, nrhs: int, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_dhop_oe_mrhs(g, _mrhs_ptr(in_even, g, EVEN, nrhs), _mrhs_ptr(out_odd, g, ODD, nrhs), int(nrhs),
                                   int(bool(dagger)), _stream(stream, g)), "dwf_dhop_oe_mrhs")


def dwf_dhop_eo_mrhs(g: int, in_odd, out_even, nrhs: int, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_dhop_eo_mrhs(g, _mrhs_ptr(in_odd, g, ODD, nrhs), _mrhs_ptr(out_even, g, EVEN, nrhs), int(nrhs),
                                   int(bool(dagger)), _stream(stream, g)), "dwf_dhop_eo_mrhs")


def dwf_dhop_oe_axpy(g: int, in_even, x_odd, a: float, b: float, out_odd, stream=None) -> None:
    _check(load().dwf_dhop_oe_axpy(g, _dev_ptr(in_even, g, EVEN), _dev_ptr(x_odd, g, ODD), float(a), float(b),
                                   _dev_ptr(out_odd, g, ODD), _stream(stream, g)), "dwf_dhop_oe_axpy")


def dwf_dhop_eo_axpy(g: int, in_odd, x_even, a: float, b: float, out_even, stream=None) -> None:
    _check(load().dwf_dhop_eo_axpy(g, _dev_ptr(in_odd, g, ODD), _dev_ptr(x_even, g, EVEN), float(a), float(b),
                                   _dev_ptr(out_even, g, EVEN), _stream(stream, g)), "dwf_dhop_eo_axpy")


def dwf_dhop_oe_norm2(g: int, in_even, out_odd, stream=None) -> float:
    r = ctypes.c_double()
    _check(load().dwf_dhop_oe_norm2(g, _dev_ptr(in_even, g, EVEN), _dev_ptr(out_odd, g, ODD), ctypes.byref(r), _stream(stream, g)),
           "dwf_dhop_oe_norm2")
    return r.value


def dwf_dhop_eo_norm2(g: int, in_odd, out_even, stream=None) -> float:
    r = ctypes.c_double()
    _check(load().dwf_dhop_eo_norm2(g, _dev_ptr(in_odd, g, ODD), _dev_ptr(out_even, g, EVEN), ctypes.byref(r), _stream(stream, g)),
           "dwf_dhop_eo_norm2")
    return r.value


def dwf_norm2(g: int, field, parity: int = FULL, stream=None) -> float:
    r = ctypes.c_double()
    _check(load().dwf_norm2(g, _dev_ptr(field, g, parity), int(parity), ctypes.byref(r), _stream(stream, g)), "dwf_norm2")
    return r.value


def dwf_dhop_oe_norm2_async(g: int, in_even, out_odd, stream=None) -> int:
    """Enqueues DhopOE + norm2 and returns the ticket of the reduction (dwf_reduction_wait collects the value)."""
    t = ctypes.c_ulonglong()
    _check(load().dwf_dhop_oe_norm2_async(g, _dev_ptr(in_even, g, EVEN), _dev_ptr(out_odd, g, ODD), ctypes.byref(t), _stream(stream, g)),
           "dwf_dhop_oe_norm2_async")
    return int(t.value)


def dwf_dhop_eo_norm2_async(g: int, in_odd, out_even, stream=None) -> int:
    t = ctypes.c_ulonglong()
    _check(load().dwf_dhop_eo_norm2_async(g, _dev_ptr(in_odd, g, ODD), _dev_ptr(out_even, g, EVEN), ctypes.byref(t), _stream(stream, g)),
           "dwf_dhop_eo_norm2_async")
    return int(t.value)


def dwf_reduction_wait(g: int, ticket: int, stream=None) -> float:
    r = ctypes.c_double()
    _check(load().dwf_reduction_wait(g, int(ticket), ctypes.byref(r), _stream(stream, g)), "dwf_reduction_wait")
    return r.value


def _f16_ptr(t, g: int, parity: int) -> int:
    """Address of a device field in fp16 storage (include/dwf.h): a float16 tensor with as many reals as the fp32 field."""
    import torch
    if not getattr(t, "is_cuda", False) or not t.is_contiguous() or t.dtype != torch.float16:
        raise DwfError(ERR_INVALID_ARG, "binding", "fp16-stored fields must be contiguous float16 CUDA tensors")
    if g in _geom_info:
        prec, dev, _ = _geom_info[g]
        if t.numel() * prec != dwf_field_bytes(g, parity) or t.device.index != dev:
            raise DwfError(ERR_INVALID_ARG, "binding", "fp16-stored field does not match the geometry (size, parity or device)")
    return t.data_ptr()


def dwf_to_f16(g: int, field_f32, parity: int, field_f16, stream=None) -> None:
    _check(load().dwf_to_f16(g, _dev_ptr(field_f32, g, parity), int(parity), _f16_ptr(field_f16, g, parity), _stream(stream, g)), "dwf_to_f16")


def dwf_from_f16(g: int, field_f16, parity: int, field_f32, stream=None) -> None:
    _check(load().dwf_from_f16(g, _f16_ptr(field_f16, g, parity), int(parity), _dev_ptr(field_f32, g, parity), _stream(stream, g)), "dwf_from_f16")


def dwf_dhop_oe_f16(g: int, in_even_f16, out_odd_f16, stream=None) -> None:
    _check(load().dwf_dhop_oe_f16(g, _f16_ptr(in_even_f16, g, EVEN), _f16_ptr(out_odd_f16, g, ODD), _stream(stream, g)), "dwf_dhop_oe_f16")


def dwf_dhop_eo_f16(g: int, in_odd_f16, out_even_f16, stream=None) -> None:
    _check(load().dwf_dhop_eo_f16(g, _f16_ptr(in_odd_f16, g, ODD), _f16_ptr(out_even_f16, g, EVEN), _stream(stream, g)), "dwf_dhop_eo_f16")


NORM2_STATIC_MAX_BYTES = 1 << 31


def dwf_norm2_static(x, result, n_reals: int | None = None, stream=None) -> None:
    """result[0] = sum x^2 without any allocation (include/dwf.h).  x: CUDA tensor (float32 / float64, contiguous),
    result: CUDA float64 tensor of one element on the same device; asynchronous on `stream` (None = torch's current
    stream on x's device).  n_reals: number of leading elements to sum (default: all)."""
    import torch
    if not (x.is_cuda and result.is_cuda and x.device == result.device and x.is_contiguous()):
        raise DwfError(ERR_INVALID_ARG, "binding", "x and result must be contiguous CUDA tensors on one device")
    if x.dtype not in (torch.float32, torch.float64) or result.dtype != torch.float64 or result.numel() < 1:
        raise DwfError(ERR_INVALID_ARG, "binding", "x must be float32 / float64, result float64 with one element")
    n = x.numel() if n_reals is None else int(n_reals)
    dev = x.device.index if x.device.index is not None else torch.cuda.current_device()
    st = int(torch.cuda.current_stream(dev).cuda_stream) if stream is None else _stream(stream)
    _check(load().dwf_norm2_static(x.data_ptr(), n, x.element_size(), dev, result.data_ptr(), st), "dwf_norm2_static")


def dwf_inner_product(g: int, a, b, parity: int = FULL, stream=None) -> complex:
    r = (ctypes.c_double * 2)()
    _check(load().dwf_inner_product(g, _dev_ptr(a, g, parity), _dev_ptr(b, g, parity), int(parity), r, _stream(stream, g)),
           "dwf_inner_product")
    return complex(r[0], r[1])


def dwf_field_bytes(g: int, parity: int = FULL) -> int:
    return int(load().dwf_field_bytes(g, int(parity)))


def dwf_import_spinor(g: int, canonical, parity: int, field_dev, stream=None) -> None:
    p, on_dev = _canon(canonical, g, parity)
    _check(load().dwf_import_spinor(g, p, on_dev, int(parity), _dev_ptr(field_dev, g, parity), _stream(stream, g)),
           "dwf_import_spinor")


def dwf_export_spinor(g: int, field_dev, parity: int, canonical, stream=None) -> None:
    p, on_dev = _canon(canonical, g, parity)
    _check(load().dwf_export_spinor(g, _dev_ptr(field_dev, g, parity), int(parity), p, on_dev, _stream(stream, g)),
           "dwf_export_spinor")


def dwf_mooee(g: int, inp, out, parity: int, M5: float, mass: float, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_mooee(g, _dev_ptr(inp, g, parity), _dev_ptr(out, g, parity), int(parity), float(M5), float(mass),
                            int(bool(dagger)), _stream(stream, g)), "dwf_mooee")


def dwf_mooee_inv(g: int, inp, out, parity: int, M5: float, mass: float, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_mooee_inv(g, _dev_ptr(inp, g, parity), _dev_ptr(out, g, parity), int(parity), float(M5), float(mass),
                                int(bool(dagger)), _stream(stream, g)), "dwf_mooee_inv")


def dwf_ddwf(g: int, in_full, out_full, M5: float, mass: float, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_ddwf(g, _dev_ptr(in_full, g, FULL), _dev_ptr(out_full, g, FULL), float(M5), float(mass),
                           int(bool(dagger)), _stream(stream, g)), "dwf_ddwf")


def dwf_schur_work_bytes(g: int) -> int:
    return int(load().dwf_schur_work_bytes(g))


def dwf_cg_work_bytes(g: int) -> int:
    return int(load().dwf_cg_work_bytes(g))


def _work_ptr(t, need: int) -> int:
    if not getattr(t, "is_cuda", False) or not t.is_contiguous() or t.numel() * t.element_size() < need:
        raise DwfError(ERR_INVALID_ARG, "binding", f"workspace must be a contiguous CUDA tensor of at least {need} bytes")
    return t.data_ptr()


def dwf_schur(g: int, inp, out, parity: int, M5: float, mass: float, work, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_schur(g, _dev_ptr(inp, g, parity), _dev_ptr(out, g, parity), int(parity), float(M5), float(mass),
                            int(bool(dagger)), _work_ptr(work, dwf_schur_work_bytes(g)), _stream(stream, g)), "dwf_schur")


def dwf_axpby(g: int, a: float, x, b: float, y, out, parity: int, stream=None) -> None:
    _check(load().dwf_axpby(g, float(a), _dev_ptr(x, g, parity), float(b), _dev_ptr(y, g, parity), _dev_ptr(out, g, parity),
                            int(parity), _stream(stream, g)), "dwf_axpby")


def dwf_cg_schur(g: int, b, x, parity: int, M5: float, mass: float, tol: float, max_iter: int, work, stream=None):
    """Returns (iterations, true relative residual)."""
    it, res = ctypes.c_int(), ctypes.c_double()
    _check(load().dwf_cg_schur(g, _dev_ptr(b, g, parity), _dev_ptr(x, g, parity), int(parity), float(M5), float(mass),
                               float(tol), int(max_iter), _work_ptr(work, dwf_cg_work_bytes(g)), ctypes.byref(it),
                               ctypes.byref(res), _stream(stream, g)), "dwf_cg_schur")
    return it.value, res.value


def dwf_face_bytes(g: int) -> int:
    return int(load().dwf_face_bytes(g))


def _face_ptr(t, g) -> int:
    if not getattr(t, "is_cuda", False) or not t.is_contiguous() or t.numel() * t.element_size() != dwf_face_bytes(g):
        raise DwfError(ERR_INVALID_ARG, "binding", "face buffers must be contiguous CUDA tensors of dwf_face_bytes bytes")
    return t.data_ptr()


def dwf_face_pack_t(g: int, inp, parity_in: int, send_down, send_up, dagger: bool = False, stream=None) -> None:
    _check(load().dwf_face_pack_t(g, _dev_ptr(inp, g, parity_in), int(parity_in), int(bool(dagger)), _face_ptr(send_down, g),
                                  _face_ptr(send_up, g), _stream(stream, g)), "dwf_face_pack_t")


def dwf_face_apply_t(g: int, recv_lo, recv_hi, sign_lo: float, sign_hi: float, out, parity_out: int, dagger: bool = False,
                     stream=None) -> None:
    _check(load().dwf_face_apply_t(g, _face_ptr(recv_lo, g), _face_ptr(recv_hi, g), float(sign_lo), float(sign_hi),
                                   _dev_ptr(out, g, parity_out), int(parity_out), int(bool(dagger)), _stream(stream, g)), "dwf_face_apply_t")


def dwf_host_wait(g: int) -> None:
    _check(load().dwf_host_wait(g), "dwf_host_wait")


def dwf_launch_count() -> int:
    return int(load().dwf_launch_count())


def dwf_kernel_info(g: int) -> str:
    buf = ctypes.create_string_buffer(128)
    _check(load().dwf_kernel_info(g, buf, 128), "dwf_kernel_info")
    return buf.value.decode()


def dwf_set_option(g: int, key: str, value: int) -> None:
    _check(load().dwf_set_option(g, key.encode(), int(value)), f"dwf_set_option({key})")


# ---------------------------------------------------------------------------------------------
# convenience wrapper: owns the handle, allocates device fields with torch
# ---------------------------------------------------------------------------------------------
class Geometry:
    """A dwf_geometry handle plus torch-allocated device fields.  No arithmetic here."""

    def __init__(self, dims, Ls: int, precision: int, bc_time: int = PERIODIC, device: int = 0):
        import torch
        self.dims = tuple(int(d) for d in dims)
        self.Ls, self.precision, self.bc_time, self.device = int(Ls), int(precision), int(bc_time), int(device)
        self.V4 = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self._torch = torch
        self.handle = dwf_create_geometry(self.dims, Ls, precision, bc_time, device)

    def close(self):
        if getattr(self, "handle", None):
            dwf_destroy_geometry(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def np_dtype(self):
        return np.float32 if self.precision == F32 else np.float64

    @property
    def torch_dtype(self):
        return self._torch.float32 if self.precision == F32 else self._torch.float64

    def nsites(self, parity: int = FULL) -> int:
        return self.V4 if parity == FULL else self.V4 // 2

    def new_field(self, parity: int = FULL):
        """Uninitialised device field (device layout), a flat torch tensor of reals."""
        n = dwf_field_bytes(self.handle, parity) // self.precision
        return self._torch.empty(n, dtype=self.torch_dtype, device=f"cuda:{self.device}")

    def load_gauge(self, U, stream=None):
        dwf_load_gauge(self.handle, U, stream)

    def import_spinor(self, canonical, parity: int = FULL, out=None, stream=None):
        out = self.new_field(parity) if out is None else out
        dwf_import_spinor(self.handle, canonical, parity, out, stream)
        return out

    def export_spinor(self, field, parity: int = FULL, out=None, stream=None):
        if out is None:
            out = np.empty((self.nsites(parity), self.Ls, 4, 3, 2), dtype=self.np_dtype)
        dwf_export_spinor(self.handle, field, parity, out, stream)
        return out

    def dhop(self, inp, out=None, stream=None):
        out = self.new_field(FULL) if out is None else out
        dwf_dhop(self.handle, inp, out, stream)
        return out

    def dhop_dag(self, inp, out=None, stream=None):
        out = self.new_field(FULL) if out is None else out
        dwf_dhop_dag(self.handle, inp, out, stream)
        return out

    def dhop_oe_dag(self, in_even, out=None, stream=None):
        out = self.new_field(ODD) if out is None else out
        dwf_dhop_oe_dag(self.handle, in_even, out, stream)
        return out

    def dhop_eo_dag(self, in_odd, out=None, stream=None):
        out = self.new_field(EVEN) if out is None else out
        dwf_dhop_eo_dag(self.handle, in_odd, out, stream)
        return out

    def dhop_oe(self, in_even, out=None, stream=None):
        out = self.new_field(ODD) if out is None else out
        dwf_dhop_oe(self.handle, in_even, out, stream)
        return out

    def dhop_oe_norm2_async(self, in_even, out=None, stream=None):
        """(out, ticket): enqueued, not waited for; reduction_wait(ticket) returns the norm2"""
        out = self.new_field(ODD) if out is None else out
        return out, dwf_dhop_oe_norm2_async(self.handle, in_even, out, stream)

    def dhop_eo_norm2_async(self, in_odd, out=None, stream=None):
        out = self.new_field(EVEN) if out is None else out
        return out, dwf_dhop_eo_norm2_async(self.handle, in_odd, out, stream)

    def reduction_wait(self, ticket: int, stream=None) -> float:
        return dwf_reduction_wait(self.handle, ticket, stream)

    # fp16 storage: float16 tensors in the fp32 device layout
    def new_field_f16(self, parity: int = FULL):
        n = dwf_field_bytes(self.handle, parity) // self.precision
        return self._torch.empty(n, dtype=self._torch.float16, device=f"cuda:{self.device}")

    def to_f16(self, field, parity: int, out=None, stream=None):
        out = self.new_field_f16(parity) if out is None else out
        dwf_to_f16(self.handle, field, parity, out, stream)
        return out

    def from_f16(self, field_f16, parity: int, out=None, stream=None):
        out = self.new_field(parity) if out is None else out
        dwf_from_f16(self.handle, field_f16, parity, out, stream)
        return out

    def dhop_oe_f16(self, in_even_f16, out=None, stream=None):
        out = self.new_field_f16(ODD) if out is None else out
        dwf_dhop_oe_f16(self.handle, in_even_f16, out, stream)
        return out

    def dhop_eo_f16(self, in_odd_f16, out=None, stream=None):
        out = self.new_field_f16(EVEN) if out is None else out
        dwf_dhop_eo_f16(self.handle, in_odd_f16, out, stream)
        return out

    def dhop_eo(self, in_odd, out=None, stream=None):
        out = self.new_field(EVEN) if out is None else out
        dwf_dhop_eo(self.handle, in_odd, out, stream)
        return out

    def dhop_oe_mrhs(self, in_even, nrhs, dagger=False, out=None, stream=None):
        """nrhs right-hand sides (fields stored one after the other) in one launch, one gauge load."""
        out = self._torch.empty_like(in_even) if out is None else out
        dwf_dhop_oe_mrhs(self.handle, in_even, out, nrhs, dagger, stream)
        return out

    def dhop_eo_mrhs(self, in_odd, nrhs, dagger=False, out=None, stream=None):
        out = self._torch.empty_like(in_odd) if out is None else out
        dwf_dhop_eo_mrhs(self.handle, in_odd, out, nrhs, dagger, stream)
        return out

    def dhop_oe_axpy(self, in_even, x_odd, a, b, out=None, stream=None):
        """out = a x + b DhopOE in (x, out odd half fields; x may be out on the fused path)."""
        out = self.new_field(ODD) if out is None else out
        dwf_dhop_oe_axpy(self.handle, in_even, x_odd, a, b, out, stream)
        return out

    def dhop_eo_axpy(self, in_odd, x_even, a, b, out=None, stream=None):
        """out = a x + b DhopEO in (x, out even half fields)."""
        out = self.new_field(EVEN) if out is None else out
        dwf_dhop_eo_axpy(self.handle, in_odd, x_even, a, b, out, stream)
        return out

    def dhop_oe_norm2(self, in_even, out=None, stream=None):
        """DhopOE fused with norm2 of its result: returns (out_odd, norm2)."""
        out = self.new_field(ODD) if out is None else out
        return out, dwf_dhop_oe_norm2(self.handle, in_even, out, stream)

    def dhop_eo_norm2(self, in_odd, out=None, stream=None):
        """DhopEO fused with norm2 of its result: returns (out_even, norm2)."""
        out = self.new_field(EVEN) if out is None else out
        return out, dwf_dhop_eo_norm2(self.handle, in_odd, out, stream)

    def norm2(self, field, parity: int = FULL, stream=None) -> float:
        return dwf_norm2(self.handle, field, parity, stream)

    def inner_product(self, a, b, parity: int = FULL, stream=None) -> complex:
        return dwf_inner_product(self.handle, a, b, parity, stream)

    # ---- the rest of the red-black domain-wall operator ----
    def new_work(self, nbytes: int):
        return self._torch.empty(nbytes, dtype=self._torch.uint8, device=f"cuda:{self.device}")

    def mooee(self, inp, parity, M5, mass, dagger=False, out=None, stream=None):
        out = self.new_field(parity) if out is None else out
        dwf_mooee(self.handle, inp, out, parity, M5, mass, dagger, stream)
        return out

    def mooee_inv(self, inp, parity, M5, mass, dagger=False, out=None, stream=None):
        out = self.new_field(parity) if out is None else out
        dwf_mooee_inv(self.handle, inp, out, parity, M5, mass, dagger, stream)
        return out

    def ddwf(self, inp, M5, mass, dagger=False, out=None, stream=None):
        out = self.new_field(FULL) if out is None else out
        dwf_ddwf(self.handle, inp, out, M5, mass, dagger, stream)
        return out

    def schur(self, inp, parity, M5, mass, dagger=False, out=None, work=None, stream=None):
        out = self.new_field(parity) if out is None else out
        work = self.new_work(dwf_schur_work_bytes(self.handle)) if work is None else work
        dwf_schur(self.handle, inp, out, parity, M5, mass, work, dagger, stream)
        return out

    def axpby(self, a, x, b, y, parity, out=None, stream=None):
        out = self.new_field(parity) if out is None else out
        dwf_axpby(self.handle, a, x, b, y, out, parity, stream)
        return out

    def cg_schur(self, b, parity, M5, mass, tol, max_iter, x=None, work=None, stream=None):
        """Solve S x = b: returns (x, iterations, true relative residual)."""
        x = self.new_field(parity) if x is None else x
        work = self.new_work(dwf_cg_work_bytes(self.handle)) if work is None else work
        it, res = dwf_cg_schur(self.handle, b, x, parity, M5, mass, tol, max_iter, work, stream)
        return x, it, res

    def host_wait(self):
        dwf_host_wait(self.handle)

    def set_option(self, key: str, value: int):
        dwf_set_option(self.handle, key, value)

    def kernel_info(self) -> str:
        return dwf_kernel_info(self.handle)
