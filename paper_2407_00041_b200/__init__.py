"""paper_2407_00041_b200 — B200-native Wilson(-clover) Dirac operator (arxiv 2407.00041 hot path).

Thin ctypes binding of the C-ABI in include/wd.h: the functions below have the same names and
argument order as the C entry points and do argument marshalling only — every step of the path
(packing on request, neighbour indexing, projection, SU(3) multiply, reconstruction, clover,
store) runs inside libwd.so's CUDA kernels.  PyTorch is used by callers for device memory and
streams only.  There is NO CPU fallback: importing works without a GPU (so that the symbol table
can be checked), but any compute call needs a CUDA device, and a missing libwd.so raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwd.so")

WD_OK, WD_EINVAL, WD_ENOMEM, WD_ESTATE, WD_ECUDA = 0, -1, -2, -3, -4
WD_FIELD_SPINOR, WD_FIELD_GAUGE, WD_FIELD_CLOVER, WD_FIELD_SPINOR_BLOCK4 = 0, 1, 2, 3
WD_OPT_VARIANT, WD_OPT_KERNEL, WD_OPT_TCHUNK, WD_OPT_ZGROUP, WD_OPT_DEVICE_PACK, WD_OPT_HOST_PIPELINE = 1, 2, 3, 4, 5, 6
WD_OPT_GMRES_GRAPH, WD_OPT_GAUGE_ROWS, WD_OPT_F32_KERNEL, WD_OPT_RHS_BLOCK = 7, 8, 9, 10

# name -> (restype, argtypes); mirrors include/wd.h declaration by declaration
_vp, _i, _d, _l, _sz, _cp = (ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_long,
                             ctypes.c_size_t, ctypes.c_char_p)
SIGNATURES = {
    "wd_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, _d, _d]),
    "wd_destroy": (_i, [_vp]),
    "wd_load_gauge": (_i, [_vp, _vp]),
    "wd_load_clover": (_i, [_vp, _vp]),
    "wd_build_clover": (_i, [_vp]),
    "wd_get_clover": (_i, [_vp, _vp]),
    "wd_apply": (_i, [_vp, _vp, _vp, _i]),
    "wd_apply_host": (_i, [_vp, _vp, _vp, _i]),
    "wd_enable_f32": (_i, [_vp]),
    "wd_spinor_bytes_f32": (_sz, [_vp, _i]),
    "wd_convert_spinor": (_i, [_vp, _vp, _vp, _i, _i]),
    "wd_apply_f32": (_i, [_vp, _vp, _vp, _i]),
    "wd_create_local": (_i, [ctypes.POINTER(_vp), ctypes.POINTER(_i), ctypes.POINTER(_i), ctypes.POINTER(_i), _d, _d]),
    "wd_dd_open_mask": (_i, [_vp]),
    "wd_dd_face_sites": (ctypes.c_longlong, [_vp, _i]),
    "wd_dd_face_bytes": (_sz, [_vp, _i, _i]),
    "wd_dd_pack": (_i, [_vp, _vp, _i, _i, _vp, _vp]),
    "wd_dd_exterior": (_i, [_vp, _vp, _i, _i, _vp, _vp]),
    "wd_gmres": (_i, [_vp, _vp, _vp, _i, _i, _d, ctypes.POINTER(_i), _vp]),
    "wd_gmres_mixed": (_i, [_vp, _vp, _vp, _i, _i, _d, ctypes.POINTER(_i), _vp]),
    "wd_gmres_last_hessenberg": (_i, [_vp, _vp, ctypes.POINTER(_i), ctypes.POINTER(_d)]),
    "wd_inner_product_static": (_i, [_vp, _vp, ctypes.c_longlong, ctypes.c_longlong, _i, _vp, _vp]),
    "wd_spinor_bytes": (_sz, [_vp, _i]),
    "wd_component_stride": (ctypes.c_longlong, [_vp]),
    "wd_pack_spinor": (_i, [_vp, _vp, _vp, _i]),
    "wd_unpack_spinor": (_i, [_vp, _vp, _vp, _i]),
    "wd_layout_bytes": (_sz, [_i, ctypes.c_longlong]),
    "wd_layout_pack_host": (_i, [_i, ctypes.c_longlong, _vp, _vp]),
    "wd_layout_unpack_host": (_i, [_i, ctypes.c_longlong, _vp, _vp]),
    "wd_set_stream": (_i, [_vp, _vp]),
    "wd_synchronize": (_i, [_vp]),
    "wd_set_option": (_i, [_vp, _i, _l]),
    "wd_get_option": (_i, [_vp, _i, ctypes.POINTER(_l)]),
    "wd_kernel_count": (_i, []),
    "wd_kernel_name": (_cp, [_i]),
    "wd_kernel_in_use": (_i, [_vp]),
    "wd_kernel_for": (_i, [_vp, _i]),
    "wd_launch_count": (_l, [_vp]),
    "wd_last_error": (_cp, [_vp]),
    "wd_version": (_cp, []),
}

_lib = None


class WDError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libwd error {code}: {text}")
        self.code = code


def lib() -> ctypes.CDLL:
    """Load libwd.so (built in-tree by paper_2407_00041_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} not found: build it with `python -m paper_2407_00041_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _ptr(x) -> int | None:
    """Marshal a pointer argument: int address, None, numpy array (host) or torch tensor."""
    if x is None or isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(type(x))


def _check(h, rc: int) -> None:
    if rc != WD_OK:
        raise WDError(rc, lib().wd_last_error(h).decode())


# ---- same names as the C entry points ------------------------------------------------------------
def wd_create(T: int, Z: int, Y: int, X: int, m0: float, csw: float) -> int:
    h = _vp()
    rc = lib().wd_create(ctypes.byref(h), T, Z, Y, X, m0, csw)
    _check(None, rc)
    return h.value


def wd_create_local(global_dims, proc_grid, proc_coords, m0: float, csw: float) -> int:
    h = _vp()
    a = [(_i * 4)(*[int(v) for v in x]) for x in (global_dims, proc_grid, proc_coords)]
    rc = lib().wd_create_local(ctypes.byref(h), a[0], a[1], a[2], m0, csw)
    _check(None, rc)
    return h.value


def wd_dd_open_mask(h) -> int:
    return int(lib().wd_dd_open_mask(h))


def wd_dd_face_sites(h, mu: int) -> int:
    return int(lib().wd_dd_face_sites(h, mu))


def wd_dd_face_bytes(h, mu: int, nrhs: int = 1) -> int:
    return int(lib().wd_dd_face_bytes(h, mu, nrhs))


def wd_dd_pack(h, dev_in, nrhs: int, mu: int, dev_send_minus, dev_send_plus) -> None:
    _check(h, lib().wd_dd_pack(h, _ptr(dev_in), nrhs, mu, _ptr(dev_send_minus), _ptr(dev_send_plus)))


def wd_dd_exterior(h, dev_out, nrhs: int, mu: int, dev_recv_from_plus, dev_recv_from_minus) -> None:
    _check(h, lib().wd_dd_exterior(h, _ptr(dev_out), nrhs, mu, _ptr(dev_recv_from_plus), _ptr(dev_recv_from_minus)))


def wd_enable_f32(h) -> None:
    _check(h, lib().wd_enable_f32(h))


def wd_spinor_bytes_f32(h, nrhs: int = 1) -> int:
    return int(lib().wd_spinor_bytes_f32(h, nrhs))


def wd_convert_spinor(h, dev_dst, dev_src, nrhs: int, to_f32: bool) -> None:
    _check(h, lib().wd_convert_spinor(h, _ptr(dev_dst), _ptr(dev_src), nrhs, 1 if to_f32 else 0))


def wd_apply_f32(h, dev_out, dev_in, nrhs: int = 1) -> None:
    _check(h, lib().wd_apply_f32(h, _ptr(dev_out), _ptr(dev_in), nrhs))


def wd_destroy(h) -> None:
    _check(h, lib().wd_destroy(h))


def wd_load_gauge(h, host_U) -> None:
    _check(h, lib().wd_load_gauge(h, _ptr(host_U)))


def wd_load_clover(h, host_C) -> None:
    _check(h, lib().wd_load_clover(h, _ptr(host_C)))


def wd_build_clover(h) -> None:
    _check(h, lib().wd_build_clover(h))


def wd_get_clover(h, host_C) -> None:
    _check(h, lib().wd_get_clover(h, _ptr(host_C)))


def wd_apply(h, dev_out, dev_in, nrhs: int = 1) -> None:
    _check(h, lib().wd_apply(h, _ptr(dev_out), _ptr(dev_in), nrhs))


def wd_apply_host(h, host_out, host_in, nrhs: int = 1) -> None:
    _check(h, lib().wd_apply_host(h, _ptr(host_out), _ptr(host_in), nrhs))


def wd_gmres(h, dev_x, dev_b, m: int, max_cycles: int, tol: float, host_resid=None) -> int:
    """Returns the number of restart cycles done; host_resid: float64 array of max_cycles + 1 entries, or None."""
    n = _i(0)
    _check(h, lib().wd_gmres(h, _ptr(dev_x), _ptr(dev_b), m, max_cycles, tol, ctypes.byref(n), _ptr(host_resid)))
    return n.value


def wd_gmres_mixed(h, dev_x, dev_b, m: int, max_cycles: int, tol: float, host_resid=None) -> int:
    """wd_gmres with single-precision Krylov vectors and operator applications (needs wd_enable_f32)."""
    n = _i(0)
    _check(h, lib().wd_gmres_mixed(h, _ptr(dev_x), _ptr(dev_b), m, max_cycles, tol, ctypes.byref(n), _ptr(host_resid)))
    return n.value


def wd_gmres_last_hessenberg(h, host_H=None) -> tuple[int, float]:
    """(Krylov dimension, recurrence residual) of the last cycle; host_H: float64 array [(m+1)*m*2] or None."""
    kd, lr = _i(0), _d(0.0)
    _check(h, lib().wd_gmres_last_hessenberg(h, _ptr(host_H), ctypes.byref(kd), ctypes.byref(lr)))
    return kd.value, lr.value


def wd_inner_product_static(dev_a, dev_b, V: int, Vs: int, nrhs: int, dev_result, cuda_stream=None) -> None:
    """dev_result[r] = <a_r, b_r> without any allocation inside the library (include/wd.h: for callers that cannot
    call cudaMalloc).  dev_result: device array of nrhs complex doubles; at most 64 right-hand sides per call."""
    _check(None, lib().wd_inner_product_static(_ptr(dev_a), _ptr(dev_b), V, Vs, nrhs, _ptr(dev_result), _ptr(cuda_stream)))


def wd_spinor_bytes(h, nrhs: int = 1) -> int:
    return int(lib().wd_spinor_bytes(h, nrhs))


def wd_component_stride(h) -> int:
    return int(lib().wd_component_stride(h))


def wd_pack_spinor(h, dev_dst, host_src, nrhs: int = 1) -> None:
    _check(h, lib().wd_pack_spinor(h, _ptr(dev_dst), _ptr(host_src), nrhs))


def wd_unpack_spinor(h, host_dst, dev_src, nrhs: int = 1) -> None:
    _check(h, lib().wd_unpack_spinor(h, _ptr(host_dst), _ptr(dev_src), nrhs))


def wd_layout_bytes(field: int, nsites: int) -> int:
    return int(lib().wd_layout_bytes(field, nsites))


def wd_layout_pack_host(field: int, nsites: int, canonical, packed) -> None:
    rc = lib().wd_layout_pack_host(field, nsites, _ptr(canonical), _ptr(packed))
    if rc != WD_OK:
        raise WDError(rc, "wd_layout_pack_host: bad argument")


def wd_layout_unpack_host(field: int, nsites: int, packed, canonical) -> None:
    rc = lib().wd_layout_unpack_host(field, nsites, _ptr(packed), _ptr(canonical))
    if rc != WD_OK:
        raise WDError(rc, "wd_layout_unpack_host: bad argument")


def wd_set_stream(h, cuda_stream) -> None:
    _check(h, lib().wd_set_stream(h, _ptr(cuda_stream)))


def wd_synchronize(h) -> None:
    _check(h, lib().wd_synchronize(h))


def wd_set_option(h, option: int, value: int) -> None:
    _check(h, lib().wd_set_option(h, option, value))


def wd_get_option(h, option: int) -> int:
    v = _l()
    _check(h, lib().wd_get_option(h, option, ctypes.byref(v)))
    return v.value


def wd_kernel_count() -> int:
    return lib().wd_kernel_count()


def wd_kernel_name(kid: int) -> str | None:
    s = lib().wd_kernel_name(kid)
    return s.decode() if s else None


def wd_kernel_in_use(h) -> int:
    return lib().wd_kernel_in_use(h)


def wd_kernel_for(h, nrhs: int) -> int:
    return int(lib().wd_kernel_for(h, nrhs))


def wd_launch_count(h) -> int:
    return int(lib().wd_launch_count(h))


def wd_last_error(h) -> str:
    return lib().wd_last_error(h).decode()


def wd_version() -> str:
    return lib().wd_version().decode()


def kernel_id(name: str) -> int:
    for k in range(wd_kernel_count()):
        if wd_kernel_name(k) == name:
            return k
    raise KeyError(name)
