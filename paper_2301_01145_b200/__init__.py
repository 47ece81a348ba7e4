"""paper_2301_01145_b200 -- thin Python binding of the B200-native spectral Poisson hot path.

Argument marshalling only: every step of the path (forward transforms, multiply, spectral
differentiation, backward transforms) runs in the CUDA kernels of
``libsailffish_b200.so`` behind the C ABI declared in ``include/sailffish.h``.  The functions here
carry the same names as the C entry points.  PyTorch is used for device memory and streams only.

There is NO CPU fallback: if the shared library is missing or cannot be loaded, importing
``lib()`` raises, and so does every call.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libsailffish_b200.so"

# enums of include/sailffish.h
SF_OK, SF_ERR_INVALID_ARG, SF_ERR_UNSUPPORTED, SF_ERR_ALLOC, SF_ERR_CUDA, SF_ERR_STATE = 0, -1, -2, -3, -4, -5
SF_BC_PERIODIC, SF_BC_DIRICHLET, SF_BC_NEUMANN, SF_BC_UNBOUNDED = 0, 1, 2, 3
SF_GRID_CELL_BOUNDARY, SF_GRID_CELL_CENTRE = 0, 1
SF_OP_PSEUDO_SPECTRAL, SF_OP_FD2, SF_OP_GREEN_GAUSS2, SF_OP_GREEN_GAUSS4, SF_OP_GREEN_GAUSS6 = 0, 1, 2, 3, 4
SF_OP_GREEN_GAUSS8, SF_OP_GREEN_GAUSS10, SF_OP_GREEN_SPECTRAL = 5, 6, 7
SF_F32, SF_F64 = 0, 1
SF_MEM_HOST, SF_MEM_DEVICE = 0, 1
SF_OUT_PSI, SF_OUT_GRAD, SF_OUT_CURL, SF_OUT_DIV, SF_OUT_LAP = 0, 1, 2, 3, 4

# every symbol include/sailffish.h declares (checked by tests/test_abi.py against the header text)
EXPORTS = (
    "sf_plan_create", "sf_set_source", "sf_set_bc_values", "sf_solve", "sf_gradient", "sf_curl",
    "sf_divergence", "sf_laplacian", "sf_get_output", "sf_output_device_ptr", "sf_synchronize",
    "sf_set_pipeline", "sf_get_output_async", "sf_pipeline_join", "sf_probe_dft16_stage", "sf_last_launch_count", "sf_device_bytes",
    "sf_enable_step_timing", "sf_step_times_ms", "sf_set_step_timing_stride", "sf_last_error", "sf_plan_destroy", "sf_version",
    "sf_periodic2d_solve_static", "sf_static_last_error",
)


class sf_options(C.Structure):
    _fields_ = [("ncomp", C.c_int), ("stream", C.c_void_p), ("rhs_sign", C.c_double), ("eps_over_h", C.c_double)]


class SailffishError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"sailffish status {status}: {message}")
        self.status = status


_lib = None


def lib() -> C.CDLL:
    """Load the C-ABI library (built in-tree by ``_build.build()``); fail loudly if it is absent."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2301_01145_b200._build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, i, ll = C.c_void_p, C.c_int, C.c_longlong
        L.sf_plan_create.argtypes = [C.POINTER(vp), i, C.POINTER(ll), C.POINTER(C.c_double), C.POINTER(i), i, i, i,
                                     C.POINTER(sf_options)]
        L.sf_set_source.argtypes = [vp, vp, i]
        L.sf_set_bc_values.argtypes = [vp, i, i, vp, i]
        L.sf_solve.argtypes = [vp]
        L.sf_gradient.argtypes = [vp]
        L.sf_curl.argtypes = [vp]
        L.sf_divergence.argtypes = [vp]
        L.sf_laplacian.argtypes = [vp]
        L.sf_get_output.argtypes = [vp, i, i, vp, i]
        L.sf_output_device_ptr.argtypes = [vp, i, i, C.POINTER(vp)]
        L.sf_synchronize.argtypes = [vp]
        L.sf_set_pipeline.argtypes = [vp, i]
        L.sf_get_output_async.argtypes = [vp, i, i, vp]
        L.sf_pipeline_join.argtypes = [vp]
        L.sf_probe_dft16_stage.argtypes = [i, i, i, vp, vp, C.POINTER(C.c_float)]
        L.sf_last_launch_count.argtypes = [vp]
        L.sf_device_bytes.argtypes = [vp]
        L.sf_device_bytes.restype = ll
        L.sf_enable_step_timing.argtypes = [vp, i]
        L.sf_step_times_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.sf_set_step_timing_stride.argtypes = [vp, i]
        L.sf_last_error.argtypes = [vp]
        L.sf_last_error.restype = C.c_char_p
        L.sf_plan_destroy.argtypes = [vp]
        L.sf_version.restype = C.c_char_p
        L.sf_periodic2d_solve_static.argtypes = [C.POINTER(ll), C.POINTER(C.c_double), i, vp, vp, vp]
        L.sf_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(plan, status: int):
    if status != SF_OK:
        msg = lib().sf_last_error(plan)
        raise SailffishError(status, msg.decode() if msg else "")


def _addr(buf):
    """(address, memory space) of a torch tensor, numpy array or raw int device pointer."""
    if buf is None:
        return None, SF_MEM_HOST
    if isinstance(buf, int):
        return buf, SF_MEM_DEVICE
    if hasattr(buf, "data_ptr"):  # torch tensor
        if not buf.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return buf.data_ptr(), (SF_MEM_DEVICE if buf.is_cuda else SF_MEM_HOST)
    if hasattr(buf, "ctypes"):  # numpy
        if not buf.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return buf.ctypes.data, SF_MEM_HOST
    raise TypeError(f"unsupported buffer type {type(buf)}")


def sf_version() -> str:
    return lib().sf_version().decode()


def sf_plan_create(n, h, bc, grid=SF_GRID_CELL_CENTRE, op=SF_OP_PSEUDO_SPECTRAL, prec=SF_F32, ncomp=1, stream=None,
                   rhs_sign=1.0, eps_over_h=0.0):
    """n, h: per-axis (x, y[, z]); bc: one value or one per axis.  Returns the opaque plan handle."""
    n = [int(v) for v in n]
    ndim = len(n)
    h = [float(v) for v in h]
    if isinstance(bc, int):
        bc = [bc] * ndim
    n3 = (C.c_longlong * 3)(*(n + [1] * (3 - ndim)))
    h3 = (C.c_double * 3)(*(h + [1.0] * (3 - ndim)))
    b3 = (C.c_int * 3)(*(list(bc) + [bc[0]] * (3 - ndim)))
    opt = sf_options(int(ncomp), C.c_void_p(int(stream) if stream else 0), float(rhs_sign), float(eps_over_h))
    plan = C.c_void_p()
    st = lib().sf_plan_create(C.byref(plan), ndim, n3, h3, b3, int(grid), int(op), int(prec), C.byref(opt))
    _check(None, st)
    return plan


def sf_set_source(plan, src):
    a, where = _addr(src)
    _check(plan, lib().sf_set_source(plan, a, where))


def sf_set_bc_values(plan, axis, side, face):
    a, where = _addr(face)
    _check(plan, lib().sf_set_bc_values(plan, int(axis), int(side), a, where))


def sf_solve(plan):
    _check(plan, lib().sf_solve(plan))


def sf_gradient(plan):
    _check(plan, lib().sf_gradient(plan))


def sf_curl(plan):
    _check(plan, lib().sf_curl(plan))


def sf_divergence(plan):
    _check(plan, lib().sf_divergence(plan))


def sf_laplacian(plan):
    _check(plan, lib().sf_laplacian(plan))


def sf_get_output(plan, field, comp, dst):
    a, where = _addr(dst)
    _check(plan, lib().sf_get_output(plan, int(field), int(comp), a, where))


def sf_output_device_ptr(plan, field, comp) -> int:
    p = C.c_void_p()
    _check(plan, lib().sf_output_device_ptr(plan, int(field), int(comp), C.byref(p)))
    return int(p.value)


def sf_synchronize(plan):
    _check(plan, lib().sf_synchronize(plan))


def sf_set_pipeline(plan, depth=2):
    _check(plan, lib().sf_set_pipeline(plan, int(depth)))


def sf_get_output_async(plan, field, comp, dst):
    a, where = _addr(dst)
    if where != SF_MEM_HOST:
        raise ValueError("sf_get_output_async copies to host memory")
    _check(plan, lib().sf_get_output_async(plan, int(field), int(comp), a))


def sf_probe_dft16_stage(variant, reps, ntiles, src, dst) -> float:
    """(see include/sailffish.h) returns the device time of one launch in milliseconds"""
    a, wa = _addr(src)
    b, wb = _addr(dst)
    if wa != SF_MEM_DEVICE or wb != SF_MEM_DEVICE:
        raise ValueError("the probe works on device buffers")
    ms = C.c_float(0.0)
    _check(None, lib().sf_probe_dft16_stage(int(variant), int(reps), int(ntiles), a, b, C.byref(ms)))
    return float(ms.value)


SF_STATIC_MAX_N = 256


def sf_periodic2d_solve_static(n, h, op, src, psi, stream=None):
    """(see include/sailffish.h) periodic 2-D fp64 solve on device buffers without any allocation"""
    a, wa = _addr(src)
    b, wb = _addr(psi)
    if wa != SF_MEM_DEVICE or wb != SF_MEM_DEVICE:
        raise ValueError("sf_periodic2d_solve_static works on device buffers")
    nn = (C.c_longlong * 2)(int(n[0]), int(n[1]))
    hh = (C.c_double * 2)(float(h[0]), float(h[1]))
    st = lib().sf_periodic2d_solve_static(nn, hh, int(op), a, b, C.c_void_p(stream or 0))
    if st != SF_OK:
        raise SailffishError(st, lib().sf_static_last_error().decode())


def sf_pipeline_join(plan):
    _check(plan, lib().sf_pipeline_join(plan))


def sf_last_launch_count(plan) -> int:
    return int(lib().sf_last_launch_count(plan))


def sf_device_bytes(plan) -> int:
    return int(lib().sf_device_bytes(plan))


def sf_enable_step_timing(plan, slots=1):
    _check(plan, lib().sf_enable_step_timing(plan, int(slots)))


def sf_set_step_timing_stride(plan, stride=1):
    _check(plan, lib().sf_set_step_timing_stride(plan, int(stride)))


def sf_step_times_ms(plan):
    ms = (C.c_float * 5)()
    _check(plan, lib().sf_step_times_ms(plan, ms))
    return [float(v) for v in ms]


def sf_last_error(plan=None) -> str:
    msg = lib().sf_last_error(plan)
    return msg.decode() if msg else ""


def sf_plan_destroy(plan):
    if plan is not None:
        lib().sf_plan_destroy(plan)
