"""CPU oracle for the SailFFish spectral Poisson hot path -- TEST INFRASTRUCTURE ONLY.

A thin ctypes binding over ``oracle/sf_oracle.c`` (plain C, fp64, written from PAPER.md).  Nothing
under ``paper_2301_01145_b200/`` may import this package; only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs do.
The oracle and the CUDA path share no code; see the header of ``sf_oracle.c`` for the passages of
the paper each function follows and for the pins that tie it to something other than itself.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sf_oracle.c"
_LIB = _HERE / "libsf_oracle.so"

OP_PS, OP_FD2 = 0, 1


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (OpenMP over independent pencils only)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.orc_num_threads.restype = C.c_int
        L.orc_green_gauss2.restype = C.c_double
        L.orc_green_gauss2.argtypes = [C.c_double, C.c_double]
        L.orc_sine_integral.restype = C.c_double
        L.orc_sine_integral.argtypes = [C.c_double]
        L.orc_green_spectral.restype = C.c_double
        L.orc_green_spectral.argtypes = [C.c_double, C.c_double]
        L.orc_green_gauss.restype = C.c_double
        L.orc_green_gauss.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_exp1.restype = C.c_double
        L.orc_exp1.argtypes = [C.c_double]
        L.orc_green2d_gauss.restype = C.c_double
        L.orc_green2d_gauss.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_bessel_cin.restype = C.c_double
        L.orc_bessel_cin.argtypes = [C.c_double]
        L.orc_green2d_spectral.restype = C.c_double
        L.orc_green2d_spectral.argtypes = [C.c_double, C.c_double]
        L.orc_unbounded_spec_size.restype = C.c_longlong
        _lib = L
    return _lib


def _i64x3(v):
    return (C.c_longlong * 3)(*[int(x) for x in v])


def _f64x3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(err, what):
    if err != 0:
        raise RuntimeError(f"oracle: {what} failed with status {err}")


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(C.c_int(int(n)))


# ---------------------------------------------------------------- 1-D transforms (pin P1)
def dft_direct(x, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    lib().orc_dft_direct(C.c_int(x.size), C.c_int(sign), _ptr(x), _ptr(out))
    return out


def fft_pow2(x, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _chk(lib().orc_fft_pow2(C.c_int(x.size), C.c_int(sign), _ptr(x), _ptr(out)), "fft_pow2")
    return out


def _r2r(name, x):
    x = _f64(x)
    out = np.empty_like(x)
    getattr(lib(), name)(C.c_int(x.size), _ptr(x), _ptr(out))
    return out


def dst1(x):
    return _r2r("orc_dst1_direct", x)


def dct2(x):
    return _r2r("orc_dct2_direct", x)


def dct3(x):
    return _r2r("orc_dct3_direct", x)


def dst2(x):
    return _r2r("orc_dst2_direct", x)


def dst3(x):
    return _r2r("orc_dst3_direct", x)


def dct1(x):
    return _r2r("orc_dct1_direct", x)


# ---------------------------------------------------------------- solvers
def _dims(shape):
    """numpy shape (z, y, x) / (y, x) -> (nd, n[3]) with x first."""
    nd = len(shape)
    n = list(reversed(shape)) + [1] * (3 - nd)
    return nd, n


def periodic(f, L, op=OP_PS, rhs_sign=1.0, want_grad=False):
    """O-PER.  f: numpy array indexed [z, y, x] (or [y, x]); L: domain length per axis (x, y, z).
    Returns psi, or (psi, grad) with grad[a] = d psi / d x_a, a in x, y(, z) order."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    Lx = list(L) + [1.0] * (3 - len(L))
    psi = np.empty_like(f)
    grad = np.empty((nd,) + f.shape, dtype=np.float64) if want_grad else None
    _chk(lib().orc_periodic(C.c_int(nd), _i64x3(n), _f64x3(Lx), C.c_int(op), C.c_double(rhs_sign),
                            _ptr(f), _ptr(psi), _ptr(grad) if want_grad else None), "periodic")
    return (psi, grad) if want_grad else psi


def periodic_divergence(f, L, op=OP_PS, rhs_sign=1.0):
    """DIV on a periodic vector plan: f[nd, (z,) y, x] -> div psi, psi_c the solution for source f_c."""
    f = _f64(f)
    nd, n = _dims(f.shape[1:])
    assert f.shape[0] == nd
    Lx = list(L) + [1.0] * (3 - len(L))
    out = np.empty(f.shape[1:])
    _chk(lib().orc_periodic_divlap(C.c_int(nd), _i64x3(n), _f64x3(Lx), C.c_int(op), C.c_double(rhs_sign), C.c_int(nd),
                                   _ptr(f), C.c_int(0), _ptr(out)), "periodic_divergence")
    return out


def periodic_laplacian(f, L, op=OP_PS, rhs_sign=1.0, ncomp=1):
    """NABLA on a periodic plan: lap psi per component (f[(z,) y, x], or f[c, ...] with ncomp = c)."""
    f = _f64(f)
    nd, n = _dims(f.shape[1:] if ncomp > 1 else f.shape)
    Lx = list(L) + [1.0] * (3 - len(L))
    out = np.empty_like(f)
    _chk(lib().orc_periodic_divlap(C.c_int(nd), _i64x3(n), _f64x3(Lx), C.c_int(op), C.c_double(rhs_sign),
                                   C.c_int(ncomp), _ptr(f), C.c_int(1), _ptr(out)), "periodic_laplacian")
    return out


def periodic_curl(f, L, op=OP_PS, rhs_sign=1.0):
    """CURL on a periodic 3-D vector plan: f[3, z, y, x] -> u = curl psi, psi_c the solution for source f_c."""
    f = _f64(f)
    assert f.ndim == 4 and f.shape[0] == 3
    nd, n = _dims(f.shape[1:])
    out = np.empty_like(f)
    _chk(lib().orc_periodic_curl(_i64x3(n), _f64x3(list(L)), C.c_int(op), C.c_double(rhs_sign), _ptr(f), _ptr(out)),
         "periodic_curl")
    return out


def _faces_arg(faces):
    """faces: dict {(axis, side): array} or None -> (const double*[6], keepalive)."""
    arr = (C.c_void_p * 6)()
    keep = []
    if faces:
        for (axis, side), g in faces.items():
            if g is None:
                continue
            g = _f64(g)
            keep.append(g)
            arr[2 * axis + side] = g.ctypes.data
    return arr, keep


def dirichlet_regular(f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """O-DIR.  f[z, y, x] on interior nodes; h = (hx, hy, hz); faces[(axis, side)] arrays indexed
    [upper remaining axis, lower remaining axis] (lower axis fastest)."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    arr, keep = _faces_arg(faces)
    _chk(lib().orc_dirichlet_regular(_i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign), _ptr(f), arr,
                                     _ptr(psi)), "dirichlet_regular")
    return psi


def dirichlet_staggered(f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """O-DIRS.  Dirichlet on a cell-centre grid (DST-II / DST-III); conventions as dirichlet_regular."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    arr, keep = _faces_arg(faces)
    _chk(lib().orc_dirichlet_staggered(_i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign), _ptr(f), arr,
                                       _ptr(psi)), "dirichlet_staggered")
    return psi


def neumann_regular(f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """O-NEUR.  Neumann on a cell-boundary grid, boundary nodes stored (DCT-I); conventions as neumann_staggered."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    arr, keep = _faces_arg(faces)
    _chk(lib().orc_neumann_regular(_i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign), _ptr(f), arr,
                                   _ptr(psi)), "neumann_regular")
    return psi


BOUNDED_KINDS = {"dirichlet_regular": 0, "neumann_staggered": 1, "dirichlet_staggered": 2, "neumann_regular": 3}


def bounded_gradient(kind, f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """psi and its spectral gradient on a Dirichlet / Neumann plan (kind: a key of BOUNDED_KINDS):
    returns psi[z, y, x], grad[3, z, y, x] (d/dx, d/dy, d/dz)."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    grad = np.empty((3,) + f.shape)
    arr, keep = _faces_arg(faces)
    _chk(lib().orc_bounded_gradient(C.c_int(BOUNDED_KINDS[kind]), _i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign),
                                    _ptr(f), arr, _ptr(psi), _ptr(grad)), "bounded_gradient")
    return psi, grad


def neumann_staggered(f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """O-NEU.  Same conventions; face values are d psi / d x_axis along +axis on both sides."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    arr, keep = _faces_arg(faces)
    _chk(lib().orc_neumann_staggered(_i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign), _ptr(f), arr,
                                     _ptr(psi)), "neumann_staggered")
    return psi


KIND_DIRICHLET_BOUNDARY, KIND_NEUMANN_CENTRE, KIND_DIRICHLET_CENTRE, KIND_NEUMANN_BOUNDARY = 0, 1, 2, 3


def bounded_mixed(kinds_xyz, f, h, faces=None, op=OP_FD2, rhs_sign=1.0):
    """O-MIX.  Dirichlet / Neumann mixed per axis: kinds_xyz[a] selects the Table-1 row of axis a (KIND_* above;
    0 and 3 live on the cell-boundary grid, 1 and 2 on the cell-centre grid).  Conventions as the uniform solvers."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    arr, keep = _faces_arg(faces)
    kk = (C.c_int * 3)(*[int(k) for k in kinds_xyz])
    _chk(lib().orc_bounded_mixed(kk, _i64x3(n), _f64x3(h), C.c_int(op), C.c_double(rhs_sign), _ptr(f), arr, _ptr(psi)),
         "bounded_mixed")
    return psi


def green_gauss2(r, eps):
    return float(lib().orc_green_gauss2(float(r), float(eps)))


def green_gauss(order, r, eps):
    """Gaussian-regularised kernel of order 2, 4, 6, 8 or 10 at distance r."""
    return float(lib().orc_green_gauss(int(order), float(r), float(eps)))


def sine_integral(x):
    return float(lib().orc_sine_integral(float(x)))


def green_spectral(r, h):
    """Hejlesen's spectrally compact kernel -Si(pi r/h)/(2 pi^2 r) at distance r."""
    return float(lib().orc_green_spectral(float(r), float(h)))


def unbounded_green(n_xyz, h, eps, order=2):
    """Green's spectrum on the doubled grid: complex array [2 nz, 2 ny, nx + 1].
    order = 2 .. 10: Gaussian kernels of width eps; order = 0: spectrally compact kernel, eps = max(h)."""
    n = [int(v) for v in n_xyz]
    ghat = np.empty((2 * n[2], 2 * n[1], n[0] + 1), dtype=np.complex128)
    _chk(lib().orc_unbounded_green_order(_i64x3(n), _f64x3(h), C.c_double(eps), C.c_int(order), _ptr(ghat)),
         "unbounded_green")
    return ghat


def unbounded_solve(f, h, ghat, rhs_sign=1.0, want_curl=False):
    """O-UNB / O-VEC.  f[z, y, x] (scalar) or f[c, z, y, x] (ncomp fields)."""
    f = _f64(f)
    vec = f.ndim == 4
    ncomp = f.shape[0] if vec else 1
    nd, n = _dims(f.shape[1:] if vec else f.shape)
    assert nd == 3
    out = np.empty_like(f)
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == (2 * n[2], 2 * n[1], n[0] + 1)
    _chk(lib().orc_unbounded_solve(_i64x3(n), _f64x3(h), _ptr(ghat), C.c_int(ncomp), C.c_double(rhs_sign),
                                   _ptr(f), C.c_int(1 if want_curl else 0), _ptr(out)), "unbounded_solve")
    return out


def unbounded_gradient(f, h, ghat, rhs_sign=1.0):
    """scalar unbounded solve with spectral gradient: returns psi[z, y, x], grad[3, z, y, x] (d/dx, d/dy, d/dz)."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    assert nd == 3
    psi = np.empty_like(f)
    grad = np.empty((3,) + f.shape)
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == (2 * n[2], 2 * n[1], n[0] + 1)
    _chk(lib().orc_unbounded_gradient(_i64x3(n), _f64x3(h), _ptr(ghat), C.c_double(rhs_sign), _ptr(f), _ptr(psi),
                                      _ptr(grad)), "unbounded_gradient")
    return psi, grad


def unbounded_divergence(f, h, ghat, rhs_sign=1.0):
    """DIV on an unbounded vector plan: f[3, z, y, x] -> div psi[z, y, x], psi_c = rhs_sign G * f_c."""
    f = _f64(f)
    assert f.ndim == 4 and f.shape[0] == 3
    nd, n = _dims(f.shape[1:])
    out = np.empty(f.shape[1:])
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == (2 * n[2], 2 * n[1], n[0] + 1)
    _chk(lib().orc_unbounded_divlap(_i64x3(n), _f64x3(h), _ptr(ghat), C.c_int(3), C.c_double(rhs_sign), _ptr(f),
                                    C.c_int(0), _ptr(out)), "unbounded_divergence")
    return out


def unbounded_laplacian(f, h, ghat, rhs_sign=1.0):
    """NABLA on an unbounded plan: lap psi per component, f[z, y, x] or f[c, z, y, x]."""
    f = _f64(f)
    vec = f.ndim == 4
    nd, n = _dims(f.shape[1:] if vec else f.shape)
    out = np.empty_like(f)
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == (2 * n[2], 2 * n[1], n[0] + 1)
    _chk(lib().orc_unbounded_divlap(_i64x3(n), _f64x3(h), _ptr(ghat), C.c_int(f.shape[0] if vec else 1),
                                    C.c_double(rhs_sign), _ptr(f), C.c_int(1), _ptr(out)), "unbounded_laplacian")
    return out


def exp1(u):
    return float(lib().orc_exp1(float(u)))


def green2d_gauss(order, r, eps):
    """2-D Gaussian-regularised kernel of order 2 .. 10 at distance r (reading A28)."""
    return float(lib().orc_green2d_gauss(int(order), float(r), float(eps)))


def _i64x2(n):
    return (C.c_longlong * 2)(int(n[0]), int(n[1]))


def _f64x2(h):
    return (C.c_double * 2)(float(h[0]), float(h[1]))


def bessel_cin(x):
    """C(x) = int_0^x (1 - J0(t)) / t dt"""
    return float(lib().orc_bessel_cin(float(x)))


def green2d_spectral(r, h):
    """the 2-D spectrally compact kernel (C(pi r / h) - ln(pi / 2h) - gamma) / (2 pi) at distance r (reading A30)"""
    return float(lib().orc_green2d_spectral(float(r), float(h)))


def unbounded2d_green(n_xy, h, eps, order=2):
    """Green's spectrum on the doubled 2-D grid: complex array [2 ny, nx + 1]."""
    n = [int(v) for v in n_xy]
    ghat = np.empty((2 * n[1], n[0] + 1), dtype=np.complex128)
    _chk(lib().orc_unbounded2d_green(_i64x2(n), _f64x2(h), C.c_double(eps), C.c_int(order), _ptr(ghat)), "unbounded2d_green")
    return ghat


def unbounded2d_solve(f, h, ghat, rhs_sign=1.0, want_grad=False):
    """O-UNB2.  f[y, x]; returns psi, or (psi, grad[2, y, x]) with grad = (d/dx, d/dy)."""
    f = _f64(f)
    assert f.ndim == 2
    n = (f.shape[1], f.shape[0])
    psi = np.empty_like(f)
    grad = np.empty((2,) + f.shape) if want_grad else None
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == (2 * n[1], n[0] + 1)
    _chk(lib().orc_unbounded2d_solve(_i64x2(n), _f64x2(h), _ptr(ghat), C.c_double(rhs_sign), _ptr(f), _ptr(psi),
                                     _ptr(grad) if want_grad else None), "unbounded2d_solve")
    return (psi, grad) if want_grad else psi


def unbounded2d_direct(f, h, eps, order=2, rhs_sign=1.0):
    """Direct O(N^4) sum of the 2-D definition -- tiny grids only."""
    f = _f64(f)
    n = (f.shape[1], f.shape[0])
    psi = np.empty_like(f)
    lib().orc_unbounded2d_direct(_i64x2(n), _f64x2(h), C.c_double(eps), C.c_int(order), C.c_double(rhs_sign), _ptr(f), _ptr(psi))
    return psi


def unbounded_direct(f, h, eps, rhs_sign=1.0):
    """Direct O(N^6) sum of the definition -- tiny grids only."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    psi = np.empty_like(f)
    lib().orc_unbounded_direct(_i64x3(n), _f64x3(h), C.c_double(eps), C.c_double(rhs_sign), _ptr(f), _ptr(psi))
    return psi


def unbounded_direct_samples(f, h, eps, idx, rhs_sign=1.0):
    """Direct sum of the definition at the linear grid indices ``idx`` (x fastest)."""
    f = _f64(f)
    nd, n = _dims(f.shape)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    psi = np.empty(idx.size, dtype=np.float64)
    lib().orc_unbounded_direct_samples(_i64x3(n), _f64x3(h), C.c_double(eps), C.c_double(rhs_sign), _ptr(f),
                                       C.c_longlong(idx.size), _ptr(idx), _ptr(psi))
    return psi
