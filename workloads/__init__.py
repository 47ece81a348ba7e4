"""Seeded synthetic inputs shaped like the paper's workloads.

This module is shared by the CPU oracle's tests and the CUDA path's tests / bench.  It holds NONE of
the method's arithmetic (no transforms of the solve, no eigenvalues, no Green's functions): only the
random-number generator and the analytic source fields.  Everything is built in float64; callers
round to float32 where a plan is fp32.

Random numbers: a counter-based generator (splitmix64 finaliser applied to ``seed * 2^32 + stream *
2^24-ish + index``), uniforms from the top 53 bits, normals by Box-Muller.  It is self-contained so
that streams do not depend on the numpy version.

Arrays are indexed [z, y, x] (x fastest in memory), vector fields [component, z, y, x].
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


class Rng:
    """Counter-based stream: draw k values -> counters [pos, pos + k)."""

    def __init__(self, seed: int):
        self.base = np.uint64((int(seed) * 0x1000003D + 0x51ED27) & 0xFFFFFFFFFFFFFFFF)
        self.pos = 0

    def _bits(self, k: int) -> np.ndarray:
        idx = np.arange(self.pos, self.pos + k, dtype=np.uint64)
        self.pos += k
        with np.errstate(over="ignore"):
            return _splitmix64(_splitmix64(idx ^ self.base) + idx)

    def uniform(self, k: int = 1, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
        u = ((self._bits(k) >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u

    def integers(self, k: int, lo: int, hi: int) -> np.ndarray:
        """uniform integers in [lo, hi] inclusive"""
        return lo + np.floor(self.uniform(k) * (hi - lo + 1)).astype(np.int64)

    def normal(self, k: int = 1) -> np.ndarray:
        u1 = self.uniform(k)
        u2 = self.uniform(k)
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def seed_for(config: int) -> int:
    return 1000 + int(config)


# ------------------------------------------------------------------------------------------------
# config 1: 2-D periodic, [0,1)^2, cell-centre, sum of 8 Fourier modes, mean removed
# ------------------------------------------------------------------------------------------------
def periodic2d_modes(n: int = 64, seed: int | None = None, nmodes: int = 8, kmax: int = 8):
    rng = Rng(seed_for(1) if seed is None else seed)
    p = rng.integers(nmodes, 1, kmax)
    q = rng.integers(nmodes, 1, kmax)
    a = rng.normal(nmodes)
    b = rng.normal(nmodes)
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")  # arrays [y, x]
    f = np.zeros((n, n))
    for j in range(nmodes):
        th = 2.0 * np.pi * (p[j] * X + q[j] * Y)
        f += a[j] * np.cos(th) + b[j] * np.sin(th)
    f -= f.mean()
    return {"f": f, "L": (1.0, 1.0), "n": (n, n), "x": x, "modes": (p, q, a, b)}


# ------------------------------------------------------------------------------------------------
# config 2: 3-D periodic, [0,2pi)^3, random-phase field with |f_k| ~ |k|^-2 up to kmax, unit rms
# ------------------------------------------------------------------------------------------------
def periodic3d_spectrum(n: int = 256, seed: int | None = None, kmax: int = 64):
    rng = Rng(seed_for(2) if seed is None else seed)
    w = rng.normal(n * n * n).reshape(n, n, n)
    wh = np.fft.fftn(w)  # generation only: any FFT may be used to draw the random phases
    del w
    m = np.fft.fftfreq(n, 1.0 / n)
    m2 = m[:, None, None] ** 2 + m[None, :, None] ** 2 + m[None, None, :] ** 2
    mask = (m2 >= 1.0) & (m2 <= float(kmax) ** 2)
    amp = np.zeros_like(m2)
    amp[mask] = 1.0 / m2[mask]
    mag = np.abs(wh)
    mag[mag == 0.0] = 1.0
    fh = wh / mag * amp
    del wh, mag, amp
    f = np.fft.ifftn(fh).real
    f -= f.mean()
    f /= np.sqrt(np.mean(f * f))
    L = 2.0 * np.pi
    return {"f": np.ascontiguousarray(f), "L": (L, L, L), "n": (n, n, n)}


# ------------------------------------------------------------------------------------------------
# config 3: Dirichlet (cell-boundary, interior nodes) and Neumann (cell-centre) on [0,1]^3:
# manufactured product of sines / cosines plus a smooth quadratic carrying the boundary values
# (eq. (12), (14), (15))
# ------------------------------------------------------------------------------------------------
def _bounded_params(seed):
    rng = Rng(seed)
    m = rng.integers(3, 1, 16)
    a = rng.uniform(3, -1.0, 1.0)
    b = rng.uniform(3, -1.0, 1.0)
    return m, a, b


def _quad(xs, a, b):
    """q(x) = sum_a a_a (1 - x_a)^2 + b_a x_a^2 on the tensor grid, array [z, y, x]"""
    qx = a[0] * (1 - xs[0]) ** 2 + b[0] * xs[0] ** 2
    qy = a[1] * (1 - xs[1]) ** 2 + b[1] * xs[1] ** 2
    qz = a[2] * (1 - xs[2]) ** 2 + b[2] * xs[2] ** 2
    return qz[:, None, None] + qy[None, :, None] + qx[None, None, :]


def dirichlet3d_manufactured(nc: int = 256, seed: int | None = None, inhomogeneous: bool = True, modes=None):
    """Interior nodes x_j = (j+1) h, j < nc-1, h = 1/nc.  Faces carry q on the boundary nodes.
    ``modes`` overrides the drawn (m_x, m_y, m_z) (convergence studies on coarse grids)."""
    m, a, b = _bounded_params(seed_for(3) if seed is None else seed)
    if modes is not None:
        m = np.asarray(modes, dtype=np.int64)
    if not inhomogeneous:
        a = np.zeros(3)
        b = np.zeros(3)
    n = nc - 1
    h = 1.0 / nc
    x = (np.arange(n) + 1.0) * h
    xs = (x, x, x)
    sx, sy, sz = (np.sin(m[i] * np.pi * x) for i in range(3))
    prod = sz[:, None, None] * sy[None, :, None] * sx[None, None, :]
    u = prod + _quad(xs, a, b)
    f = -(np.pi ** 2) * float(np.sum(m ** 2)) * prod + 2.0 * float(np.sum(a + b))
    faces = {}
    if inhomogeneous:
        for axis in range(3):
            rem = [i for i in range(3) if i != axis]  # lower remaining axis first
            for side in (0, 1):
                xb = float(side)
                qa = a[axis] * (1 - xb) ** 2 + b[axis] * xb ** 2
                q_lo = a[rem[0]] * (1 - x) ** 2 + b[rem[0]] * x ** 2
                q_hi = a[rem[1]] * (1 - x) ** 2 + b[rem[1]] * x ** 2
                faces[(axis, side)] = qa + q_hi[:, None] + q_lo[None, :]  # [upper rem, lower rem]
    return {"f": f, "u": u, "faces": faces, "h": (h, h, h), "n": (n, n, n), "m": m, "a": a, "b": b, "x": x}


def neumann3d_manufactured(nc: int = 256, seed: int | None = None, inhomogeneous: bool = True, modes=None):
    """Cell centres x_j = (j+1/2) h.  Faces carry d q / d x_axis (along +axis) on both sides."""
    m, a, b = _bounded_params(seed_for(3) if seed is None else seed)
    if modes is not None:
        m = np.asarray(modes, dtype=np.int64)
    if not inhomogeneous:
        a = np.zeros(3)
        b = np.zeros(3)
    n = nc
    h = 1.0 / nc
    x = (np.arange(n) + 0.5) * h
    xs = (x, x, x)
    cx, cy, cz = (np.cos(m[i] * np.pi * x) for i in range(3))
    prod = cz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    u = prod + _quad(xs, a, b)
    f = -(np.pi ** 2) * float(np.sum(m ** 2)) * prod + 2.0 * float(np.sum(a + b))
    faces = {}
    if inhomogeneous:
        for axis in range(3):
            faces[(axis, 0)] = np.full((n, n), -2.0 * a[axis])
            faces[(axis, 1)] = np.full((n, n), +2.0 * b[axis])
    else:
        f = f - f.mean()
    return {"f": f, "u": u, "faces": faces, "h": (h, h, h), "n": (n, n, n), "m": m, "a": a, "b": b, "x": x}


def dirichlet3d_centre_manufactured(nc: int = 256, seed: int | None = None, inhomogeneous: bool = True, modes=None):
    """The Dirichlet problem of config 3 on a cell-centre grid (Table 1 row 2): x_j = (j+1/2) h, j < nc,
    h = 1/nc; faces carry u = q on the domain faces x_a = 0, 1 at the cell centres of the other two axes."""
    m, a, b = _bounded_params(seed_for(3) if seed is None else seed)
    if modes is not None:
        m = np.asarray(modes, dtype=np.int64)
    if not inhomogeneous:
        a = np.zeros(3)
        b = np.zeros(3)
    n = nc
    h = 1.0 / nc
    x = (np.arange(n) + 0.5) * h
    xs = (x, x, x)
    sx, sy, sz = (np.sin(m[i] * np.pi * x) for i in range(3))
    prod = sz[:, None, None] * sy[None, :, None] * sx[None, None, :]
    u = prod + _quad(xs, a, b)
    f = -(np.pi ** 2) * float(np.sum(m ** 2)) * prod + 2.0 * float(np.sum(a + b))
    faces = {}
    if inhomogeneous:
        for axis in range(3):
            rem = [i for i in range(3) if i != axis]
            for side in (0, 1):
                xb = float(side)
                qa = a[axis] * (1 - xb) ** 2 + b[axis] * xb ** 2
                q_lo = a[rem[0]] * (1 - x) ** 2 + b[rem[0]] * x ** 2
                q_hi = a[rem[1]] * (1 - x) ** 2 + b[rem[1]] * x ** 2
                faces[(axis, side)] = qa + q_hi[:, None] + q_lo[None, :]
    return {"f": f, "u": u, "faces": faces, "h": (h, h, h), "n": (n, n, n), "m": m, "a": a, "b": b, "x": x}


def neumann3d_boundary_manufactured(nc: int = 256, seed: int | None = None, inhomogeneous: bool = True, modes=None):
    """The Neumann problem of config 3 on a cell-boundary grid (Table 1 row 3): nodes x_j = j h, j <= nc,
    h = 1/nc, boundary nodes stored (nc + 1 per axis); faces carry d q / d x_axis (along +axis)."""
    m, a, b = _bounded_params(seed_for(3) if seed is None else seed)
    if modes is not None:
        m = np.asarray(modes, dtype=np.int64)
    if not inhomogeneous:
        a = np.zeros(3)
        b = np.zeros(3)
    n = nc + 1
    h = 1.0 / nc
    x = np.arange(n) * h
    xs = (x, x, x)
    cx, cy, cz = (np.cos(m[i] * np.pi * x) for i in range(3))
    prod = cz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    u = prod + _quad(xs, a, b)
    f = -(np.pi ** 2) * float(np.sum(m ** 2)) * prod + 2.0 * float(np.sum(a + b))
    faces = {}
    if inhomogeneous:
        for axis in range(3):
            faces[(axis, 0)] = np.full((n, n), -2.0 * a[axis])
            faces[(axis, 1)] = np.full((n, n), +2.0 * b[axis])
    return {"f": f, "u": u, "faces": faces, "h": (h, h, h), "n": (n, n, n), "m": m, "a": a, "b": b, "x": x}


# ------------------------------------------------------------------------------------------------
# config 4: unbounded, [0,1]^3 cell-centre, 16 Gaussian blobs
# ------------------------------------------------------------------------------------------------
def gaussian_blobs(n: int = 256, seed: int | None = None, nblobs: int = 16, sigma_h=(2.0, 6.0),
                   inner=(0.2, 0.8)):
    rng = Rng(seed_for(4) if seed is None else seed)
    h = 1.0 / n
    centres = np.empty((nblobs, 3))
    sigmas = np.empty(nblobs)
    q = np.empty(nblobs)
    for bidx in range(nblobs):
        centres[bidx] = rng.uniform(3, inner[0], inner[1])
        sigmas[bidx] = rng.uniform(1, sigma_h[0] * h, sigma_h[1] * h)[0]
        q[bidx] = rng.normal(1)[0]
    x = (np.arange(n) + 0.5) * h
    f = np.zeros((n, n, n))
    for bidx in range(nblobs):
        s = sigmas[bidx]
        gx = np.exp(-((x - centres[bidx, 0]) ** 2) / (2 * s * s))
        gy = np.exp(-((x - centres[bidx, 1]) ** 2) / (2 * s * s))
        gz = np.exp(-((x - centres[bidx, 2]) ** 2) / (2 * s * s))
        f += q[bidx] * (2 * np.pi * s * s) ** -1.5 * (gz[:, None, None] * gy[None, :, None] * gx[None, None, :])
    return {"f": f, "h": (h, h, h), "n": (n, n, n), "x": x, "centres": centres, "sigmas": sigmas, "q": q}


# ------------------------------------------------------------------------------------------------
# config 5: Gaussian-core vortex ring, [0,1]^3 cell-centre, radius 0.25, core sigma = 4h,
# axis = z with a seeded +-5 % tilt
# ------------------------------------------------------------------------------------------------
def vortex_ring(n: int = 512, seed: int | None = None, radius: float = 0.25, sigma_h: float = 4.0,
                gamma: float = 1.0, tilt: float = 0.05):
    rng = Rng(seed_for(5) if seed is None else seed)
    t = rng.uniform(2, -tilt, tilt)
    axis = np.array([t[0], t[1], 1.0])
    axis /= np.linalg.norm(axis)
    h = 1.0 / n
    sigma = sigma_h * h
    x = (np.arange(n) + 0.5) * h - 0.5
    omega = np.empty((3, n, n, n))
    X = x[None, None, :]
    Y = x[None, :, None]
    for iz in range(n):  # plane by plane keeps the temporaries small
        Z = x[iz]
        zp = X * axis[0] + Y * axis[1] + Z * axis[2]          # coordinate along the ring axis
        rx, ry, rz = X - zp * axis[0], Y - zp * axis[1], Z - zp * axis[2]  # radial vector
        rho = np.sqrt(rx * rx + ry * ry + rz * rz)
        mag = gamma / (2 * np.pi * sigma * sigma) * np.exp(-((rho - radius) ** 2 + zp * zp) / (2 * sigma * sigma))
        rho_s = np.where(rho > 0, rho, 1.0)
        # e_theta = axis x e_rho
        ex, ey, ez = rx / rho_s, ry / rho_s, rz / rho_s
        omega[0, iz] = (mag * (axis[1] * ez - axis[2] * ey))[0]
        omega[1, iz] = (mag * (axis[2] * ex - axis[0] * ez))[0]
        omega[2, iz] = (mag * (axis[0] * ey - axis[1] * ex))[0]
    return {"omega": omega, "h": (h, h, h), "n": (n, n, n), "axis": axis, "radius": radius, "sigma": sigma,
            "gamma": gamma}
