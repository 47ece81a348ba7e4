"""Closed forms used to pin the oracle (and, through it, the CUDA path).  Pure mathematics of the
test functions -- none of this is part of either implementation."""
import math

import numpy as np
from scipy.special import erf


def periodic2d_closed_form(w):
    """cfg 1 / pin P2: f = sum a cos(th) + b sin(th), th = 2 pi (p x + q y)
    => phi = -f_j / (4 pi^2 (p^2 + q^2)) mode by mode; gradient analytic."""
    p, q, a, b = w["modes"]
    x = w["x"]
    X, Y = np.meshgrid(x, x, indexing="xy")
    phi = np.zeros_like(X)
    gx = np.zeros_like(X)
    gy = np.zeros_like(X)
    for j in range(len(p)):
        th = 2 * np.pi * (p[j] * X + q[j] * Y)
        k2 = 4 * np.pi ** 2 * (p[j] ** 2 + q[j] ** 2)
        phi += -(a[j] * np.cos(th) + b[j] * np.sin(th)) / k2
        dth = -(-a[j] * np.sin(th) + b[j] * np.cos(th)) / k2
        gx += dth * 2 * np.pi * p[j]
        gy += dth * 2 * np.pi * q[j]
    return phi, gx, gy


def fd2_amplitude(m, h):
    """ratio (continuum eigenvalue) / (FD2 eigenvalue) for prod_a sin|cos(m_a pi x_a) on spacing h:
    the 3-point second difference of sin(m pi x) is -(4/h^2) sin^2(m pi h / 2) sin(m pi x)."""
    m = np.asarray(m, dtype=np.float64)
    return (np.pi ** 2 * np.sum(m ** 2)) / np.sum((4.0 / h ** 2) * np.sin(m * np.pi * h / 2) ** 2)


def bounded_discrete_solution(d, kind):
    """pins P3 / P4: the exact solution of the (2d+1)-point system for the manufactured source:
    A * prod + q, since the quadratic q is reproduced exactly by the second difference."""
    x = d["x"]
    m = d["m"]
    fn = np.sin if kind == "dirichlet" else np.cos
    tx, ty, tz = (fn(m[i] * np.pi * x) for i in range(3))
    prod = tz[:, None, None] * ty[None, :, None] * tx[None, None, :]
    A = fd2_amplitude(m, d["h"][0])
    q = d["u"] - prod
    return A * prod + q


def gaussian_blob_potential(g, eps, sign=-1.0):
    """pin P5: a Gaussian blob (strength q, width sigma) convolved with the Gaussian-regularised
    kernel of width eps gives  sign * q erf(r / (sqrt 2 s)) / (4 pi r),  s^2 = sigma^2 + eps^2
    (Gaussians convolve to Gaussians; the erf/r form is the potential of a Gaussian charge)."""
    x = g["x"]
    out = np.zeros((x.size,) * 3)
    for c, sig, q in zip(g["centres"], g["sigmas"], g["q"]):
        s = np.sqrt(sig ** 2 + eps ** 2)
        r = np.sqrt((x[:, None, None] - c[2]) ** 2 + (x[None, :, None] - c[1]) ** 2 + (x[None, None, :] - c[0]) ** 2)
        r = np.maximum(r, 1e-300)
        out += sign * q * erf(r / (np.sqrt(2) * s)) / (4 * np.pi * r)
    return out


def gaussian_blob_potential_gradient(g, eps, sign=-1.0):
    """gradient of the above: d/dr [erf(r/(sqrt2 s))/(4 pi r)] along (x - c)/r; returns (gx, gy, gz)"""
    x = g["x"]
    gx = np.zeros((x.size,) * 3)
    gy = np.zeros_like(gx)
    gz = np.zeros_like(gx)
    for c, sig, q in zip(g["centres"], g["sigmas"], g["q"]):
        s = np.sqrt(sig ** 2 + eps ** 2)
        dx = x[None, None, :] - c[0]
        dy = x[None, :, None] - c[1]
        dz = x[:, None, None] - c[2]
        r = np.maximum(np.sqrt(dx ** 2 + dy ** 2 + dz ** 2), 1e-300)
        dpdr = (np.sqrt(2 / np.pi) / s * np.exp(-r ** 2 / (2 * s * s)) * r - erf(r / (np.sqrt(2) * s))) / (4 * np.pi * r ** 2)
        gx += sign * q * dpdr * dx / r
        gy += sign * q * dpdr * dy / r
        gz += sign * q * dpdr * dz / r
    return gx, gy, gz


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def gaussian_blob_potential_order(g, eps, order, sign=-1.0):
    """pin for the kernels of order P = 2 .. 10 (reading A25): in spectral space the blob
    q exp(-sigma^2 k^2/2) times G^_P = -exp(-eps^2 k^2/2) sum_{n<P/2} (eps^2 k^2/2)^n / n! / k^2 is
    -q exp(-s^2 k^2/2) [1/k^2 + sum_{n>=1} (eps^2/2)^n/n! k^(2n-2)], s^2 = sigma^2 + eps^2, hence
        phi_P = -q erf(r/(sqrt2 s))/(4 pi r) - q sum_{n=1}^{P/2-1} (eps^2/2)^n/n! (-lap)^(n-1) g_s(r)
    with g_s the unit Gaussian of width s; lap^m g_s is taken here by repeated application of the
    radial Laplacian f'' + 2 f'/r to the polynomial prefactor (sympy-free, exact polynomial algebra)."""
    from numpy.polynomial import polynomial as P
    x = g["x"]
    out = gaussian_blob_potential(g, eps, sign)
    for c, sig, q in zip(g["centres"], g["sigmas"], g["q"]):
        s2 = sig ** 2 + eps ** 2
        r2 = (x[:, None, None] - c[2]) ** 2 + (x[None, :, None] - c[1]) ** 2 + (x[None, None, :] - c[0]) ** 2
        gs = (2 * np.pi * s2) ** -1.5 * np.exp(-r2 / (2 * s2))
        # f = p(t) exp(-t/(2 s2)) with t = r^2:  lap f = [4 t p'' + (6 - 4 t/(2 s2)... ] -- derived below
        # d/dr = 2 r d/dt;  f'' + 2 f'/r = 4 t f_tt + 6 f_t  (f_t = d f/dt), and with f = p e^{-a t}, a = 1/(2 s2):
        #   f_t = (p' - a p) e,  f_tt = (p'' - 2 a p' + a^2 p) e
        a = 1.0 / (2 * s2)
        p = np.array([1.0])          # polynomial in t, lowest degree first
        for n in range(1, order // 2):
            # term n uses (-lap)^(n-1) g_s
            out += sign * q * (eps ** 2 / 2) ** n / math.factorial(n) * P.polyval(r2, p) * gs
            d1, d2 = P.polyder(p), P.polyder(p, 2)
            ft = P.polysub(d1, a * p)
            ftt = P.polyadd(P.polysub(d2, 2 * a * d1), a * a * p)
            lap = P.polyadd(P.polymul([0.0, 4.0], ftt), 6.0 * ft)
            p = -lap                 # next power of (-lap)
    return out
