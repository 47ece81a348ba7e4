"""Pins for the 2-D unbounded oracle (reading A28): kernels, Hockney-Eastwood solve,
gradient."""
import math

import numpy as np
import pytest
import scipy.special as sp

import oracle as O


def test_exponential_integral_and_kernel_values():
    for u in (1e-8, 1e-3, 0.1, 0.999, 1.0, 1.001, 2.5, 7.0, 40.0, 300.0):
        assert O.exp1(u) == pytest.approx(sp.exp1(u), rel=5e-15, abs=1e-300)
    eps = 0.13
    g0 = (math.log(2 * eps * eps) - np.euler_gamma) / (4 * math.pi)
    assert O.green2d_gauss(2, 0.0, eps) == pytest.approx(g0, rel=1e-15)
    assert O.green2d_gauss(2, 1e-7, eps) == pytest.approx(g0, rel=1e-10)          # continuous at the origin
    assert O.green2d_gauss(2, 9.0 * eps, eps) == pytest.approx(math.log(9.0 * eps) / (2 * math.pi), rel=1e-14)  # ln r / 2 pi outside
    # radial field: G'(r) = (1 - exp(-r^2 / 2 eps^2)) / (2 pi r)  (Gauss's law for the Gaussian charge)
    for r in (0.3 * eps, eps, 2.7 * eps):
        d = 1e-6 * eps
        num = (O.green2d_gauss(2, r + d, eps) - O.green2d_gauss(2, r - d, eps)) / (2 * d)
        assert num == pytest.approx((1 - math.exp(-r * r / (2 * eps * eps))) / (2 * math.pi * r), rel=1e-8)
    # G_P(0) = G_2(0) - (1 / 4 pi) sum_{n < P/2} 1/n   (L_n(0) = 1, g(0) = 1 / (2 pi eps^2))
    for order in (4, 6, 8, 10):
        want = g0 - sum(1.0 / n for n in range(1, order // 2)) / (4 * math.pi)
        assert O.green2d_gauss(order, 0.0, eps) == pytest.approx(want, rel=1e-14)
    # beyond a few eps every order is the free-space kernel
    for order in (2, 4, 6, 8, 10):
        assert O.green2d_gauss(order, 12 * eps, eps) == pytest.approx(math.log(12 * eps) / (2 * math.pi), rel=1e-13)


@pytest.mark.parametrize("order", [2, 6])
def test_fft_solve_is_the_direct_sum(order):
    """the definition psi_i = rhs_sign hx hy sum_j G(|x_i - x_j|) f_j by brute force, non-square anisotropic grid"""
    rng = np.random.default_rng(31)
    f = rng.normal(size=(8, 16))
    h = (0.1, 0.07)
    gh = O.unbounded2d_green((16, 8), h, 0.25, order)
    assert np.abs(gh.imag).max() < 1e-15 * np.abs(gh.real).max()       # real, even kernel
    got = O.unbounded2d_solve(f, h, gh, rhs_sign=-1.0)
    ref = O.unbounded2d_direct(f, h, 0.25, order, rhs_sign=-1.0)
    assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max()
    # a unit source returns the kernel itself
    e = np.zeros((8, 16))
    e[5, 3] = 1.0
    psi = O.unbounded2d_solve(e, h, gh)
    for (iy, ix) in ((5, 3), (0, 0), (7, 15), (5, 4), (6, 3)):
        r = math.hypot((ix - 3) * h[0], (iy - 5) * h[1])
        assert psi[iy, ix] == pytest.approx(h[0] * h[1] * O.green2d_gauss(order, r, 0.25), rel=1e-12, abs=1e-16)


def _blob_fields(n, order, eps, blobs, h):
    """closed forms for Gaussian charges q g_sigma: potential of order P and the order-2 radial field.
    Gaussians convolve to Gaussians (s^2 = sigma^2 + eps^2); term n of the order-P kernel is
    -(eps^2/2)^n / n! (-lap)^(n-1) g_eps, and lap^m g_s = (-2)^m m! / s^(2m) L_m(r^2 / 2 s^2) g_s in 2-D."""
    x = (np.arange(n) + 0.5) * h
    X, Y = x[None, :], x[:, None]
    f = np.zeros((n, n)); psi = np.zeros((n, n)); gx = np.zeros((n, n)); gy = np.zeros((n, n))
    for (cx, cy, sig, q) in blobs:
        r2 = (X - cx) ** 2 + (Y - cy) ** 2
        f += q * np.exp(-r2 / (2 * sig * sig)) / (2 * np.pi * sig * sig)
        s2 = sig * sig + eps * eps
        u = np.maximum(r2, 1e-300) / (2 * s2)
        gs = np.exp(-r2 / (2 * s2)) / (2 * np.pi * s2)
        pot = (0.5 * np.log(np.maximum(r2, 1e-300)) + 0.5 * sp.exp1(u)) / (2 * np.pi)
        for nn in range(1, order // 2):
            m = nn - 1
            pot = pot - (eps * eps / 2) ** nn / math.factorial(nn) * (2.0 ** m * math.factorial(m) / s2 ** m) * sp.eval_laguerre(m, r2 / (2 * s2)) * gs
        psi += q * pot
        dpdr_over_r = (1 - np.exp(-r2 / (2 * s2))) / (2 * np.pi * np.maximum(r2, 1e-300))
        gx += q * dpdr_over_r * (X - cx)
        gy += q * dpdr_over_r * (Y - cy)
    return f, psi, gx, gy


@pytest.mark.parametrize("order", [2, 4, 10])
def test_gaussian_charges_closed_form(order):
    n, h = 64, 1.0 / 64
    eps = 2 * h
    blobs = [(0.40, 0.55, 3.0 * h, 1.3), (0.62, 0.35, 2.5 * h, -0.7), (0.50, 0.50, 4.0 * h, 0.4)]
    f, psi_a, gx_a, gy_a = _blob_fields(n, order, eps, blobs, h)
    gh = O.unbounded2d_green((n, n), (h, h), eps, order)
    psi, grad = O.unbounded2d_solve(f, (h, h), gh, want_grad=True)
    assert np.abs(psi - psi_a).max() < 2e-9 * np.abs(psi_a).max()
    assert np.array_equal(psi, O.unbounded2d_solve(f, (h, h), gh))
    if order == 2:
        scale = max(np.abs(gx_a).max(), np.abs(gy_a).max())
        assert np.abs(grad[0] - gx_a).max() < 1e-7 * scale
        assert np.abs(grad[1] - gy_a).max() < 1e-7 * scale


# ------------------------------------------------------------------------- the spectrally compact kernel in 2-D (A30)
def test_bessel_cin_against_its_definition_and_a_bessel_series():
    """C(x) = int_0^x (1 - J0(t)) / t dt: adaptive quadrature of the definition, its derivative, the identity
    C(x) = sum_{i>=1} (2 H_i - 1/i) J_{2i}(x) with scipy's Bessel functions, and the large-argument form ln(x/2) + gamma"""
    from scipy import integrate, special

    for x in (0.0, 1e-3, 0.7, 3.0, 11.9, 12.0, 12.1, 25.0, 80.0, 303.5):
        ref = integrate.quad(lambda t: (1.0 - special.j0(t)) / t if t > 0 else 0.0, 0.0, x, limit=2000, epsabs=1e-13, epsrel=1e-13)[0] if x > 0 else 0.0
        assert abs(O.bessel_cin(x) - ref) <= 2e-12 * max(1.0, abs(ref)), x
        if x > 0:
            i = np.arange(1, int(x) + 60)
            hs = np.cumsum(1.0 / i)
            ser = float(np.sum((2.0 * hs - 1.0 / i) * special.jv(2 * i, x)))
            assert abs(O.bessel_cin(x) - ser) <= 1e-12 * max(1.0, abs(ser)), x
    for x in (2.0, 9.0, 40.0):       # d C / d x = (1 - J0(x)) / x
        d = 1e-5
        num = (O.bessel_cin(x + d) - O.bessel_cin(x - d)) / (2 * d)
        assert abs(num - (1.0 - special.j0(x)) / x) <= 1e-8
    x = 5000.0
    assert abs(O.bessel_cin(x) - (np.log(x / 2) + np.euler_gamma)) <= 2.0 / x ** 1.5


def test_spectral_kernel_2d_origin_far_field_and_quadrature_of_its_definition():
    h = 0.05
    kc = np.pi / h
    assert abs(O.green2d_spectral(0.0, h) + (np.log(kc / 2) + np.euler_gamma) / (2 * np.pi)) <= 1e-15
    r = 40.0 * h      # far field: ln r / (2 pi) up to the decaying oscillation ~ (k_c r)^(-3/2)
    assert abs(O.green2d_spectral(r, h) - np.log(r) / (2 * np.pi)) <= 1.0 / (2 * np.pi) / (kc * r) ** 1.5
    # the definition: -1/k^2 inside the disc, i.e. G(r) - G(0) = (1 / 2 pi) int_0^kc (1 - J0(k r)) / k dk
    from scipy import integrate, special
    for r in (0.3 * h, 2.0 * h, 7.5 * h):
        q = integrate.quad(lambda k: (1.0 - special.j0(k * r)) / k, 0.0, kc, limit=500, epsabs=1e-13, epsrel=1e-13)[0]
        assert abs((O.green2d_spectral(r, h) - O.green2d_spectral(0.0, h)) - q / (2 * np.pi)) <= 1e-12


def test_spectral_kernel_2d_solves_a_resolved_gaussian_charge_to_rounding():
    """a Gaussian charge whose spectrum has died out at k_c is solved exactly by the truncated kernel:
    psi = q (ln r + E1(r^2 / 2 s^2) / 2) / (2 pi) (the closed form of reading A28 with eps -> 0)"""
    from scipy import special
    n, L = 64, 1.0
    h = (L / n, L / n)
    s = 3.0 * h[0]      # spectrum e^{-(k s)^2 / 2} = 5e-20 at k_c; 9 widths from the nearest edge of the box
    x = (np.arange(n) + 0.5) * h[0]
    X, Y = np.meshgrid(x, x, indexing="xy")
    cx, cy = 0.47, 0.55
    r2 = (X - cx) ** 2 + (Y - cy) ** 2
    f = np.exp(-r2 / (2 * s * s)) / (2 * np.pi * s * s)
    gh = O.unbounded2d_green((n, n), h, 0.0, order=0)
    psi = O.unbounded2d_solve(f, h, gh)
    r = np.sqrt(r2)
    exact = (np.log(r) + 0.5 * special.exp1(r2 / (2 * s * s))) / (2 * np.pi)
    err = np.abs(psi - exact).max()
    print("2-D spectral kernel, resolved Gaussian charge: max error", err)
    assert err <= 5e-13
