"""Pins P1 / P12: every 1-D transform of the oracle against brute force, exact
special cases and library routines."""
import numpy as np
import pytest
import scipy.fft as sfft

import oracle as O

RNG = np.random.default_rng(20230101)


def _c(n):
    return RNG.normal(size=n) + 1j * RNG.normal(size=n)


def test_dft_direct_delta_pins_sign_and_index():
    # eq. (8): forward kernel exp(-2 pi i k n / N); delta at n=1 -> exp(-2 pi i k/N)
    n = 8
    x = np.zeros(n, complex)
    x[1] = 1.0
    X = O.dft_direct(x)
    k = np.arange(n)
    assert np.allclose(X.real, np.cos(2 * np.pi * k / n), atol=1e-15)
    assert np.allclose(X.imag, -np.sin(2 * np.pi * k / n), atol=1e-15)
    Xb = O.dft_direct(x, +1)
    assert np.allclose(Xb.imag, +np.sin(2 * np.pi * k / n), atol=1e-15)


@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 64, 256, 512, 1024])
def test_fft_pow2_vs_brute_force_and_library(n):
    x = _c(n)
    ref = np.fft.fft(x)
    tol = 1e-14 * max(1.0, np.log2(max(n, 2))) * np.abs(ref).max()
    assert np.abs(O.fft_pow2(x) - ref).max() <= tol
    assert np.abs(O.fft_pow2(x, +1) - np.fft.ifft(x) * n).max() <= tol
    if n <= 64:
        assert np.abs(O.fft_pow2(x) - O.dft_direct(x)).max() <= tol
        assert np.abs(O.dft_direct(x) - ref).max() <= tol


def test_fft_roundtrip_and_parseval():
    n = 128
    x = _c(n)
    X = O.fft_pow2(x)
    assert np.allclose(O.fft_pow2(X, +1) / n, x, atol=1e-13)
    assert np.isclose(np.sum(np.abs(X) ** 2) / n, np.sum(np.abs(x) ** 2), rtol=1e-13)


def test_fft_rejects_non_pow2():
    with pytest.raises(RuntimeError):
        O.fft_pow2(_c(12))


@pytest.mark.parametrize("n", [4, 7, 8, 15, 16, 255])
def test_r2r_vs_library(n):
    x = RNG.normal(size=n)
    tol = 1e-13 * n
    assert np.abs(O.dst1(x) - sfft.dst(x, type=1)).max() <= tol
    assert np.abs(O.dct2(x) - sfft.dct(x, type=2)).max() <= tol
    assert np.abs(O.dct3(x) - sfft.dct(x, type=3)).max() <= tol


@pytest.mark.parametrize("n", [7, 15, 16])
def test_r2r_eigenvectors_and_inverses(n):
    j = np.arange(n)
    for m in (1, 2, n - 1):
        # Table 1 row 1: DST-I basis sin(pi (j+1)(k+1)/(N+1)); orthogonality gives (N+1) delta
        y = O.dst1(np.sin(np.pi * (j + 1) * m / (n + 1)))
        e = np.zeros(n)
        e[m - 1] = n + 1
        assert np.abs(y - e).max() < 1e-12
        # Table 1 row 4: DCT-II basis cos(pi (j+1/2) k / N) -> N delta_k,m
        y = O.dct2(np.cos(np.pi * (j + 0.5) * m / n))
        e = np.zeros(n)
        e[m] = n
        assert np.abs(y - e).max() < 1e-12
    assert np.abs(O.dct2(np.ones(n)) - np.eye(n)[0] * 2 * n).max() < 1e-12
    x = RNG.normal(size=n)
    assert np.allclose(O.dst1(O.dst1(x)), 2 * (n + 1) * x, atol=1e-11)
    assert np.allclose(O.dct3(O.dct2(x)), 2 * n * x, atol=1e-11)
    assert np.allclose(O.dct2(O.dct3(x)), 2 * n * x, atol=1e-11)


def test_dst1_is_odd_extension_dft():
    # PAPER.md:122 "Dirichlet (odd function extension)": DFT of (0, x, 0, -reversed x) = -i * DST-I
    n = 15
    x = RNG.normal(size=n)
    ext = np.concatenate([[0.0], x, [0.0], -x[::-1]])
    E = O.fft_pow2(ext.astype(complex))
    assert np.allclose(E[1:n + 1], -1j * O.dst1(x), atol=1e-12)


def test_dct2_is_even_extension_dft():
    # PAPER.md:123 "Neumann (even function extension)": half-sample-symmetric extension
    n = 16
    x = RNG.normal(size=n)
    ext = np.concatenate([x, x[::-1]])
    E = O.fft_pow2(ext.astype(complex))
    k = np.arange(n)
    assert np.allclose(E[:n] * np.exp(-1j * np.pi * k / (2 * n)), O.dct2(x), atol=1e-12)
