"""Pins P2, P8, P9 for the periodic oracle O-PER."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from analytic import periodic2d_closed_form, rel_l2


def test_cfg1_closed_form_with_gradient():
    # P2: band-limited source => pseudo-spectral solve is exact ("spectral accuracy")
    w = W.periodic2d_modes(64)
    psi, grad = O.periodic(w["f"], w["L"], O.OP_PS, want_grad=True)
    phi, gx, gy = periodic2d_closed_form(w)
    assert np.abs(psi - phi).max() < 1e-14
    assert np.abs(grad[0] - gx).max() < 1e-13
    assert np.abs(grad[1] - gy).max() < 1e-13
    # distinct p, q per mode make a transposed axis or a swapped gradient component fail here
    assert np.abs(grad[0] - gy).max() > 1e-3


def test_cfg1_rectangular_domain_and_sign():
    w = W.periodic2d_modes(32, seed=7, kmax=4)
    psi = O.periodic(w["f"], w["L"], O.OP_PS)
    psi_m = O.periodic(w["f"], w["L"], O.OP_PS, rhs_sign=-1.0)
    assert np.array_equal(psi_m, -psi)
    # single mode on a non-square domain: f = cos(2 pi x / Lx) -> psi = -f / (2 pi / Lx)^2
    n, Lx, Ly = 16, 3.0, 0.5
    x = (np.arange(n) + 0.5) * Lx / n
    f = np.cos(2 * np.pi * x / Lx)[None, :] * np.ones((n, 1))
    psi, grad = O.periodic(f, (Lx, Ly), O.OP_PS, want_grad=True)
    assert np.abs(psi + f / (2 * np.pi / Lx) ** 2).max() < 1e-14
    assert np.abs(grad[0] - np.sin(2 * np.pi * x / Lx)[None, :] / (2 * np.pi / Lx)).max() < 1e-13
    assert np.abs(grad[1]).max() < 1e-13


def test_cfg2_ps_known_in_spectral_space():
    # P8: on [0, 2 pi)^3 the wavenumber is the integer mode m: phi_hat = -f_hat / (m.m)
    w = W.periodic3d_spectrum(32, kmax=8)
    f = w["f"]
    assert abs(f.mean()) < 1e-12 and abs(np.sqrt(np.mean(f * f)) - 1) < 1e-12
    psi, grad = O.periodic(f, w["L"], O.OP_PS, want_grad=True)
    n = f.shape[0]
    m = np.fft.fftfreq(n, 1.0 / n)
    m2 = m[:, None, None] ** 2 + m[None, :, None] ** 2 + m[None, None, :] ** 2
    fh = np.fft.fftn(f)
    m2[0, 0, 0] = 1.0
    ph = -fh / m2
    ph[0, 0, 0] = 0.0
    assert rel_l2(psi, np.fft.ifftn(ph).real) < 1e-13
    mz, my, mx = np.meshgrid(m, m, m, indexing="ij")
    for a, mm in enumerate((mx, my, mz)):
        assert rel_l2(grad[a], np.fft.ifftn(1j * mm * ph).real) < 1e-12


@pytest.mark.parametrize("shape", [(16, 16, 16), (8, 16, 32)])
def test_fd2_satisfies_the_periodic_stencil(shape):
    # P9: FD2 eigenvalues (Table 1) <=> exact zero-mean solution of the 7-point system
    rng = np.random.default_rng(5)
    f = rng.normal(size=shape)
    L = (1.0, 2.0, 0.5)
    h = [L[a] / shape[2 - a] for a in range(3)]  # shape is (z, y, x)
    psi = O.periodic(f, L, O.OP_FD2)
    lap = np.zeros_like(psi)
    for a, ax in enumerate((2, 1, 0)):
        lap += (np.roll(psi, 1, ax) - 2 * psi + np.roll(psi, -1, ax)) / h[a] ** 2
    assert np.abs(lap - (f - f.mean())).max() < 1e-10
    assert abs(psi.mean()) < 1e-14


def test_fd2_second_order_convergence():
    # north_star: "second-order convergence of the FD operator"
    errs = []
    for n in (16, 32, 64):
        x = np.arange(n) / n
        f1 = np.sin(2 * np.pi * x)
        f = f1[:, None, None] * f1[None, :, None] * f1[None, None, :]
        exact = -f / (3 * (2 * np.pi) ** 2)
        errs.append(np.abs(O.periodic(f, (1.0, 1.0, 1.0), O.OP_FD2) - exact).max())
    assert 3.8 < errs[0] / errs[1] < 4.2 and 3.9 < errs[1] / errs[2] < 4.1


def test_nyquist_mode_has_zero_spectral_derivative():
    # reading A20: i*kappa := 0 at k = N/2; the PS eigenvalue there is (pi N / L)^2 (reading A4)
    n = 16
    x = np.arange(n) / n
    f = np.cos(np.pi * n * x)[None, None, :] * np.ones((n, n, 1))
    psi, grad = O.periodic(f, (1.0, 1.0, 1.0), O.OP_PS, want_grad=True)
    assert np.abs(psi + f / (np.pi * n) ** 2).max() < 1e-15
    assert np.abs(grad).max() < 1e-15
