"""Pins for the DIV and NABLA operators of the oracle (reading A27): closed
forms the mathematics fixes, chosen so that a dropped term, a wrong sign or a swapped axis fails one."""
import numpy as np

import oracle as O
import workloads as W
from analytic import gaussian_blob_potential_gradient


def _grid(n, L):
    return [np.arange(m) * (l / m) for m, l in zip(n, L)]


def test_periodic_divergence_of_plane_wave_potentials():
    """psi_c = A_c sin(kappa . x + phi_c): lap psi_c = -|kappa|^2 psi_c is the source, and
    div psi = sum_c A_c kappa_c cos(kappa . x + phi_c); three different amplitudes, phases and
    wavenumbers per axis on a non-cubic box, pseudo-spectral operator -> exact to rounding."""
    n = (32, 16, 8)          # x, y, z
    L = (2.0, 1.0, 3.0)
    x, y, z = _grid(n, L)
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
    m = (3, -2, 1)
    kap = [2 * np.pi * m[a] / L[a] for a in range(3)]
    ph = kap[0] * X + kap[1] * Y + kap[2] * Z
    A, phi = (0.7, -1.3, 0.4), (0.1, 0.9, -0.5)
    k2 = sum(k * k for k in kap)
    f = np.stack([-k2 * A[c] * np.sin(ph + phi[c]) for c in range(3)])
    want = sum(A[c] * kap[c] * np.cos(ph + phi[c]) for c in range(3))
    got = O.periodic_divergence(f, L, O.OP_PS)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    # rhs_sign flips the result; a single component reduces to the matching gradient component
    assert np.allclose(O.periodic_divergence(f, L, O.OP_PS, rhs_sign=-1.0), -want, rtol=0, atol=1e-12 * np.abs(want).max())
    for c in range(3):
        fc = np.zeros_like(f)
        fc[c] = f[c]
        _, grad = O.periodic(f[c], L, O.OP_PS, want_grad=True)
        assert np.abs(O.periodic_divergence(fc, L, O.OP_PS) - grad[c]).max() <= 1e-13 * np.abs(grad[c]).max()


def test_periodic_divergence_2d():
    n, L = (16, 32), (1.0, 2.0)
    x, y = _grid(n, L)
    X, Y = x[None, :], y[:, None]
    kx, ky = 2 * np.pi * 2 / L[0], 2 * np.pi * 5 / L[1]
    ph = kx * X + ky * Y
    f = np.stack([-(kx * kx + ky * ky) * np.sin(ph), -(kx * kx + ky * ky) * 0.5 * np.cos(ph)])
    want = kx * np.cos(ph) - 0.5 * ky * np.sin(ph)
    got = O.periodic_divergence(f, L, O.OP_PS)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()


def test_periodic_laplacian_returns_the_source():
    """pseudo-spectral: lap(lap^-1 f) = f - mean(f) for a band-limited source; the Nyquist plane, which
    i kappa drops (reading A20), is dropped twice (reading A27)"""
    w = W.periodic3d_spectrum(32, kmax=8)
    f = w["f"] + 0.37                       # a mean the zero mode removes
    got = O.periodic_laplacian(f, w["L"], O.OP_PS)
    assert np.abs(got - w["f"]).max() <= 1e-12 * np.abs(w["f"]).max()
    assert np.allclose(O.periodic_laplacian(f, w["L"], O.OP_PS, rhs_sign=-1.0), -w["f"], rtol=0, atol=1e-12 * np.abs(w["f"]).max())
    nyq = np.cos(np.pi * np.arange(32))[None, None, :] * np.ones((32, 32, 1))
    got = O.periodic_laplacian(w["f"] + nyq, w["L"], O.OP_PS)
    assert np.abs(got - w["f"]).max() <= 1e-12 * np.abs(w["f"]).max()
    # vector input = component by component
    f3 = np.stack([w["f"], 2.0 * w["f"][::-1].copy(), -w["f"].transpose(1, 0, 2).copy()])
    got = O.periodic_laplacian(f3, w["L"], O.OP_PS, ncomp=3)
    for c in range(3):
        assert np.array_equal(got[c], O.periodic_laplacian(f3[c], w["L"], O.OP_PS))


def test_periodic_laplacian_fd2_filter():
    """FD2 operator: a single mode comes back scaled by sum kappa_a^2 / sum (4/h_a^2) sin^2(kappa_a h_a / 2)"""
    n, L = (16, 8, 32), (1.0, 2.0, 1.5)
    x, y, z = _grid(n, L)
    m = (3, 1, -5)
    kap = [2 * np.pi * m[a] / L[a] for a in range(3)]
    h = [L[a] / n[a] for a in range(3)]
    f = np.cos(kap[0] * x[None, None, :] + kap[1] * y[None, :, None] + kap[2] * z[:, None, None] + 0.3)
    fac = sum(k * k for k in kap) / sum(4 / h[a] ** 2 * np.sin(kap[a] * h[a] / 2) ** 2 for a in range(3))
    got = O.periodic_laplacian(f, L, O.OP_FD2)
    assert fac > 1.0
    assert np.abs(got - fac * f).max() <= 1e-12 * fac


def test_unbounded_laplacian_of_a_gaussian_charge():
    """lap(G_eps * f) = zeta_eps * f: a Gaussian charge of width sigma comes back as the Gaussian of width
    s, s^2 = sigma^2 + eps^2 (the regularised kernel is the potential of the unit Gaussian zeta_eps)"""
    n = 64
    g = W.gaussian_blobs(n, nblobs=3, sigma_h=(2.5, 3.5), inner=(0.3, 0.7))
    eps = 2 * g["h"][0]
    gh = O.unbounded_green(g["n"], g["h"], eps)
    got = O.unbounded_laplacian(g["f"], g["h"], gh)
    x = g["x"]
    want = np.zeros_like(got)
    for c, sig, q in zip(g["centres"], g["sigmas"], g["q"]):
        s2 = sig ** 2 + eps ** 2
        r2 = (x[:, None, None] - c[2]) ** 2 + (x[None, :, None] - c[1]) ** 2 + (x[None, None, :] - c[0]) ** 2
        want += q * (2 * np.pi * s2) ** -1.5 * np.exp(-r2 / (2 * s2))
    assert np.abs(got - want).max() <= 2e-9 * np.abs(want).max()      # measured 2.9e-10
    f3 = np.stack([g["f"], -2.0 * g["f"], g["f"][::-1].copy()])
    got3 = O.unbounded_laplacian(f3, g["h"], gh, rhs_sign=-1.0)
    assert np.abs(got3[1] - 2.0 * got).max() <= 1e-12 * np.abs(got).max()
    assert np.abs(got3[2] + got[::-1]).max() <= 1e-12 * np.abs(got).max()


def test_unbounded_divergence_of_gaussian_charges():
    """div psi for three different sets of Gaussian charges, one per component, against the analytic
    derivative of -q erf(r/(sqrt2 s))/(4 pi r) along the matching axis; and term by term against the
    gradient routine on a non-cubic anisotropic grid (each component picks its own axis)."""
    n = 64
    gs = [W.gaussian_blobs(n, seed=77 + i, nblobs=2, sigma_h=(2.5, 3.5), inner=(0.3, 0.7)) for i in range(3)]
    eps = 2 * gs[0]["h"][0]
    gh = O.unbounded_green(gs[0]["n"], gs[0]["h"], eps)
    f = np.stack([q["f"] for q in gs])
    got = O.unbounded_divergence(f, gs[0]["h"], gh)
    want = sum(gaussian_blob_potential_gradient(gs[a], eps)[a] for a in range(3))
    assert np.abs(got - want).max() <= 1e-10 * np.abs(want).max()     # measured 6.6e-12
    rng = np.random.default_rng(11)
    f = rng.normal(size=(3, 8, 16, 32))
    h = (0.11, 0.07, 0.13)
    gh = O.unbounded_green((32, 16, 8), h, 0.3)
    div = O.unbounded_divergence(f, h, gh, rhs_sign=-1.0)
    ref = sum(O.unbounded_gradient(f[a], h, gh, rhs_sign=-1.0)[1][a] for a in range(3))
    assert np.abs(div - ref).max() <= 1e-13 * np.abs(ref).max()


def test_periodic_curl_of_plane_wave_potentials():
    """psi_c = A_c sin(kappa . x + phi_c) with three different amplitudes and phases and a different integer
    wavenumber per axis on a non-cubic box: the source is lap psi_c = -|kappa|^2 psi_c and the curl is
    u_a = kappa_b A_c cos(. + phi_c) - kappa_c A_b cos(. + phi_b), (a, b, c) cyclic -- a swapped axis, a wrong
    sign or a dropped term fails; pseudo-spectral operator, exact to rounding."""
    n = (32, 16, 8)          # x, y, z
    L = (2.0, 1.0, 3.0)
    x, y, z = _grid(n, L)
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
    m = (3, -2, 1)
    kap = [2 * np.pi * m[a] / L[a] for a in range(3)]
    ph = kap[0] * X + kap[1] * Y + kap[2] * Z
    A, phi = (0.7, -1.3, 0.4), (0.1, 0.9, -0.5)
    k2 = sum(k * k for k in kap)
    f = np.stack([-k2 * A[c] * np.sin(ph + phi[c]) for c in range(3)])
    want = np.stack([kap[(a + 1) % 3] * A[(a + 2) % 3] * np.cos(ph + phi[(a + 2) % 3])
                     - kap[(a + 2) % 3] * A[(a + 1) % 3] * np.cos(ph + phi[(a + 1) % 3]) for a in range(3)])
    got = O.periodic_curl(f, L, O.OP_PS)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    assert np.abs(O.periodic_curl(f, L, O.OP_PS, rhs_sign=-1.0) + want).max() <= 1e-12 * np.abs(want).max()


def test_periodic_curl_from_the_pinned_gradient_and_divergence_free():
    """white noise, FD2 operator: u_a = d_b psi_c - d_c psi_b with the derivatives of the (separately pinned)
    scalar solve; div u = 0 in spectral space (kappa . (kappa x psi) = 0), checked with the spectral divergence
    of three plain gradients"""
    rng = np.random.default_rng(8)
    shape = (8, 16, 32)
    L = (1.0, 2.0, 0.5)
    f = rng.normal(size=(3,) + shape)
    u = O.periodic_curl(f, L, O.OP_FD2)
    grads = [O.periodic(f[c], L, O.OP_FD2, want_grad=True)[1] for c in range(3)]
    for a in range(3):
        b, c = (a + 1) % 3, (a + 2) % 3
        want = grads[c][b] - grads[b][c]
        assert np.abs(u[a] - want).max() <= 1e-12 * np.abs(want).max()
    # divergence of u through the pseudo-spectral derivative of each component (solve lap^-1, then lap = identity
    # on zero-mean band-limited data is avoided: differentiate directly with numpy's FFT as a third opinion)
    div = np.zeros(shape)
    for a in range(3):
        ax = 2 - a
        k = 2 * np.pi * np.fft.fftfreq(shape[ax], d=L[a] / shape[ax])
        k[shape[ax] // 2] = 0.0
        sl = [None] * 3
        sl[ax] = slice(None)
        div += np.fft.ifft(1j * k[tuple(sl)] * np.fft.fft(u[a], axis=ax), axis=ax).real
    assert np.abs(div).max() <= 1e-11 * max(np.abs(u).max() * np.abs(k).max(), 1.0)
