"""The oracle against the stored closed-form values of tests/golden/ (written by
tests/golden/make_golden.py from the Python standard library only; citations in each file header)."""
from pathlib import Path

import numpy as np

import oracle as O

G = Path(__file__).resolve().parent / "golden"


def _rows(name):
    return [ln.split() for ln in (G / name).read_text().splitlines() if ln and not ln.startswith("#")]


def test_green_kernel_values():
    for r, eps, g in _rows("green_gauss2.txt"):
        assert abs(O.green_gauss2(float(r), float(eps)) - float(g)) <= 2e-15 * abs(float(g))


def test_green_kernel_orders_and_dimensions():
    for dim, order, r, eps, g in _rows("green_orders.txt"):
        dim, order, r, eps, g = int(dim), int(order), float(r), float(eps), float(g)
        if dim == 3 and order == 0:
            got = O.green_spectral(r, eps)
        elif dim == 3:
            got = O.green_gauss(order, r, eps)
        else:
            got = O.green2d_gauss(order, r, eps)
        assert abs(got - g) <= 1e-13 * abs(g), (dim, order, r, eps, got, g)


def test_gaussian_blob_potential():
    rows = _rows("gaussian_blob.txt")
    for sh, eh in sorted({(r[1], r[2]) for r in rows}):
        sel = [r for r in rows if (r[1], r[2]) == (sh, eh)]
        n, q = int(sel[0][0]), float(sel[0][3])
        h = 1.0 / n
        sig = float(sh) * h
        x = (np.arange(n) + 0.5) * h - (32 + 0.5) * h
        g1 = np.exp(-x * x / (2 * sig * sig))
        f = q * (2 * np.pi * sig * sig) ** -1.5 * g1[:, None, None] * g1[None, :, None] * g1[None, None, :]
        gh = O.unbounded_green((n, n, n), (h, h, h), float(eh) * h)
        psi = O.unbounded_solve(f, (h, h, h), gh)
        for r in sel:
            ix, iy, iz, phi = int(r[4]), int(r[5]), int(r[6]), float(r[7])
            assert abs(psi[iz, iy, ix] - phi) <= 1e-11 * abs(phi) + 1e-13, (r, psi[iz, iy, ix])


def test_fd2_dirichlet_amplification():
    for nc, mx, my, mz, A in _rows("fd2_dirichlet.txt"):
        nc, m, A = int(nc), (int(mx), int(my), int(mz)), float(A)
        h = 1.0 / nc
        x = (np.arange(nc - 1) + 1.0) * h
        prod = (np.sin(m[2] * np.pi * x)[:, None, None] * np.sin(m[1] * np.pi * x)[None, :, None]
                * np.sin(m[0] * np.pi * x)[None, None, :])
        f = -(np.pi ** 2) * sum(v * v for v in m) * prod
        psi = O.dirichlet_regular(f, (h, h, h))
        assert np.abs(psi - A * prod).max() <= 1e-12 * abs(A)


def test_periodic_single_mode():
    rows = _rows("periodic_mode.txt")
    for key in sorted({tuple(r[:5]) for r in rows}):
        n, p, q, a, b = int(key[0]), int(key[1]), int(key[2]), float(key[3]), float(key[4])
        x = (np.arange(n) + 0.5) / n
        X, Y = np.meshgrid(x, x, indexing="xy")
        th = 2 * np.pi * (p * X + q * Y)
        psi, grad = O.periodic(a * np.cos(th) + b * np.sin(th), (1.0, 1.0), O.OP_PS, want_grad=True)
        for r in [r for r in rows if tuple(r[:5]) == key]:
            ix, iy = int(r[5]), int(r[6])
            assert abs(psi[iy, ix] - float(r[7])) <= 1e-14
            assert abs(grad[0][iy, ix] - float(r[8])) <= 1e-13
            assert abs(grad[1][iy, ix] - float(r[9])) <= 1e-13
