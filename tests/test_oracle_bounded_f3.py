"""Pins for the other two rows of Table 1: Dirichlet on a cell-centre grid
(DST-II / DST-III) and Neumann on a cell-boundary grid (DCT-I)."""
import numpy as np
import pytest
import scipy.fft as sfft

import oracle as O
import workloads as W
from analytic import fd2_amplitude


def _lap(ext, h):
    c = ext[1:-1, 1:-1, 1:-1]
    lap = (ext[1:-1, 1:-1, :-2] + ext[1:-1, 1:-1, 2:] - 2 * c) / h[0] ** 2
    lap += (ext[1:-1, :-2, 1:-1] + ext[1:-1, 2:, 1:-1] - 2 * c) / h[1] ** 2
    lap += (ext[:-2, 1:-1, 1:-1] + ext[2:, 1:-1, 1:-1] - 2 * c) / h[2] ** 2
    return lap


def stencil_dirichlet_centre(psi, h, faces):
    """7-point Laplacian on cell centres; the face value g sits half a cell outside the first centre:
    psi_ghost = 2 g - psi_first (linear interpolation through the face)."""
    ext = np.pad(psi, 1)
    g = lambda k: (faces[k] if faces and k in faces else 0.0)
    ext[1:-1, 1:-1, 0] = 2 * g((0, 0)) - psi[:, :, 0]
    ext[1:-1, 1:-1, -1] = 2 * g((0, 1)) - psi[:, :, -1]
    ext[1:-1, 0, 1:-1] = 2 * g((1, 0)) - psi[:, 0, :]
    ext[1:-1, -1, 1:-1] = 2 * g((1, 1)) - psi[:, -1, :]
    ext[0, 1:-1, 1:-1] = 2 * g((2, 0)) - psi[0, :, :]
    ext[-1, 1:-1, 1:-1] = 2 * g((2, 1)) - psi[-1, :, :]
    return _lap(ext, h)


def stencil_neumann_boundary(psi, h, faces):
    """7-point Laplacian on nodes including the boundary nodes; the ghost node mirrors the second node
    through the boundary node: psi_ghost = psi_second -/+ 2 h g, g = d psi / d x_a along +axis."""
    ext = np.pad(psi, 1)
    g = lambda k: (faces[k] if faces and k in faces else 0.0)
    ext[1:-1, 1:-1, 0] = psi[:, :, 1] - 2 * h[0] * g((0, 0))
    ext[1:-1, 1:-1, -1] = psi[:, :, -2] + 2 * h[0] * g((0, 1))
    ext[1:-1, 0, 1:-1] = psi[:, 1, :] - 2 * h[1] * g((1, 0))
    ext[1:-1, -1, 1:-1] = psi[:, -2, :] + 2 * h[1] * g((1, 1))
    ext[0, 1:-1, 1:-1] = psi[1, :, :] - 2 * h[2] * g((2, 0))
    ext[-1, 1:-1, 1:-1] = psi[-2, :, :] + 2 * h[2] * g((2, 1))
    return _lap(ext, h)


def test_transforms_against_their_definitions():
    # two-point case by hand: DST-II of (a, b) = (sqrt2 (a + b), 2 (a - b)); DCT-I of (a, b, c) = (a + 2b + c, a - c, a - 2b + c)
    a, b, c = 0.3, -1.1, 0.7
    assert np.allclose(O.dst2(np.array([a, b])), [np.sqrt(2) * (a + b), 2 * (a - b)], rtol=0, atol=1e-15)
    assert np.allclose(O.dct1(np.array([a, b, c])), [a + 2 * b + c, a - c, a - 2 * b + c], rtol=0, atol=1e-15)
    rng = np.random.default_rng(5)
    for n in (3, 8, 17, 33):
        x = rng.normal(size=n)
        assert np.abs(O.dst2(x) - sfft.dst(x, type=2)).max() < 1e-13 * n
        assert np.abs(O.dst3(x) - sfft.dst(x, type=3)).max() < 1e-13 * n
        assert np.abs(O.dct1(x) - sfft.dct(x, type=1)).max() < 1e-13 * n
        assert np.abs(O.dst3(O.dst2(x)) - 2 * n * x).max() < 1e-12 * n            # inverse pair up to 2N
        assert np.abs(O.dct1(O.dct1(x)) - 2 * (n - 1) * x).max() < 1e-12 * n      # own inverse up to 2(N-1)
    # the basis vectors: DST-II of sin(pi (j+1/2) m / N) is N at k = m - 1 and zero elsewhere
    n, m = 16, 5
    j = np.arange(n)
    y = O.dst2(np.sin(np.pi * (j + 0.5) * m / n))
    want = np.zeros(n)
    want[m - 1] = n
    assert np.abs(y - want).max() < 1e-13
    y = O.dct1(np.cos(np.pi * np.arange(n + 1) * m / n))
    want = np.zeros(n + 1)
    want[m] = n
    assert np.abs(y - want).max() < 1e-13


@pytest.mark.parametrize("nc", [8, 16, 32])
def test_dirichlet_centre_closed_form_and_stencil(nc):
    # homogeneous faces: the product of sines is an eigenvector of the ghost-cell system
    d = W.dirichlet3d_centre_manufactured(nc, inhomogeneous=False)
    psi = O.dirichlet_staggered(d["f"], d["h"], None)
    assert np.abs(psi - fd2_amplitude(d["m"], d["h"][0]) * d["u"]).max() < 1e-12
    assert np.abs(stencil_dirichlet_centre(psi, d["h"], None) - d["f"]).max() < 1e-9
    # inhomogeneous faces: the definition
    d = W.dirichlet3d_centre_manufactured(nc)
    psi = O.dirichlet_staggered(d["f"], d["h"], d["faces"])
    assert np.abs(stencil_dirichlet_centre(psi, d["h"], d["faces"]) - d["f"]).max() < 1e-9


def test_dirichlet_centre_faces_are_not_interchangeable():
    rng = np.random.default_rng(12)
    shape = (4, 8, 16)    # z, y, x
    h = (0.11, 0.07, 0.13)
    f = rng.normal(size=shape)
    faces = {(0, 0): rng.normal(size=(4, 8)), (0, 1): rng.normal(size=(4, 8)), (1, 0): rng.normal(size=(4, 16)),
             (1, 1): rng.normal(size=(4, 16)), (2, 0): rng.normal(size=(8, 16)), (2, 1): rng.normal(size=(8, 16))}
    psi = O.dirichlet_staggered(f, h, faces)
    assert np.abs(stencil_dirichlet_centre(psi, h, faces) - f).max() < 1e-9
    sw = dict(faces)
    sw[(0, 0)], sw[(0, 1)] = faces[(0, 1)], faces[(0, 0)]
    assert np.abs(stencil_dirichlet_centre(psi, h, sw) - f).max() > 1e-2


@pytest.mark.parametrize("nc", [8, 16, 32])
def test_neumann_boundary_closed_form_and_stencil(nc):
    # product of cosines (eigenvector) plus the quadratic, which the mirrored ghost node reproduces exactly
    d = W.neumann3d_boundary_manufactured(nc)
    psi = O.neumann_regular(d["f"], d["h"], d["faces"])
    x, m = d["x"], d["m"]
    tx, ty, tz = (np.cos(m[i] * np.pi * x) for i in range(3))
    prod = tz[:, None, None] * ty[None, :, None] * tx[None, None, :]
    ref = fd2_amplitude(m, d["h"][0]) * prod + (d["u"] - prod)
    assert np.abs((psi - psi.mean()) - (ref - ref.mean())).max() < 1e-11
    assert np.abs(stencil_neumann_boundary(psi, d["h"], d["faces"]) - d["f"]).max() < 1e-9
    # zero-mode convention: the k = 0 coefficient, i.e. the trapezoid-weighted mean, vanishes
    w = np.ones(nc + 1)
    w[0] = w[-1] = 0.5
    assert abs(np.einsum("zyx,z,y,x->", psi, w, w, w)) < 1e-11


def test_neumann_boundary_recovers_a_random_field():
    """data built from the definition: f = stencil(psi0, faces) with random psi0 and random fluxes is
    compatible by construction; the solve returns psi0 up to a constant"""
    rng = np.random.default_rng(13)
    shape = (5, 9, 17)
    h = (0.11, 0.07, 0.13)
    psi0 = rng.normal(size=shape)
    faces = {(0, 0): rng.normal(size=(5, 9)), (0, 1): rng.normal(size=(5, 9)), (1, 0): rng.normal(size=(5, 17)),
             (1, 1): rng.normal(size=(5, 17)), (2, 0): rng.normal(size=(9, 17)), (2, 1): rng.normal(size=(9, 17))}
    f = stencil_neumann_boundary(psi0, h, faces)
    psi = O.neumann_regular(f, h, faces)
    assert np.abs((psi - psi.mean()) - (psi0 - psi0.mean())).max() < 1e-10
    tr = dict(faces)
    tr[(0, 0)], tr[(0, 1)] = faces[(0, 1)], faces[(0, 0)]
    bad = O.neumann_regular(f, h, tr)
    assert np.abs((bad - bad.mean()) - (psi0 - psi0.mean())).max() > 1e-3


def test_dirichlet_centre_recovers_a_random_field():
    rng = np.random.default_rng(14)
    shape = (4, 8, 16)
    h = (0.11, 0.07, 0.13)
    psi0 = rng.normal(size=shape)
    faces = {(0, 0): rng.normal(size=(4, 8)), (0, 1): rng.normal(size=(4, 8)), (1, 0): rng.normal(size=(4, 16)),
             (1, 1): rng.normal(size=(4, 16)), (2, 0): rng.normal(size=(8, 16)), (2, 1): rng.normal(size=(8, 16))}
    f = stencil_dirichlet_centre(psi0, h, faces)
    assert np.abs(O.dirichlet_staggered(f, h, faces) - psi0).max() < 1e-11


def test_f3_second_order_convergence_and_ps_exactness():
    for gen, solve, zero_mean in ((W.dirichlet3d_centre_manufactured, O.dirichlet_staggered, False),
                                  (W.neumann3d_boundary_manufactured, O.neumann_regular, True)):
        errs = []
        for nc in (16, 32, 64):
            d = gen(nc, modes=(3, 1, 2))
            psi = solve(d["f"], d["h"], d["faces"])
            if zero_mean:
                errs.append(np.abs((psi - psi.mean()) - (d["u"] - d["u"].mean())).max())
            else:
                errs.append(np.abs(psi - d["u"]).max())
        assert 3.5 < errs[0] / errs[1] < 4.5 and 3.8 < errs[1] / errs[2] < 4.2, errs
    d = W.dirichlet3d_centre_manufactured(32, inhomogeneous=False)
    assert np.abs(O.dirichlet_staggered(d["f"], d["h"], None, op=O.OP_PS) - d["u"]).max() < 1e-13
    d = W.neumann3d_boundary_manufactured(32, inhomogeneous=False)
    psi = O.neumann_regular(d["f"], d["h"], None, op=O.OP_PS)
    assert np.abs((psi - psi.mean()) - (d["u"] - d["u"].mean())).max() < 1e-13


# ------------------------------------------------------------------- spectral gradient on bounded plans
def _grid_of(kind, n, L):
    """grid points and basis functions of the four Table-1 rows on [0, L]"""
    if kind == "dirichlet_regular":
        h = L / (n + 1)
        return h, (np.arange(n) + 1.0) * h, np.sin, np.cos, 1.0
    if kind == "dirichlet_staggered":
        h = L / n
        return h, (np.arange(n) + 0.5) * h, np.sin, np.cos, 1.0
    if kind == "neumann_staggered":
        h = L / n
        return h, (np.arange(n) + 0.5) * h, np.cos, np.sin, -1.0
    h = L / (n - 1)
    return h, np.arange(n) * h, np.cos, np.sin, -1.0


@pytest.mark.parametrize("kind,shape", [("dirichlet_regular", (7, 15, 31)), ("dirichlet_staggered", (8, 16, 32)),
                                        ("neumann_staggered", (8, 16, 32)), ("neumann_regular", (9, 17, 33))])
def test_bounded_gradient_of_the_basis_functions(kind, shape):
    """u = prod_a sin|cos(m_a pi x_a / L_a) on a non-cubic, anisotropic box: with the pseudo-spectral eigenvalues
    the solve returns u and the gradient m_a pi / L_a cos|(-sin)(...) to rounding; with FD2 both
    carry the amplitude ratio of the eigenvalues.  Different m, n and L per axis: components cannot be swapped."""
    nz, ny, nx = shape
    L = (1.0, 0.7, 1.3)
    m = (3, 2, 5)
    hs, xs, t, dt = [], [], [], []
    for a, n in enumerate((nx, ny, nz)):
        h, x, fn, dfn, sg = _grid_of(kind, n, L[a])
        kap = m[a] * np.pi / L[a]
        hs.append(h); xs.append(x); t.append(fn(kap * x)); dt.append(sg * kap * dfn(kap * x))
    outer = lambda v: v[2][:, None, None] * v[1][None, :, None] * v[0][None, None, :]
    u = outer(t)
    k2 = sum((m[a] * np.pi / L[a]) ** 2 for a in range(3))
    f = -k2 * u
    psi, grad = O.bounded_gradient(kind, f, hs, None, op=O.OP_PS)
    assert np.abs(psi - u).max() < 1e-13
    for a in range(3):
        want = outer([dt[i] if i == a else t[i] for i in range(3)])
        assert np.abs(grad[a] - want).max() < 1e-12 * np.abs(want).max(), (kind, a)
    lam_fd = sum((4 / hs[a] ** 2) * np.sin(m[a] * np.pi * hs[a] / (2 * L[a])) ** 2 for a in range(3))
    psi2, grad2 = O.bounded_gradient(kind, f, hs, None, op=O.OP_FD2, rhs_sign=-1.0)
    assert np.abs(psi2 + (k2 / lam_fd) * u).max() < 1e-13
    for a in range(3):
        assert np.abs(grad2[a] + (k2 / lam_fd) * grad[a]).max() < 1e-11 * np.abs(grad[a]).max()
    # psi is the plain solver's
    assert np.abs(psi2 - getattr(O, kind)(f, hs, None, op=O.OP_FD2, rhs_sign=-1.0)).max() < 1e-14 * np.abs(psi2).max()


def test_bounded_gradient_is_linear_and_axis_specific():
    """white noise on a non-cubic anisotropic grid: the gradient is linear in the source, flips with rhs_sign,
    and d/dx_a of a field that varies along x_a only has no other component"""
    rng = np.random.default_rng(21)
    shape, h = (8, 16, 32), (0.11, 0.07, 0.13)
    f1, f2 = rng.normal(size=shape), rng.normal(size=shape)
    for kind in ("dirichlet_staggered", "neumann_staggered"):
        _, g1 = O.bounded_gradient(kind, f1, h)
        _, g2 = O.bounded_gradient(kind, f2, h)
        _, g12 = O.bounded_gradient(kind, 2 * f1 - 3 * f2, h, rhs_sign=-1.0)
        assert np.abs(g12 + 2 * g1 - 3 * g2).max() < 1e-12 * np.abs(g12).max()
        fx = np.broadcast_to(rng.normal(size=(1, 1, 32)), shape).copy()
        _, g = O.bounded_gradient(kind, fx, h)
        if kind.startswith("neumann"):     # constant along y, z is a basis function (k = 0): pure x dependence
            assert np.abs(g[1]).max() < 1e-12 * np.abs(g[0]).max() and np.abs(g[2]).max() < 1e-12 * np.abs(g[0]).max()
