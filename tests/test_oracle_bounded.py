"""Pins P3, P4, P12 for the Dirichlet (DST-I) and Neumann (DCT-II/III) oracles."""
import numpy as np
import pytest
import scipy.fft as sfft

import oracle as O
import workloads as W
from analytic import bounded_discrete_solution


def _stencil_dirichlet(psi, h, faces):
    """7-point Laplacian on interior nodes with the boundary-node values taken from `faces`."""
    n = psi.shape[0]
    ext = np.zeros((n + 2,) * 3)
    ext[1:-1, 1:-1, 1:-1] = psi
    if faces:
        # faces[(axis, side)][upper remaining, lower remaining]; array axes are (z, y, x) = (2, 1, 0)
        ext[1:-1, 1:-1, 0] = faces[(0, 0)]      # x lo: [z, y]
        ext[1:-1, 1:-1, -1] = faces[(0, 1)]
        ext[1:-1, 0, 1:-1] = faces[(1, 0)]      # y lo: [z, x]
        ext[1:-1, -1, 1:-1] = faces[(1, 1)]
        ext[0, 1:-1, 1:-1] = faces[(2, 0)]      # z lo: [y, x]
        ext[-1, 1:-1, 1:-1] = faces[(2, 1)]
    c = ext[1:-1, 1:-1, 1:-1]
    lap = (ext[1:-1, 1:-1, :-2] + ext[1:-1, 1:-1, 2:] - 2 * c) / h[0] ** 2
    lap += (ext[1:-1, :-2, 1:-1] + ext[1:-1, 2:, 1:-1] - 2 * c) / h[1] ** 2
    lap += (ext[:-2, 1:-1, 1:-1] + ext[2:, 1:-1, 1:-1] - 2 * c) / h[2] ** 2
    return lap


def _stencil_neumann(psi, h, faces):
    """7-point Laplacian on cell centres with ghost cells psi_ghost = psi_edge -/+ h g (g = d psi/dx_a)."""
    n = psi.shape[0]
    ext = np.zeros((n + 2,) * 3)
    ext[1:-1, 1:-1, 1:-1] = psi
    g = lambda k: (faces[k] if faces and k in faces else 0.0)
    ext[1:-1, 1:-1, 0] = psi[:, :, 0] - h[0] * g((0, 0))
    ext[1:-1, 1:-1, -1] = psi[:, :, -1] + h[0] * g((0, 1))
    ext[1:-1, 0, 1:-1] = psi[:, 0, :] - h[1] * g((1, 0))
    ext[1:-1, -1, 1:-1] = psi[:, -1, :] + h[1] * g((1, 1))
    ext[0, 1:-1, 1:-1] = psi[0, :, :] - h[2] * g((2, 0))
    ext[-1, 1:-1, 1:-1] = psi[-1, :, :] + h[2] * g((2, 1))
    c = ext[1:-1, 1:-1, 1:-1]
    lap = (ext[1:-1, 1:-1, :-2] + ext[1:-1, 1:-1, 2:] - 2 * c) / h[0] ** 2
    lap += (ext[1:-1, :-2, 1:-1] + ext[1:-1, 2:, 1:-1] - 2 * c) / h[1] ** 2
    lap += (ext[:-2, 1:-1, 1:-1] + ext[2:, 1:-1, 1:-1] - 2 * c) / h[2] ** 2
    return lap


@pytest.mark.parametrize("nc", [8, 16, 32])
def test_dirichlet_discrete_closed_form_and_stencil(nc):
    d = W.dirichlet3d_manufactured(nc)
    psi = O.dirichlet_regular(d["f"], d["h"], d["faces"])
    assert np.abs(psi - bounded_discrete_solution(d, "dirichlet")).max() < 1e-12      # P3
    assert np.abs(_stencil_dirichlet(psi, d["h"], d["faces"]) - d["f"]).max() < 1e-9   # the definition


def test_dirichlet_faces_are_not_interchangeable():
    # different random face arrays on all six faces: a swapped axis/side or a transposed face fails
    rng = np.random.default_rng(11)
    n = 7
    h = (1.0 / 8, 1.0 / 8, 1.0 / 8)
    f = rng.normal(size=(n, n, n))
    faces = {(a, s): rng.normal(size=(n, n)) for a in range(3) for s in range(2)}
    psi = O.dirichlet_regular(f, h, faces)
    assert np.abs(_stencil_dirichlet(psi, h, faces) - f).max() < 1e-10
    swapped = dict(faces)
    swapped[(0, 0)], swapped[(1, 0)] = faces[(1, 0)], faces[(0, 0)]
    assert np.abs(_stencil_dirichlet(psi, h, swapped) - f).max() > 1e-2
    tr = dict(faces)
    tr[(2, 1)] = faces[(2, 1)].T
    assert np.abs(_stencil_dirichlet(psi, h, tr) - f).max() > 1e-2


@pytest.mark.parametrize("nc", [8, 16, 32])
def test_neumann_discrete_closed_form_and_stencil(nc):
    d = W.neumann3d_manufactured(nc)
    psi = O.neumann_staggered(d["f"], d["h"], d["faces"])
    ref = bounded_discrete_solution(d, "neumann")
    assert np.abs(psi - (ref - ref.mean())).max() < 1e-12                              # P4
    assert abs(psi.mean()) < 1e-13
    assert np.abs(_stencil_neumann(psi, d["h"], d["faces"]) - d["f"]).max() < 1e-9


def test_neumann_homogeneous_and_random_faces():
    d = W.neumann3d_manufactured(16, inhomogeneous=False)
    psi = O.neumann_staggered(d["f"], d["h"], None)
    assert np.abs(_stencil_neumann(psi, d["h"], None) - d["f"]).max() < 1e-10
    rng = np.random.default_rng(3)
    n = 8
    h = (1.0 / 8,) * 3
    faces = {(a, s): rng.normal(size=(n, n)) for a in range(3) for s in range(2)}
    f = rng.normal(size=(n, n, n))
    # make the discrete problem compatible: sum f' = 0
    flux = sum((faces[(a, 0)].sum() - faces[(a, 1)].sum()) / h[a] for a in range(3))
    f -= (f.sum() + flux) / f.size
    psi = O.neumann_staggered(f, h, faces)
    assert np.abs(_stencil_neumann(psi, h, faces) - f).max() < 1e-10


def test_second_order_convergence_to_the_continuum_solution():
    # FD2 eigenvalues converge quadratically, also with inhomogeneous BCs
    for gen, solve, zero_mean in ((W.dirichlet3d_manufactured, O.dirichlet_regular, False),
                                  (W.neumann3d_manufactured, O.neumann_staggered, True)):
        errs = []
        for nc in (16, 32, 64):
            d = gen(nc, modes=(3, 1, 2))  # low modes: resolved on all three grids
            psi = solve(d["f"], d["h"], d["faces"])
            u = d["u"] - d["u"].mean() if zero_mean else d["u"]
            errs.append(np.abs(psi - u).max())
        assert 3.5 < errs[0] / errs[1] < 4.5 and 3.8 < errs[1] / errs[2] < 4.2


def test_pseudo_spectral_eigenvalues_are_exact_for_the_basis_functions():
    # PS eigenvalues give spectral accuracy for homogeneous BCs
    d = W.dirichlet3d_manufactured(32, inhomogeneous=False)
    psi = O.dirichlet_regular(d["f"], d["h"], None, op=O.OP_PS)
    assert np.abs(psi - d["u"]).max() < 1e-13
    d = W.neumann3d_manufactured(32, inhomogeneous=False)
    psi = O.neumann_staggered(d["f"], d["h"], None, op=O.OP_PS)
    assert np.abs(psi - (d["u"] - d["u"].mean())).max() < 1e-13


def test_library_third_opinion():
    # P12: the same three steps with scipy's dstn / dctn
    rng = np.random.default_rng(8)
    n, h = 15, 1.0 / 16
    f = rng.normal(size=(n, n, n))
    k = np.arange(n)
    lam1 = -(4 / h ** 2) * np.sin(np.pi * (k + 1) / (2 * (n + 1))) ** 2
    lam = lam1[:, None, None] + lam1[None, :, None] + lam1[None, None, :]
    ref = sfft.dstn(sfft.dstn(f, type=1) / lam, type=1) / (2 * (n + 1)) ** 3
    assert np.abs(O.dirichlet_regular(f, (h,) * 3) - ref).max() < 1e-13
    n, h = 16, 1.0 / 16
    f = rng.normal(size=(n, n, n))
    f -= f.mean()
    k = np.arange(n)
    lam1 = -(4 / h ** 2) * np.sin(np.pi * k / (2 * n)) ** 2
    lam = lam1[:, None, None] + lam1[None, :, None] + lam1[None, None, :]
    lam[0, 0, 0] = 1.0
    fh = sfft.dctn(f, type=2) / lam
    fh[0, 0, 0] = 0.0
    ref = sfft.dctn(fh, type=3) / (2 * n) ** 3
    assert np.abs(O.neumann_staggered(f, (h,) * 3) - ref).max() < 1e-13
