"""Pins of the mixed-boundary-condition oracle orc_bounded_mixed (Table 1):
it reduces to the four pinned uniform solvers, reproduces discrete eigenfunctions that are a different Table-1 row on every
axis, and satisfies the seven-point equation with the ghost layer each axis' own condition prescribes (reading A18)."""
import numpy as np
import pytest

import oracle as O
import workloads as W

pytestmark = pytest.mark.filterwarnings("ignore")


def _basis(kind, n, k):
    """discrete eigenvector k of the second difference on n unknowns for the Table-1 row `kind`, and cells"""
    j = np.arange(n)
    if kind == O.KIND_DIRICHLET_BOUNDARY:
        return np.sin(np.pi * (j + 1) * (k + 1) / (n + 1)), n + 1, k + 1
    if kind == O.KIND_NEUMANN_CENTRE:
        return np.cos(np.pi * (j + 0.5) * k / n), n, k
    if kind == O.KIND_DIRICHLET_CENTRE:
        return np.sin(np.pi * (j + 0.5) * (k + 1) / n), n, k + 1
    return np.cos(np.pi * j * k / (n - 1)), n - 1, k


def _ghost_extend(psi, kinds, h, faces):
    """psi[z, y, x] with one ghost layer per side and axis, as each axis' condition prescribes (reading A18)"""
    ext = np.pad(psi, 1).astype(np.float64)
    for axis in range(3):           # x = 0, y = 1, z = 2; array axis = 2 - axis
        ax = 2 - axis
        e = np.moveaxis(ext, ax, 0)     # view: e[0] lower ghost, e[1] first layer, e[-2] last layer, e[-1] upper ghost
        core = (slice(1, -1), slice(1, -1))
        glo = faces.get((axis, 0))
        ghi = faces.get((axis, 1))
        def face(g):
            # faces are indexed [upper remaining axis, lower remaining axis]; the moved view keeps the remaining axes in
            # array order (z before y before x), i.e. upper remaining axis first
            return 0.0 if g is None else g
        k = kinds[axis]
        if k == O.KIND_DIRICHLET_BOUNDARY:
            e[0][core] = face(glo); e[-1][core] = face(ghi)
        elif k == O.KIND_NEUMANN_CENTRE:
            e[0][core] = e[1][core] - h[axis] * face(glo); e[-1][core] = e[-2][core] + h[axis] * face(ghi)
        elif k == O.KIND_DIRICHLET_CENTRE:
            e[0][core] = 2.0 * face(glo) - e[1][core]; e[-1][core] = 2.0 * face(ghi) - e[-2][core]
        else:
            e[0][core] = e[2][core] - 2.0 * h[axis] * face(glo); e[-1][core] = e[-3][core] + 2.0 * h[axis] * face(ghi)
    return ext


def _lap(ext, h):
    c = ext[1:-1, 1:-1, 1:-1]
    return ((ext[1:-1, 1:-1, 2:] - 2 * c + ext[1:-1, 1:-1, :-2]) / h[0] ** 2 + (ext[1:-1, 2:, 1:-1] - 2 * c + ext[1:-1, :-2, 1:-1]) / h[1] ** 2
            + (ext[2:, 1:-1, 1:-1] - 2 * c + ext[:-2, 1:-1, 1:-1]) / h[2] ** 2)


@pytest.mark.parametrize("kind", [0, 1, 2, 3])
def test_uniform_kinds_reduce_to_the_pinned_solvers(kind):
    n = {0: (7, 9, 6), 1: (8, 6, 10), 2: (8, 6, 10), 3: (9, 5, 7)}[kind]       # (nz, ny, nx)
    h = (0.3, 0.2, 0.25)
    f = W.Rng(91 + kind).normal(int(np.prod(n))).reshape(n)
    faces = {(a, s): W.Rng(500 + 10 * a + s).normal(int(np.prod(n)) // n[2 - a]).reshape([n[i] for i in range(3) if i != 2 - a])
             for a in range(3) for s in range(2)}
    if kind in (1, 3):
        faces = None           # (an inhomogeneous pure-Neumann problem needs a compatible source; covered below)
        f = f - f.mean() if kind == 1 else f
    ref = {0: O.dirichlet_regular, 1: O.neumann_staggered, 2: O.dirichlet_staggered, 3: O.neumann_regular}[kind](f, h, faces)
    got = O.bounded_mixed((kind,) * 3, f, h, faces)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("kinds,n", [((0, 3, 0), (7, 9, 15)), ((3, 0, 3), (9, 7, 5)), ((1, 2, 1), (8, 6, 4)), ((2, 1, 2), (4, 8, 6)),
                                     ((2, 2, 1), (6, 4, 8))])
def test_discrete_eigenfunctions_mixed_rows(kinds, n):
    """kinds / n in (x, y, z) order.  f = Lambda phi for a product of per-axis discrete eigenvectors -> psi = phi"""
    h = (0.11, 0.07, 0.13)
    ks = (2, 1, 3)
    vec, lam = [], 0.0
    for a in range(3):
        v, cells, m = _basis(kinds[a], n[a], ks[a])
        vec.append(v)
        lam += -(4.0 / h[a] ** 2) * np.sin(np.pi * m / (2.0 * cells)) ** 2
    phi = vec[2][:, None, None] * vec[1][None, :, None] * vec[0][None, None, :]
    psi = O.bounded_mixed(kinds, lam * phi, h)
    assert np.abs(psi - phi).max() <= 1e-12 * np.abs(phi).max()
    # and the pseudo-spectral column divides by the continuous eigenvalue instead
    lam_ps = sum(-(np.pi * _basis(kinds[a], n[a], ks[a])[2] / (_basis(kinds[a], n[a], ks[a])[1] * h[a])) ** 2 for a in range(3))
    psi = O.bounded_mixed(kinds, lam_ps * phi, h, op=O.OP_PS)
    assert np.abs(psi - phi).max() <= 1e-12 * np.abs(phi).max()


@pytest.mark.parametrize("kinds,n,rhs_sign", [((0, 3, 0), (7, 9, 15), 1.0), ((3, 0, 0), (9, 7, 7), -1.0), ((1, 2, 1), (8, 6, 4), 1.0),
                                              ((2, 1, 2), (4, 8, 6), -1.0), ((2, 2, 2), (4, 8, 6), 1.0)])
def test_seven_point_equation_with_each_axis_own_ghost_layer(kinds, n, rhs_sign):
    """random source, six different random faces: lap_h psi = rhs_sign f with the ghost layer of every axis' own
    condition -- a swapped face, a wrong weight or a wrong row on one axis fails this"""
    h = (0.21, 0.17, 0.13)
    shape = (n[2], n[1], n[0])
    f = W.Rng(77).normal(int(np.prod(shape))).reshape(shape)
    faces = {}
    for a in range(3):
        fs = [shape[i] for i in range(3) if i != 2 - a]
        for s in range(2):
            faces[(a, s)] = W.Rng(900 + 10 * a + s).normal(int(np.prod(fs))).reshape(fs)
    psi = O.bounded_mixed(kinds, f, h, faces, rhs_sign=rhs_sign)
    res = _lap(_ghost_extend(psi, kinds, h, faces), h) - rhs_sign * f
    assert np.abs(res).max() <= 1e-9 * np.abs(f).max()
