"""Boundary values with rhs_sign = -1: the face arrays hold psi (Dirichlet) or d psi / d x_a (Neumann)
whatever the sign convention of the right-hand side is.  The discrete equation is lap_h psi = rhs_sign f with the
face values in the ghost layer (eq. (2), reading A8; fold PAPER.md:173), so data built from the
definition, f = rhs_sign * stencil(psi0, faces), must give psi0 back.  Parity alone cannot see a mistake here
(both sides would share the formula): the pin is the seven-point equation itself, for all four rows of Table 1,
on the oracle (CPU) and on the CUDA path (GPU)."""
import numpy as np
import pytest

import oracle as O
import paper_2301_01145_b200 as sf
from test_oracle_bounded import _stencil_dirichlet, _stencil_neumann
from test_oracle_bounded_f3 import stencil_dirichlet_centre, stencil_neumann_boundary


def _faces(rng, shape):
    nz, ny, nx = shape
    return {(0, 0): rng.normal(size=(nz, ny)), (0, 1): rng.normal(size=(nz, ny)), (1, 0): rng.normal(size=(nz, nx)),
            (1, 1): rng.normal(size=(nz, nx)), (2, 0): rng.normal(size=(ny, nx)), (2, 1): rng.normal(size=(ny, nx))}


# row of Table 1 -> (oracle solver, stencil with ghost layer, cubic size, Neumann?)
ROWS = {
    "dirichlet_boundary": (O.dirichlet_regular, _stencil_dirichlet, 7, False),
    "neumann_centre": (O.neumann_staggered, _stencil_neumann, 8, True),
    "dirichlet_centre": (O.dirichlet_staggered, stencil_dirichlet_centre, 8, False),
    "neumann_boundary": (O.neumann_regular, stencil_neumann_boundary, 9, True),
}


def _case(row, seed):
    solver, stencil, n, neumann = ROWS[row]
    rng = np.random.default_rng(seed)
    shape = (n, n, n)
    h = (0.11, 0.07, 0.13)
    psi0 = rng.normal(size=shape)
    faces = _faces(rng, shape)
    return solver, stencil, shape, h, psi0, faces, neumann


@pytest.mark.parametrize("row", sorted(ROWS))
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_oracle_recovers_a_field_from_its_stencil_for_both_signs(row, sign):
    solver, stencil, shape, h, psi0, faces, neumann = _case(row, 21)
    f = sign * stencil(psi0, h, faces)
    psi = solver(f, h, faces, rhs_sign=sign)
    if neumann:
        psi, psi0 = psi - psi.mean(), psi0 - psi0.mean()
    assert np.abs(psi - psi0).max() < 1e-10
    # the residual of the equation with the TRUE faces vanishes; with the negated faces it does not
    assert np.abs(sign * stencil(psi, h, faces) - f - (sign * stencil(psi, h, faces) - f).mean() * neumann).max() < 1e-9
    neg = {k: -v for k, v in faces.items()}
    assert np.abs(sign * stencil(psi, h, neg) - f).max() > 1.0


@pytest.mark.gpu
@pytest.mark.parametrize("row", sorted(ROWS))
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cuda_path_recovers_a_field_from_its_stencil_with_negative_sign(row, prec):
    from gpu_solve import Plan, rounded
    solver, stencil, shape, h, psi0, faces, neumann = _case(row, 22)
    f = rounded(-stencil(psi0, h, faces), prec)
    faces = {k: rounded(v, prec) for k, v in faces.items()}
    bc = sf.SF_BC_NEUMANN if neumann else sf.SF_BC_DIRICHLET
    grid = sf.SF_GRID_CELL_BOUNDARY if row.endswith("boundary") else sf.SF_GRID_CELL_CENTRE
    with Plan(shape, h, bc, grid=grid, op=sf.SF_OP_FD2, prec=prec, rhs_sign=-1.0) as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI).astype(np.float64)
    ref = solver(f.astype(np.float64), h, {k: v.astype(np.float64) for k, v in faces.items()}, rhs_sign=-1.0)
    if neumann:
        got, ref, psi0 = got - got.mean(), ref - ref.mean(), psi0 - psi0.mean()
    tol = 1e-12 if prec == "f64" else 2e-5
    assert np.linalg.norm(got - ref) <= tol * np.linalg.norm(ref)
    assert np.abs(got - psi0).max() < (1e-9 if prec == "f64" else 2e-3) * np.abs(psi0).max()
