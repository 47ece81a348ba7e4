"""Parity of the other two Table-1 rows through the C ABI against the
oracle: Dirichlet on a cell-centre grid (DST-II forward, DST-III backward) and Neumann on a
cell-boundary grid that stores its boundary nodes (DCT-I both ways)."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import paper_2301_01145_b200 as sf
from gpu_solve import TOL, Plan, rel_l2, rounded

pytestmark = pytest.mark.gpu


def _rand(shape, seed):
    return W.Rng(seed).normal(int(np.prod(shape))).reshape(shape)


def _report(name, got, ref, prec):
    e = rel_l2(got, ref)
    print(f"{name}: rel-L2 {e:.3e} (tol {TOL[prec]:.0e})")
    assert np.isfinite(e) and e <= TOL[prec], f"{name}: rel-L2 {e:.3e} > {TOL[prec]:.0e}"


def _faces(shape, seed):
    nz, ny, nx = shape
    return {(0, 0): _rand((nz, ny), seed), (0, 1): _rand((nz, ny), seed + 1), (1, 0): _rand((nz, nx), seed + 2),
            (1, 1): _rand((nz, nx), seed + 3), (2, 0): _rand((ny, nx), seed + 4), (2, 1): _rand((ny, nx), seed + 5)}


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("inhom", [True, False])
def test_dirichlet_cell_centre(prec, inhom):
    d = W.dirichlet3d_centre_manufactured(nc=32, inhomogeneous=inhom, modes=(3, 5, 2))
    f = rounded(d["f"], prec)
    faces = {k: rounded(v, prec) for k, v in d["faces"].items()}
    psi_o = O.dirichlet_staggered(f.astype(np.float64), d["h"], {k: v.astype(np.float64) for k, v in faces.items()})
    with Plan(f.shape, d["h"], sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2, prec=prec) as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        assert sf.sf_last_launch_count(p.plan) == 5
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, prec)


@pytest.mark.parametrize("shape", [(16, 32, 64), (8, 128, 16), (4, 8, 256)])
def test_dirichlet_cell_centre_noncubic_random_faces(shape):
    f = _rand(shape, 81)
    nz, ny, nx = shape
    h = (0.9 / nx, 1.1 / ny, 1.0 / nz)
    faces = _faces(shape, 82)
    psi_o = O.dirichlet_staggered(f, h, faces)
    with Plan(shape, h, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f64")


def test_dirichlet_cell_centre_pseudo_spectral_and_2d():
    d = W.dirichlet3d_centre_manufactured(nc=32, inhomogeneous=False, modes=(3, 5, 2))
    psi_o = O.dirichlet_staggered(d["f"], d["h"], None, op=O.OP_PS)
    with Plan(d["f"].shape, d["h"], sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_PSEUDO_SPECTRAL,
              prec="f64") as p:
        p.set_source(d["f"])
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
        _report("psi (PS)", got, psi_o, "f64")
        assert np.abs(got - d["u"]).max() < 1e-12      # spectral accuracy for the basis functions


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("inhom", [True, False])
def test_neumann_cell_boundary(prec, inhom):
    d = W.neumann3d_boundary_manufactured(nc=32, inhomogeneous=inhom, modes=(3, 5, 2))
    f = rounded(d["f"], prec)
    faces = {k: rounded(v, prec) for k, v in d["faces"].items()}
    psi_o = O.neumann_regular(f.astype(np.float64), d["h"], {k: v.astype(np.float64) for k, v in faces.items()})
    with Plan(f.shape, d["h"], sf.SF_BC_NEUMANN, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2, prec=prec) as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI).astype(np.float64)
        _report("psi", got - got.mean(), psi_o - psi_o.mean(), prec)


@pytest.mark.parametrize("shape", [(9, 17, 33), (5, 129, 17), (5, 9, 257)])
def test_neumann_cell_boundary_noncubic_random(shape):
    f = _rand(shape, 91)
    nz, ny, nx = shape
    h = (0.9 / nx, 1.1 / ny, 1.0 / nz)
    faces = _faces(shape, 92)
    psi_o = O.neumann_regular(f, h, faces)
    with Plan(shape, h, sf.SF_BC_NEUMANN, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
        # incompatible random data: both sides drop the zero mode (reading A21), the rest is unique
        _report("psi", got - got.mean(), psi_o - psi_o.mean(), "f64")


def test_f3_size_rules():
    with pytest.raises(sf.SailffishError) as ei:      # cell-centre Dirichlet wants 2^k cells
        Plan((15, 15, 15), (0.1,) * 3, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2)
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED
    with pytest.raises(sf.SailffishError) as ei:      # cell-boundary Neumann wants 2^k + 1 nodes
        Plan((16, 16, 16), (0.1,) * 3, sf.SF_BC_NEUMANN, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2)
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED


# ------------------------------------------------------------------- spectral gradient on bounded plans
_KINDS = {
    "dirichlet_regular": (sf.SF_BC_DIRICHLET, sf.SF_GRID_CELL_BOUNDARY, (7, 31, 63)),
    "dirichlet_staggered": (sf.SF_BC_DIRICHLET, sf.SF_GRID_CELL_CENTRE, (8, 32, 64)),
    "neumann_staggered": (sf.SF_BC_NEUMANN, sf.SF_GRID_CELL_CENTRE, (8, 32, 64)),
    "neumann_regular": (sf.SF_BC_NEUMANN, sf.SF_GRID_CELL_BOUNDARY, (9, 33, 65)),
}


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("kind", list(_KINDS))
def test_bounded_gradient_white_noise(kind, prec):
    """sf_gradient on Dirichlet / Neumann plans: psi and the three derivative fields against the oracle,
    white noise on a non-cubic anisotropic grid (every coefficient carries signal), then a plain solve"""
    bc, grid, shape = _KINDS[kind]
    f = rounded(_rand(shape, 95), prec)
    if bc == sf.SF_BC_NEUMANN:
        f -= f.mean().astype(f.dtype)
    h = (0.011, 0.023, 0.13)
    psi_o, grad_o = O.bounded_gradient(kind, f.astype(np.float64), h, None, op=O.OP_FD2, rhs_sign=-1.0)
    with Plan(shape, h, bc, grid=grid, op=sf.SF_OP_FD2, prec=prec, rhs_sign=-1.0) as p:
        p.set_source(f)
        sf.sf_gradient(p.plan)
        assert sf.sf_last_launch_count(p.plan) == 5
        got = p.get(sf.SF_OUT_PSI).astype(np.float64)
        if bc == sf.SF_BC_NEUMANN:
            _report(f"{kind} psi", got - got.mean(), psi_o - psi_o.mean(), prec)
        else:
            _report(f"{kind} psi", got, psi_o, prec)
        for a in range(3):
            _report(f"{kind} grad[{a}]", p.get(sf.SF_OUT_GRAD, a), grad_o[a], prec)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI).astype(np.float64)
        ref = getattr(O, kind)(f.astype(np.float64), h, None, rhs_sign=-1.0)
        _report(f"{kind} psi (solve after gradient)", got - got.mean(), ref - ref.mean(), prec)
        with pytest.raises(sf.SailffishError):
            p.get(sf.SF_OUT_GRAD, 0)


def test_bounded_gradient_pseudo_spectral_is_exact_for_basis_functions():
    """the analytic gradient of prod sin(m pi x) through the CUDA path itself"""
    d = W.dirichlet3d_centre_manufactured(nc=32, inhomogeneous=False, modes=(3, 5, 2))
    x, m = d["x"], d["m"]
    t = [np.sin(m[i] * np.pi * x) for i in range(3)]
    dt = [m[i] * np.pi * np.cos(m[i] * np.pi * x) for i in range(3)]
    with Plan(d["f"].shape, d["h"], sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_PSEUDO_SPECTRAL,
              prec="f64") as p:
        p.set_source(d["f"])
        sf.sf_gradient(p.plan)
        for a in range(3):
            tt = [dt[i] if i == a else t[i] for i in range(3)]
            want = tt[2][:, None, None] * tt[1][None, :, None] * tt[0][None, None, :]
            assert np.abs(p.get(sf.SF_OUT_GRAD, a) - want).max() < 1e-11 * np.abs(want).max()
