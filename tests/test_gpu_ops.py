"""Parity of the DIV and NABLA operators (reading A27) through
the C ABI against the oracle, element by element on seeded white noise: every spectral coefficient
carries signal, so a wrong wavenumber table, sign or component fails."""
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


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("op", [O.OP_PS, O.OP_FD2])
def test_periodic_divergence_and_laplacian(prec, op):
    shape = (16, 64, 32)   # z, y, x
    L = (2.0, 1.0, 3.0)
    f = rounded(_rand((3,) + shape, 71), prec)
    f -= f.mean(axis=(1, 2, 3), keepdims=True).astype(f.dtype)
    h = (L[0] / 32, L[1] / 64, L[2] / 16)
    sop = sf.SF_OP_PSEUDO_SPECTRAL if op == O.OP_PS else sf.SF_OP_FD2
    div_o = O.periodic_divergence(f.astype(np.float64), L, op, rhs_sign=-1.0)
    lap_o = O.periodic_laplacian(f.astype(np.float64), L, op, rhs_sign=-1.0, ncomp=3)
    with Plan(shape, h, sf.SF_BC_PERIODIC, op=sop, prec=prec, ncomp=3, rhs_sign=-1.0) as p:
        p.set_source(f)
        sf.sf_divergence(p.plan)
        assert sf.sf_last_launch_count(p.plan) == 5
        _report("div psi", p.get(sf.SF_OUT_DIV), div_o, prec)
        with pytest.raises(sf.SailffishError) as ei:
            p.get(sf.SF_OUT_PSI, 0)
        assert ei.value.status == sf.SF_ERR_STATE
        sf.sf_laplacian(p.plan)
        for c in range(3):
            _report(f"lap psi[{c}]", p.get(sf.SF_OUT_LAP, c), lap_o[c], prec)
        with pytest.raises(sf.SailffishError):
            p.get(sf.SF_OUT_DIV)
        sf.sf_solve(p.plan)      # the plan is still a plain solver afterwards
        psi_o = O.periodic(f[1].astype(np.float64), L, op, rhs_sign=-1.0)
        _report("psi[1] after the operators", p.get(sf.SF_OUT_PSI, 1), psi_o, prec)


def test_periodic_laplacian_2d_scalar():
    shape = (32, 128)
    L = (1.0, 0.5)
    f = _rand(shape, 72)
    f -= f.mean()
    lap_o = O.periodic_laplacian(f, L, O.OP_FD2)
    with Plan(shape, (L[0] / 128, L[1] / 32), sf.SF_BC_PERIODIC, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        sf.sf_laplacian(p.plan)
        _report("lap psi 2-D", p.get(sf.SF_OUT_LAP), lap_o, "f64")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_unbounded_divergence_and_laplacian(prec):
    shape = (8, 32, 16)
    h = (0.1, 0.05, 0.2)
    f = rounded(_rand((3,) + shape, 73), prec)
    gh = O.unbounded_green(tuple(reversed(shape)), h, 2.0 * max(h))
    div_o = O.unbounded_divergence(f.astype(np.float64), h, gh)
    lap_o = O.unbounded_laplacian(f.astype(np.float64), h, gh)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec=prec, ncomp=3) as p:
        p.set_source(f)
        sf.sf_divergence(p.plan)
        _report("div psi", p.get(sf.SF_OUT_DIV), div_o, prec)
        sf.sf_laplacian(p.plan)
        for c in range(3):
            _report(f"lap psi[{c}]", p.get(sf.SF_OUT_LAP, c), lap_o[c], prec)


def test_unbounded_laplacian_on_a_fast_path_plan():
    """sf_laplacian (generation-1 kernels) and sf_solve (generation 2) interleaved on one fp32 plan; the
    Laplacian of the regularised solution is the source smoothed by the Gaussian of width eps"""
    shape = (256, 256, 32)
    f = rounded(_rand(shape, 74), "f32")
    h = (1.0 / 256,) * 3
    gh = O.unbounded_green((32, 256, 256), h, 2.0 * h[0])
    lap_o = O.unbounded_laplacian(f.astype(np.float64), h, gh)
    psi_o = O.unbounded_solve(f.astype(np.float64), h, gh)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f32") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f32")
        sf.sf_laplacian(p.plan)
        _report("lap psi", p.get(sf.SF_OUT_LAP), lap_o, "f32")
        sf.sf_solve(p.plan)
        _report("psi again", p.get(sf.SF_OUT_PSI), psi_o, "f32")


def test_operator_error_paths():
    with Plan((16, 16, 16), (0.1,) * 3, sf.SF_BC_PERIODIC, prec="f64") as p:     # scalar plan
        p.set_source(_rand((16, 16, 16), 75))
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_divergence(p.plan)
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED
        sf.sf_laplacian(p.plan)
        with pytest.raises(sf.SailffishError) as ei:
            p.get(sf.SF_OUT_LAP, 1)
        assert ei.value.status == sf.SF_ERR_INVALID_ARG
    with Plan((15, 15, 15), (0.1,) * 3, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2) as p:
        p.set_source(_rand((15, 15, 15), 76))
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_laplacian(p.plan)
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("op", ["ps", "fd2"])
def test_periodic_curl(prec, op):
    """sf_curl on a PERIODIC vector plan (eq. (10) PAPER.md:141-148 on the component-wise solve):
    white noise on a non-cubic box against the oracle, element by element"""
    shape = (16, 64, 32)
    L = (2.0, 1.0, 3.0)
    f = rounded(_rand((3,) + shape, 99), prec)
    f -= f.mean(axis=(1, 2, 3), keepdims=True, dtype=np.float64).astype(f.dtype)
    oop, sop = (O.OP_PS, sf.SF_OP_PSEUDO_SPECTRAL) if op == "ps" else (O.OP_FD2, sf.SF_OP_FD2)
    u_o = O.periodic_curl(f.astype(np.float64), L, oop, rhs_sign=-1.0)
    h = (L[0] / shape[2], L[1] / shape[1], L[2] / shape[0])
    with Plan(shape, h, sf.SF_BC_PERIODIC, op=sop, prec=prec, ncomp=3, rhs_sign=-1.0) as p:
        p.set_source(f)
        sf.sf_curl(p.plan)
        for c in range(3):
            _report(f"periodic curl {op} u[{c}]", p.get(sf.SF_OUT_CURL, c), u_o[c], prec)
