"""Edge cases of the CUDA path against the oracle: the smallest and the largest transform lengths the library
builds (complex pass length 4 .. 2048), sizes just outside them, and the degenerate sources of the method
(all-zero, constant = pure zero mode, a single non-zero cell)."""
import numpy as np
import pytest

import oracle as O
import workloads as W
import paper_2301_01145_b200 as sf
from gpu_solve import TOL, Plan, rel_l2

pytestmark = pytest.mark.gpu
C, B = sf.SF_GRID_CELL_CENTRE, sf.SF_GRID_CELL_BOUNDARY


def _rand(shape, seed):
    return W.Rng(seed).normal(int(np.prod(shape))).reshape(shape)


def _solve(shape, h, bc, grid, op, f, **kw):
    with Plan(shape, h, bc, grid=grid, op=op, prec="f64", **kw) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        return p.get(sf.SF_OUT_PSI)


def _oracle(kind, f, h, shape):
    nz, ny, nx = shape
    if kind == "periodic":
        return O.periodic(f, (nx * h[0], ny * h[1], nz * h[2]), O.OP_FD2)
    if kind == "unbounded":
        return O.unbounded_solve(f, h, O.unbounded_green((nx, ny, nz), h, 2.0 * max(h)))
    return getattr(O, kind)(f, h, None)


_CASES = {
    # kind: (bc, grid, op, smallest shape, shapes with one axis at the largest built length)
    "periodic": (sf.SF_BC_PERIODIC, C, sf.SF_OP_FD2, (4, 4, 8), [(4, 4, 4096), (4, 2048, 8), (2048, 4, 8)]),
    "unbounded": (sf.SF_BC_UNBOUNDED, C, sf.SF_OP_GREEN_GAUSS2, (4, 4, 8), [(4, 4, 2048), (4, 1024, 8), (1024, 4, 8)]),
    "dirichlet_regular": (sf.SF_BC_DIRICHLET, B, sf.SF_OP_FD2, (3, 3, 7), [(3, 3, 2047), (3, 2047, 7)]),
    "dirichlet_staggered": (sf.SF_BC_DIRICHLET, C, sf.SF_OP_FD2, (4, 4, 8), [(4, 4, 2048), (2048, 4, 8)]),
    "neumann_staggered": (sf.SF_BC_NEUMANN, C, sf.SF_OP_FD2, (4, 4, 8), [(4, 4, 2048), (4, 2048, 8)]),
    "neumann_regular": (sf.SF_BC_NEUMANN, B, sf.SF_OP_FD2, (5, 5, 9), [(5, 5, 2049), (2049, 5, 9)]),
}


@pytest.mark.parametrize("kind", list(_CASES))
def test_smallest_and_largest_transform_lengths(kind):
    bc, grid, op, small, large = _CASES[kind]
    for i, shape in enumerate([small] + large):
        f = _rand(shape, 900 + i)
        if kind in ("periodic", "neumann_staggered", "neumann_regular"):
            f -= f.mean()
        h = (0.013, 0.021, 0.017)
        got = _solve(shape, h, bc, grid, op, f)
        ref = _oracle(kind, f, h, shape)
        if kind.startswith("neumann"):
            got, ref = got - got.mean(), ref - ref.mean()
        e = rel_l2(got, ref)
        print(f"{kind} {shape}: rel-L2 {e:.3e}")
        assert e <= TOL["f64"], (kind, shape, e)


def test_sizes_outside_the_built_range():
    for shape, bc, grid in (((4, 4, 8192), sf.SF_BC_PERIODIC, C), ((4, 4, 4), sf.SF_BC_PERIODIC, C), ((4, 2, 8), sf.SF_BC_PERIODIC, C),
                            ((4, 4, 4096), sf.SF_BC_UNBOUNDED, C), ((3, 3, 4095), sf.SF_BC_DIRICHLET, B), ((4, 4, 12), sf.SF_BC_NEUMANN, C)):
        op = sf.SF_OP_GREEN_GAUSS2 if bc == sf.SF_BC_UNBOUNDED else sf.SF_OP_FD2
        with pytest.raises(sf.SailffishError) as ei:
            Plan(shape, (0.1,) * 3, bc, grid=grid, op=op)
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED, shape


@pytest.mark.parametrize("kind", list(_CASES))
def test_degenerate_sources(kind):
    bc, grid, op, _, _ = _CASES[kind]
    shape = {"dirichlet_regular": (7, 15, 31), "neumann_regular": (9, 17, 33)}.get(kind, (8, 16, 32))
    h = (0.1, 0.07, 0.13)
    with Plan(shape, h, bc, grid=grid, op=op, prec="f64") as p:
        p.set_source(np.zeros(shape))
        sf.sf_solve(p.plan)
        assert not p.get(sf.SF_OUT_PSI).any()                       # zero in, exactly zero out
        if kind in ("periodic", "neumann_staggered", "neumann_regular"):
            p.set_source(np.full(shape, 3.7))                        # pure zero mode: dropped
            sf.sf_solve(p.plan)
            assert np.abs(p.get(sf.SF_OUT_PSI)).max() < 1e-12
        e = np.zeros(shape)
        e[shape[0] - 1, 0, shape[2] - 1] = 1.0                      # one cell, in a corner
        if kind in ("periodic", "neumann_staggered", "neumann_regular"):
            e -= e.mean()
        p.set_source(e)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
    ref = _oracle(kind, e, h, shape)
    if kind.startswith("neumann"):
        got, ref = got - got.mean(), ref - ref.mean()
    assert rel_l2(got, ref) <= TOL["f64"]


def test_gradient_shared_memory_limit_is_checked_at_the_call():
    """a 2048-point fp64 pencil fits the fused pass once (solve) but not twice (gradient): the plan is
    created, the solve runs, sf_gradient reports UNSUPPORTED and leaves the plan usable"""
    shape = (2048, 4, 8)
    f = _rand(shape, 950)
    f -= f.mean()
    h = (0.013, 0.021, 0.017)
    ref = _oracle("periodic", f, h, shape)
    with Plan(shape, h, sf.SF_BC_PERIODIC, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        assert rel_l2(p.get(sf.SF_OUT_PSI), ref) <= TOL["f64"]
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_gradient(p.plan)
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED
        sf.sf_solve(p.plan)
        assert rel_l2(p.get(sf.SF_OUT_PSI), ref) <= TOL["f64"]
