"""Dirichlet / Neumann conditions mixed per axis through the C ABI (Table 1)
against orc_bounded_mixed: every axis in turn carries the other condition, both grid types, both precisions, both operator
columns, inhomogeneous faces on every side, rhs_sign = -1; and what stays unsupported."""
import numpy as np
import pytest

import oracle as O
import paper_2301_01145_b200 as sf
import workloads as W
from gpu_solve import Plan, rel_l2, rounded

pytestmark = pytest.mark.gpu
D, N = sf.SF_BC_DIRICHLET, sf.SF_BC_NEUMANN
TOL = {"f32": 2e-5, "f64": 1e-12}


def _kind(bc, grid):
    if bc == D:
        return O.KIND_DIRICHLET_BOUNDARY if grid == sf.SF_GRID_CELL_BOUNDARY else O.KIND_DIRICHLET_CENTRE
    return O.KIND_NEUMANN_CENTRE if grid == sf.SF_GRID_CELL_CENTRE else O.KIND_NEUMANN_BOUNDARY


def _size(bc, grid, k):
    """a supported size around 2^k for the Table-1 row of (bc, grid)"""
    if grid == sf.SF_GRID_CELL_CENTRE:
        return 2 ** k
    return 2 ** k - 1 if bc == D else 2 ** k + 1


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("grid", [sf.SF_GRID_CELL_BOUNDARY, sf.SF_GRID_CELL_CENTRE])
@pytest.mark.parametrize("bcs", [(N, D, D), (D, N, D), (D, D, N), (N, N, D), (D, N, N), (N, D, N)])
def test_mixed_dirichlet_neumann_against_the_oracle(bcs, grid, prec):
    n = [_size(bcs[0], grid, 5), _size(bcs[1], grid, 4), _size(bcs[2], grid, 6)]      # x, y, z
    shape = (n[2], n[1], n[0])
    h = (0.013, 0.021, 0.017)
    f = rounded(W.Rng(8100 + n[0]).normal(int(np.prod(shape))).reshape(shape), prec)
    faces = {}
    for a in range(3):
        fs = [shape[i] for i in range(3) if i != 2 - a]
        for s in range(2):
            faces[(a, s)] = rounded(W.Rng(8200 + 10 * a + s).normal(int(np.prod(fs))).reshape(fs), prec)
    kinds = [_kind(b, grid) for b in bcs]
    for op, oop, fc, rs in ((sf.SF_OP_FD2, O.OP_FD2, faces, -1.0), (sf.SF_OP_PSEUDO_SPECTRAL, O.OP_PS, None, 1.0)):
        ref = O.bounded_mixed(kinds, f.astype(np.float64), h, None if fc is None else {k: v.astype(np.float64) for k, v in fc.items()},
                              op=oop, rhs_sign=rs)
        with Plan(shape, h, list(bcs), grid=grid, op=op, prec=prec, rhs_sign=rs) as p:
            p.set_source(f)
            if fc is not None:
                p.set_faces(fc)
            sf.sf_solve(p.plan)
            sf.sf_solve(p.plan)
            got = p.get(sf.SF_OUT_PSI)
            assert sf.sf_last_launch_count(p.plan) == 5
        e = rel_l2(got, ref)
        print(f"mixed {bcs} grid {grid} op {op} {prec}: rel-L2 {e:.3e}")
        assert e <= TOL[prec]


def test_mixed_full_width_pencils_and_2d():
    """256-point pencils on every axis (the generation-2 X pass runs next to generation-1 strided passes), and a 2-D plan"""
    shape = (256, 255, 256)       # z Neumann (cell-centre would need one grid type: use the cell-boundary grid: D 255, N 257)
    bcs = (D, D, N)
    grid = sf.SF_GRID_CELL_BOUNDARY
    shape = (257, 255, 255)
    h = (1.0 / 256,) * 3
    f = W.Rng(8300).normal(int(np.prod(shape))).reshape(shape)
    ref = O.bounded_mixed([_kind(b, grid) for b in bcs], f, h)
    with Plan(shape, h, list(bcs), grid=grid, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
    e = rel_l2(got, ref)
    print(f"mixed D D N 255x255x257 f64: rel-L2 {e:.3e}")
    assert e <= 1e-12


def test_mixed_plans_reject_what_is_not_built():
    with pytest.raises(sf.SailffishError):
        sf.sf_plan_create([32, 32, 32], [0.1] * 3, [sf.SF_BC_PERIODIC, D, D])
    with pytest.raises(sf.SailffishError):
        sf.sf_plan_create([32, 32, 32], [0.1] * 3, [D, sf.SF_BC_UNBOUNDED, D], op=sf.SF_OP_GREEN_GAUSS2)
    plan = sf.sf_plan_create([32, 32, 32], [0.1] * 3, [D, N, D], grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2, prec=sf.SF_F64)
    try:
        src = torch_zeros = None
        import torch
        sf.sf_set_source(plan, torch.zeros((32, 32, 32), dtype=torch.float64, device="cuda"))
        with pytest.raises(sf.SailffishError):
            sf.sf_gradient(plan)
    finally:
        sf.sf_plan_destroy(plan)
