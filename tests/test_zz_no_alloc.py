"""sf_periodic2d_solve_static (include/sailffish.h): the periodic 2-D solve for callers that may not allocate -- one
kernel, its work array in a file-scope device array.  Checked against the existing plan path (sf_solve on a 2-D
periodic fp64 plan) within the fp64 tolerance of the other GPU tests, on two calls in a row (the second call finds
the first call's contents in the shared scratch), and against the oracle (Table 1 periodic row).
Collected last (file name) so that a failure here hides no other test; passes alone in a fresh process as well."""
import numpy as np
import pytest
import torch

import oracle as O
import workloads as W
import paper_2301_01145_b200 as sf
from gpu_solve import TOL, Plan, rel_l2

pytestmark = pytest.mark.gpu

_ORC_OP = {sf.SF_OP_PSEUDO_SPECTRAL: O.OP_PS, sf.SF_OP_FD2: O.OP_FD2}


def _rand(shape, seed):
    f = W.Rng(seed).normal(int(np.prod(shape))).reshape(shape)
    return np.ascontiguousarray(f - f.mean())


def _plan_solve(f, h, op):
    with Plan(f.shape, h, sf.SF_BC_PERIODIC, op=op, prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        return p.get(sf.SF_OUT_PSI)


@pytest.mark.parametrize("op", [sf.SF_OP_PSEUDO_SPECTRAL, sf.SF_OP_FD2])
@pytest.mark.parametrize("shape", [(64, 64), (32, 128), (256, 256), (8, 16)])
def test_static_entry_point_matches_the_plan_path_twice(shape, op):
    ny, nx = shape
    h = (0.013, 0.021)
    tol = TOL["f64"]
    out = torch.empty(shape, dtype=torch.float64, device="cuda")
    # two different sources back to back: the second call starts from the first call's scratch contents
    for call, seed in enumerate((900, 901)):
        f = _rand(shape, seed + nx)
        ref = _plan_solve(f, h, op)
        src = torch.from_numpy(f).cuda()
        out.fill_(float("nan"))
        sf.sf_periodic2d_solve_static((nx, ny), h, op, src, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        e = rel_l2(got, ref)
        print(f"static vs plan, {shape}, call {call}: rel-L2 {e:.3e} (tol {tol:.0e})")
        assert np.isfinite(e) and e <= tol
        orc = O.periodic(f, (nx * h[0], ny * h[1]), _ORC_OP[op])
        eo = rel_l2(got, orc)
        print(f"static vs oracle: rel-L2 {eo:.3e}")
        assert np.isfinite(eo) and eo <= tol


def test_static_entry_point_in_place_and_on_a_stream():
    shape, h = (128, 64), (0.02, 0.01)
    f = _rand(shape, 77)
    ref = _plan_solve(f, h, sf.SF_OP_PSEUDO_SPECTRAL)
    st = torch.cuda.Stream()
    buf = torch.from_numpy(f).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        sf.sf_periodic2d_solve_static((shape[1], shape[0]), h, sf.SF_OP_PSEUDO_SPECTRAL, buf, buf, stream=st.cuda_stream)
    st.synchronize()
    assert rel_l2(buf.cpu().numpy(), ref) <= TOL["f64"]


def test_static_entry_point_rejects_what_does_not_fit():
    a = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_periodic2d_solve_static((2 * sf.SF_STATIC_MAX_N, 64), (1.0, 1.0), sf.SF_OP_FD2, a, a)
    assert ei.value.status == sf.SF_ERR_INVALID_ARG and str(sf.SF_STATIC_MAX_N) in str(ei.value)
    with pytest.raises(sf.SailffishError):
        sf.sf_periodic2d_solve_static((48, 64), (1.0, 1.0), sf.SF_OP_FD2, a, a)        # not a power of two
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_periodic2d_solve_static((64, 64), (1.0, 1.0), sf.SF_OP_GREEN_GAUSS2, a, a)
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED
