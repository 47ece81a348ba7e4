"""The copy pipeline of the C ABI (sf_set_pipeline / sf_get_output_async / sf_pipeline_join; include/sailffish.h):
the call sequence Set_Input -> solve -> Get_Output of PAPER.md:268-272 with host buffers, upload, compute and
download of neighbouring steps overlapped on three streams.  Every step's result must be that of its own source."""
import numpy as np
import pytest
import torch

import oracle as O
import paper_2301_01145_b200 as sf
import workloads as W
from gpu_solve import Plan, rel_l2

pytestmark = pytest.mark.gpu


def _sources(n, count, seed):
    return [np.ascontiguousarray(W.Rng(seed + k).normal(n ** 3).reshape(n, n, n).astype(np.float32)) for k in range(count)]


def test_pipelined_steps_return_their_own_results():
    n, steps = 64, 7
    h = (1.0 / n,) * 3
    srcs = _sources(n, steps, 4242)
    gh = O.unbounded_green((n, n, n), h, 2.0 * h[0])
    refs = [O.unbounded_solve(s.astype(np.float64), h, gh) for s in srcs]
    with Plan((n, n, n), h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f32") as p:
        sf.sf_set_pipeline(p.plan, 2)
        pinned_in = [torch.from_numpy(s).pin_memory() for s in srcs]
        pinned_out = [torch.empty((n, n, n), dtype=torch.float32).pin_memory() for _ in range(steps)]
        for k in range(steps):
            sf.sf_set_source(p.plan, pinned_in[k])
            sf.sf_solve(p.plan)
            sf.sf_get_output_async(p.plan, sf.SF_OUT_PSI, 0, pinned_out[k])
        sf.sf_synchronize(p.plan)
        for k in range(steps):
            e = rel_l2(pinned_out[k].numpy(), refs[k])
            assert e <= 2e-5, f"step {k}: rel-L2 {e:.3e}"
        # two solves on one source, a device-resident source, and the blocking call, all inside the pipeline
        sf.sf_set_source(p.plan, pinned_in[1])
        sf.sf_solve(p.plan)
        sf.sf_solve(p.plan)
        got = np.empty((n, n, n), dtype=np.float32)
        sf.sf_get_output(p.plan, sf.SF_OUT_PSI, 0, got)
        assert rel_l2(got, refs[1]) <= 2e-5
        dev = torch.from_numpy(srcs[2]).cuda()
        sf.sf_set_source(p.plan, dev)
        sf.sf_solve(p.plan)
        sf.sf_get_output_async(p.plan, sf.SF_OUT_PSI, 0, pinned_out[0])
        sf.sf_pipeline_join(p.plan)
        sf.sf_synchronize(p.plan)
        assert rel_l2(pinned_out[0].numpy(), refs[2]) <= 2e-5
        # back to the single stream
        sf.sf_set_pipeline(p.plan, 1)
        sf.sf_set_source(p.plan, pinned_in[3])
        sf.sf_solve(p.plan)
        sf.sf_get_output(p.plan, sf.SF_OUT_PSI, 0, got)
        assert rel_l2(got, refs[3]) <= 2e-5


def test_pipeline_with_gradient_work_set_and_bad_depth():
    n = 32
    h = (1.0 / n,) * 3
    srcs = _sources(n, 3, 99)
    gh = O.unbounded_green((n, n, n), h, 2.0 * h[0])
    with Plan((n, n, n), h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f64") as p:
        with pytest.raises(sf.SailffishError):
            sf.sf_set_pipeline(p.plan, 3)
        sf.sf_set_pipeline(p.plan, 2)
        outs = [torch.empty((n, n, n), dtype=torch.float64).pin_memory() for _ in range(3)]
        ins = [torch.from_numpy(srcs[k].astype(np.float64)).pin_memory() for k in range(3)]   # alive until the copies ran
        for k in range(3):
            sf.sf_set_source(p.plan, ins[k])
            sf.sf_gradient(p.plan)      # unbounded plans: results in the four-field work set, one buffer
            sf.sf_get_output_async(p.plan, sf.SF_OUT_PSI, 0, outs[k])
        sf.sf_synchronize(p.plan)
        for k in range(3):
            ref = O.unbounded_solve(srcs[k].astype(np.float64), h, gh)
            assert rel_l2(outs[k].numpy(), ref) <= 1e-12
