"""Generation-2 kernels on plans that reach them from an unusual side: the fp64 X passes (sf_fastx64.cuh) on 2-D plans and on
3-D plans whose strided passes stay on generation 1, the 512-pencil kernels on a scalar plan, odd row counts (the last
tile of an X pass is ragged).  Everything against the oracle, through the C ABI."""
import numpy as np
import pytest

import oracle as O
import paper_2301_01145_b200 as sf
import workloads as W
from gpu_solve import TOL, Plan, rel_l2, rounded

pytestmark = pytest.mark.gpu


def _rand(shape, seed):
    return W.Rng(seed).normal(int(np.prod(shape))).reshape(shape)


def _report(name, got, ref, prec):
    e = rel_l2(got, ref)
    print(f"{name}: rel-L2 {e:.3e} (tol {TOL[prec]:.0e})")
    assert np.isfinite(e) and e <= TOL[prec], f"{name}: rel-L2 {e:.3e}"


def test_fp64_x_passes_on_2d_plans():
    # periodic rows of 256 (fast_xp64_kernel), gradient
    f = _rand((36, 256), 21)
    f -= f.mean()
    L = (2.0, 1.5)
    with pytest.raises(sf.SailffishError):     # 36 is not a power of two: the size rule still applies
        Plan(f.shape, (L[0] / 256, L[1] / 36), sf.SF_BC_PERIODIC, prec="f64")
    f = _rand((32, 256), 21)
    f -= f.mean()
    psi_o, grad_o = O.periodic(f, L, O.OP_PS, want_grad=True)
    with Plan(f.shape, (L[0] / 256, L[1] / 32), sf.SF_BC_PERIODIC, prec="f64") as p:
        p.set_source(f)
        sf.sf_gradient(p.plan)
        _report("2-D periodic 32x256 psi", p.get(sf.SF_OUT_PSI), psi_o, "f64")
        _report("2-D periodic 32x256 dpsi/dx", p.get(sf.SF_OUT_GRAD, 0), grad_o[0], "f64")
    # zero-padded rows of 256 (fast_xg_kernel<X_ZEROPAD>)
    f = _rand((16, 256), 22)
    h = (0.01, 0.013)
    gh = O.unbounded2d_green((256, 16), h, 2.0 * max(h), 2)
    with Plan(f.shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        _report("2-D unbounded 16x256 psi", p.get(sf.SF_OUT_PSI), O.unbounded2d_solve(f, h, gh), "f64")


@pytest.mark.parametrize("kind,shape", [("dirichlet", (7, 3, 255)), ("neumann", (4, 8, 256)), ("dirichlet", (15, 3, 255))])
def test_fp64_x_passes_with_generation_1_strided_passes(kind, shape):
    """rows of 255 / 256 with few, odd numbers of rows: ragged last tile of the X pass, generation-1 y / z passes"""
    f = _rand(shape, 31 + shape[0])
    h = (0.004, 0.11, 0.09)
    faces = {}
    for a in range(3):
        fs = [shape[i] for i in range(3) if i != 2 - a]
        for s in range(2):
            faces[(a, s)] = _rand(fs, 40 + 10 * a + s)
    if kind == "dirichlet":
        ref = O.dirichlet_regular(f, h, faces)
        bc, grid = sf.SF_BC_DIRICHLET, sf.SF_GRID_CELL_BOUNDARY
    else:
        # a compatible pure-Neumann problem: homogeneous fluxes, zero-mean source
        faces = None
        f = f - f.mean()
        ref = O.neumann_staggered(f, h, None)
        bc, grid = sf.SF_BC_NEUMANN, sf.SF_GRID_CELL_CENTRE
    with Plan(shape, h, bc, grid=grid, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        if faces:
            p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
    if kind == "neumann":
        got, ref = got - got.mean(), ref - ref.mean()
    _report(f"{kind} {shape} f64", got, ref, "f64")


def test_scalar_plan_on_512_pencils():
    """sf_solve of a scalar fp32 unbounded plan with 512-long y / z pencils (the fused pass of sf_fast512.cuh with one component)"""
    shape = (512, 512, 16)
    f = rounded(_rand(shape, 51), "f32")
    h = (1.0 / 512,) * 3
    gh = O.unbounded_green((16, 512, 512), h, 2.0 * h[0])
    ref = O.unbounded_solve(f.astype(np.float64), h, gh)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f32") as p:
        p.set_source(f)
        for _ in range(2):
            sf.sf_solve(p.plan)
        _report("scalar 512x512x16 f32", p.get(sf.SF_OUT_PSI), ref, "f32")


@pytest.mark.parametrize("env", ["SF_X_CTA", "SF_FUSED_2P", "SF_FUSED_1P", "SF_PAD_1H"])
def test_launch_time_kernel_switches_agree(env, monkeypatch):
    """the kernels that the default launch no longer picks (X passes with one pipeline per CTA; the fused z pass with one
    half of two pencils / of one pencil per thread; the y passes with one half per thread) stay correct: same plan, same
    source, switch read at launch time"""
    shape = (256, 256, 32)
    f = rounded(_rand(shape, 77), "f32")
    h = (0.010, 0.012, 0.011)
    gh = O.unbounded_green((32, 256, 256), h, 2.0 * max(h))
    ref = O.unbounded_solve(f.astype(np.float64), h, gh)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f32") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        a = p.get(sf.SF_OUT_PSI)
        monkeypatch.setenv(env, "1")
        sf.sf_solve(p.plan)
        b = p.get(sf.SF_OUT_PSI)
        monkeypatch.delenv(env)
    _report("default kernels", a, ref, "f32")
    _report(f"{env}=1", b, ref, "f32")
    assert rel_l2(a, b.astype(np.float64)) <= 1e-6


@pytest.mark.parametrize("case", ["periodic_f32", "periodic_f64", "dirichlet_f64", "vector_f32"])
def test_cta_x_kernels_agree(case, monkeypatch):
    """SF_X_CTA=1 on the other plans with warp-autonomous X passes"""
    if case.startswith("periodic"):
        prec = case[-3:]
        shape = (256, 256, 256) if prec == "f32" else (256, 256, 256)
        f = rounded(_rand(shape, 5), prec)
        f -= f.mean(dtype=np.float64).astype(f.dtype)
        mk = lambda: Plan(shape, (1.0 / 256,) * 3, sf.SF_BC_PERIODIC, prec=prec)
    elif case == "dirichlet_f64":
        prec, shape = "f64", (255, 255, 255)
        f = rounded(_rand(shape, 6), prec)
        mk = lambda: Plan(shape, (1.0 / 256,) * 3, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2, prec=prec)
    else:
        prec, shape = "f32", (512, 16, 512)
        f = rounded(_rand(shape, 7), prec)
        mk = lambda: Plan(shape, (0.01,) * 3, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec=prec)
    with mk() as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        a = p.get(sf.SF_OUT_PSI).astype(np.float64)
        monkeypatch.setenv("SF_X_CTA", "1")
        sf.sf_solve(p.plan)
        b = p.get(sf.SF_OUT_PSI).astype(np.float64)
        monkeypatch.delenv("SF_X_CTA")
    e = rel_l2(a, b)
    print(f"{case}: warp vs CTA X kernels rel-L2 {e:.3e}")
    assert np.isfinite(e) and e <= (1e-6 if prec == "f32" else 1e-13)
