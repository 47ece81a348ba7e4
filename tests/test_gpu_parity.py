"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on
the same seeded inputs (BASELINE.json north_star: rel-L2 <= 1e-12 fp64, <= 2e-5 fp32).

Sizes here are ones the oracle finishes in seconds; they span several tiles of every kernel (tiles
are 16 x-columns / 2..16 rows), ragged last tiles (x widths 17, 33, 31, 15 ... are not multiples of
16) and non-cubic shapes.  Full-size cases live in test_gpu_fullsize.py."""
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
    m = float(np.abs(np.asarray(got, dtype=np.float64) - ref).max())
    print(f"{name}: rel-L2 {e:.3e} max-abs {m:.3e} (tol {TOL[prec]:.0e})")
    assert np.isfinite(e) and e <= TOL[prec], f"{name}: rel-L2 {e:.3e} > {TOL[prec]:.0e}"


# ------------------------------------------------------------------------------- config 1
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [64, 16])
def test_cfg1_periodic_2d_ps_gradient(prec, n):
    w = W.periodic2d_modes(n, kmax=min(8, n // 4))
    f = rounded(w["f"], prec)
    psi_o, grad_o = O.periodic(f.astype(np.float64), w["L"], O.OP_PS, want_grad=True)
    h = (w["L"][0] / n, w["L"][1] / n)
    with Plan(f.shape, h, sf.SF_BC_PERIODIC, op=sf.SF_OP_PSEUDO_SPECTRAL, prec=prec) as p:
        p.set_source(f)
        sf.sf_gradient(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, prec)
        _report("dpsi/dx", p.get(sf.SF_OUT_GRAD, 0), grad_o[0], prec)
        _report("dpsi/dy", p.get(sf.SF_OUT_GRAD, 1), grad_o[1], prec)
        assert sf.sf_last_launch_count(p.plan) == 3


def test_cfg1_rectangular_2d():
    f = _rand((32, 128), 11)
    f -= f.mean()
    L = (3.0, 0.7)
    psi_o, grad_o = O.periodic(f, L, O.OP_FD2, want_grad=True)
    with Plan(f.shape, (L[0] / 128, L[1] / 32), sf.SF_BC_PERIODIC, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f, device=False)
        sf.sf_gradient(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI, device=True), psi_o, "f64")
        _report("dpsi/dy", p.get(sf.SF_OUT_GRAD, 1, device=True), grad_o[1], "f64")


# ------------------------------------------------------------------------------- config 2
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("op", [O.OP_PS, O.OP_FD2])
def test_cfg2_periodic_3d(prec, op):
    n = 64
    w = W.periodic3d_spectrum(n, kmax=16)
    f = rounded(w["f"], prec)
    psi_o, grad_o = O.periodic(f.astype(np.float64), w["L"], op, want_grad=True)
    h = tuple(L / n for L in w["L"])
    with Plan(f.shape, h, sf.SF_BC_PERIODIC, op=sf.SF_OP_PSEUDO_SPECTRAL if op == O.OP_PS else sf.SF_OP_FD2,
              prec=prec) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        _report("psi(solve)", p.get(sf.SF_OUT_PSI), psi_o, prec)
        with pytest.raises(sf.SailffishError):
            p.get(sf.SF_OUT_GRAD, 0)  # not produced by sf_solve
        sf.sf_gradient(p.plan)
        _report("psi(gradient)", p.get(sf.SF_OUT_PSI), psi_o, prec)
        for a in range(3):
            _report(f"grad[{a}]", p.get(sf.SF_OUT_GRAD, a), grad_o[a], prec)
        assert sf.sf_last_launch_count(p.plan) == 5


@pytest.mark.parametrize("shape", [(8, 16, 32), (16, 128, 8), (4, 4, 256), (32, 8, 64)])
def test_cfg2_periodic_3d_noncubic_white_noise(shape):
    # white noise excites every mode including all the Nyquist planes (reading A20)
    f = _rand(shape, 21)
    L = (1.3, 2.0, 0.9)
    psi_o, grad_o = O.periodic(f, L, O.OP_PS, want_grad=True)
    h = tuple(L[a] / shape[2 - a] for a in range(3))
    with Plan(shape, h, sf.SF_BC_PERIODIC, prec="f64") as p:
        p.set_source(f)
        sf.sf_gradient(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f64")
        for a in range(3):
            _report(f"grad[{a}]", p.get(sf.SF_OUT_GRAD, a), grad_o[a], "f64")


# ------------------------------------------------------------------------------- config 3
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("inhom", [True, False])
def test_cfg3_dirichlet(prec, inhom):
    d = W.dirichlet3d_manufactured(nc=32, inhomogeneous=inhom, modes=(3, 5, 2))
    f = rounded(d["f"], prec)
    faces = {k: rounded(v, prec) for k, v in d["faces"].items()}
    psi_o = O.dirichlet_regular(f.astype(np.float64), d["h"], {k: v.astype(np.float64) for k, v in faces.items()})
    with Plan(f.shape, d["h"], sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2, prec=prec) as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, prec)


@pytest.mark.parametrize("shape", [(15, 31, 63), (7, 127, 15), (31, 7, 255)])
def test_cfg3_dirichlet_noncubic_random_faces(shape):
    f = _rand(shape, 31)
    nz, ny, nx = shape
    h = (0.9 / (nx + 1), 1.1 / (ny + 1), 1.0 / (nz + 1))
    faces = {(0, 0): _rand((nz, ny), 32), (0, 1): _rand((nz, ny), 33), (1, 0): _rand((nz, nx), 34),
             (1, 1): _rand((nz, nx), 35), (2, 0): _rand((ny, nx), 36), (2, 1): _rand((ny, nx), 37)}
    psi_o = O.dirichlet_regular(f, h, faces)
    with Plan(shape, h, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        p.set_faces(faces, device=False)
        sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f64")
        # resetting one face to homogeneous changes the answer accordingly
        sf.sf_set_bc_values(p.plan, 2, 1, None)
        sf.sf_solve(p.plan)
        faces2 = dict(faces)
        faces2.pop((2, 1))
        _report("psi(face reset)", p.get(sf.SF_OUT_PSI), O.dirichlet_regular(f, h, faces2), "f64")


def test_cfg3_dirichlet_pseudo_spectral():
    f = _rand((15, 31, 31), 38)
    h = (1 / 32, 1 / 32, 1 / 16)
    psi_o = O.dirichlet_regular(f, h, None, op=O.OP_PS)
    with Plan(f.shape, h, sf.SF_BC_DIRICHLET, grid=sf.SF_GRID_CELL_BOUNDARY, op=sf.SF_OP_PSEUDO_SPECTRAL,
              prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f64")
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_set_bc_values(p.plan, 0, 0, f[0])
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("inhom", [True, False])
def test_cfg3_neumann(prec, inhom):
    d = W.neumann3d_manufactured(nc=32, inhomogeneous=inhom, modes=(3, 5, 2))
    f = rounded(d["f"], prec)
    faces = {k: rounded(v, prec) for k, v in d["faces"].items()}
    psi_o = O.neumann_staggered(f.astype(np.float64), d["h"], {k: v.astype(np.float64) for k, v in faces.items()})
    with Plan(f.shape, d["h"], sf.SF_BC_NEUMANN, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2, prec=prec) as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI).astype(np.float64)
        # unique up to a constant (reading A21/A24): both sides are compared zero-mean
        _report("psi", got - got.mean(), psi_o - psi_o.mean(), prec)
        if prec == "f64":
            assert abs(got.mean()) < 1e-12 * np.abs(got).max()  # zero-mode convention


@pytest.mark.parametrize("shape", [(16, 32, 64), (8, 128, 16), (4, 8, 256)])
def test_cfg3_neumann_noncubic_random(shape):
    f = _rand(shape, 41)
    nz, ny, nx = shape
    h = (0.9 / nx, 1.1 / ny, 1.0 / nz)
    faces = {(0, 0): _rand((nz, ny), 42), (0, 1): _rand((nz, ny), 43), (1, 0): _rand((nz, nx), 44),
             (1, 1): _rand((nz, nx), 45), (2, 0): _rand((ny, nx), 46), (2, 1): _rand((ny, nx), 47)}
    psi_o = O.neumann_staggered(f, h, faces)
    with Plan(shape, h, sf.SF_BC_NEUMANN, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_FD2, prec="f64") as p:
        p.set_source(f)
        p.set_faces(faces)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
        _report("psi", got - got.mean(), psi_o - psi_o.mean(), "f64")


# ------------------------------------------------------------------------------- config 4
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [32, 64])
def test_cfg4_unbounded_blobs(prec, n):
    g = W.gaussian_blobs(n, nblobs=4)
    f = rounded(g["f"], prec)
    eps = 2.0 * g["h"][0]
    gh = O.unbounded_green(g["n"], g["h"], eps)
    psi_o = O.unbounded_solve(f.astype(np.float64), g["h"], gh)
    with Plan(f.shape, g["h"], sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec=prec) as p:
        p.set_source(f)
        for _ in range(2):  # the stored spectrum is reused across solves
            sf.sf_solve(p.plan)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, prec)
        assert sf.sf_last_launch_count(p.plan) == 5


@pytest.mark.parametrize("shape", [(8, 16, 32), (32, 8, 16), (4, 64, 8)])
def test_cfg4_unbounded_noncubic_white_noise(shape):
    f = _rand(shape, 51)
    h = (0.11, 0.07, 0.13)
    eps = 1.5 * max(h)
    n = tuple(reversed(shape))
    gh = O.unbounded_green(n, h, eps)
    psi_o = O.unbounded_solve(f, h, gh, rhs_sign=-1.0)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f64", rhs_sign=-1.0, eps_over_h=1.5) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
        _report("psi", got, psi_o, "f64")
    # and against the definition itself (direct O(N^6) sum) on samples
    idx = np.array([0, 17, f.size // 2 + 5, f.size - 1])
    ref = O.unbounded_direct_samples(f, h, eps, idx, rhs_sign=-1.0)
    assert np.allclose(got.ravel()[idx], ref, rtol=1e-11, atol=1e-13 * np.abs(psi_o).max())


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("order,op", [(4, sf.SF_OP_GREEN_GAUSS4), (6, sf.SF_OP_GREEN_GAUSS6), (8, sf.SF_OP_GREEN_GAUSS8),
                                      (10, sf.SF_OP_GREEN_GAUSS10)])
def test_cfg4_higher_order_kernels(prec, order, op):
    """Hejlesen's Gaussian kernels of order 4 .. 10 -- plan-time only, the
    solve kernels are the same; vs the oracle and vs the closed form of a Gaussian charge."""
    from analytic import gaussian_blob_potential_order
    n = 64
    g = W.gaussian_blobs(n, nblobs=1, sigma_h=(2.0, 2.0), inner=(0.45, 0.55))
    f = rounded(g["f"], prec)
    eps = 2.0 * g["h"][0]
    psi_o = O.unbounded_solve(f.astype(np.float64), g["h"], O.unbounded_green(g["n"], g["h"], eps, order=order))
    with Plan(f.shape, g["h"], sf.SF_BC_UNBOUNDED, op=op, prec=prec) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
    _report(f"psi order {order}", got, psi_o, prec)
    e = rel_l2(got, gaussian_blob_potential_order(g, eps, order))
    assert e <= (5e-6 if prec == "f32" else 1e-11), e


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cfg4_spectrally_compact_kernel(prec):
    """Hejlesen's spectrally compact kernel -- vs the oracle on white noise
    (anisotropic spacing: h = max spacing, reading A26) and vs the free-space potential of a resolved
    Gaussian charge, which it reproduces to rounding."""
    from analytic import gaussian_blob_potential
    shape = (16, 32, 64)
    f = rounded(_rand(shape, 77), prec)
    hs = (0.11, 0.07, 0.13)
    psi_o = O.unbounded_solve(f.astype(np.float64), hs, O.unbounded_green((64, 32, 16), hs, max(hs), order=0))
    with Plan(shape, hs, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_SPECTRAL, prec=prec, eps_over_h=123.0) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        _report("psi spectral kernel, white noise", p.get(sf.SF_OUT_PSI), psi_o, prec)
    g = W.gaussian_blobs(64, nblobs=1, sigma_h=(3.0, 3.0), inner=(0.47, 0.53))
    f = rounded(g["f"], prec)
    with Plan(f.shape, g["h"], sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_SPECTRAL, prec=prec) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        e = rel_l2(p.get(sf.SF_OUT_PSI), gaussian_blob_potential(g, 0.0))
    print(f"spectral kernel vs free-space potential: rel-L2 {e:.3e}")
    assert e <= (5e-6 if prec == "f32" else 1e-11)


def test_spectral_kernel_unit_source_against_the_library_sine_integral():
    """the DEVICE sine integral (Bessel-function series / asymptotic auxiliary functions; shares no expansion
    with the oracle's series + continued fraction) pinned to scipy's Si: a unit source returns
    h^3 G(|x - x0|) = -h^3 Si(pi r / h) / (2 pi^2 r) itself (reading A26).  Arguments pi r / h from 3 to 340
    cross the switch between the two device expansions at 50."""
    from scipy.special import sici
    n, h = 64, 1.0 / 64
    f = np.zeros((n, n, n))
    x0 = (40, 3, 63)
    f[x0] = 1.0
    with Plan(f.shape, (h, h, h), sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_SPECTRAL, prec="f64") as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        got = p.get(sf.SF_OUT_PSI)
    iz, iy, ix = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    r = h * np.sqrt((iz - x0[0]) ** 2.0 + (iy - x0[1]) ** 2.0 + (ix - x0[2]) ** 2.0)
    want = np.full(r.shape, -1.0 / (2 * np.pi * h))
    nz = r > 0
    want[nz] = -sici(np.pi * r[nz] / h)[0] / (2 * np.pi ** 2 * r[nz])
    want *= h ** 3
    assert (np.pi * r.max() / h) > 300 and (np.pi * r[nz].min() / h) < 4
    # the transform round trip adds rounding ~ 1e-16 |G|_max, so the tolerance is absolute against the peak
    assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()
    assert rel_l2(got, want) <= 1e-13


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cfg4_unbounded_gradient(prec):
    """sf_gradient on a scalar unbounded plan (north_star: ik gradients from the same spectrum):
    psi and the three derivatives vs the oracle on a non-cubic white-noise case, then a solve on the
    same plan still returns psi (the gradient call uses its own work arrays)."""
    shape = (16, 32, 64)
    f = rounded(_rand(shape, 91), prec)
    hs = (0.11, 0.07, 0.13)
    gh = O.unbounded_green((64, 32, 16), hs, 2.0 * max(hs))
    psi_o, grad_o = O.unbounded_gradient(f.astype(np.float64), hs, gh, rhs_sign=-1.0)
    with Plan(shape, hs, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec=prec, rhs_sign=-1.0) as p:
        p.set_source(f)
        sf.sf_solve(p.plan)
        with pytest.raises(sf.SailffishError):
            p.get(sf.SF_OUT_GRAD, 0)
        sf.sf_gradient(p.plan)
        _report("psi(gradient)", p.get(sf.SF_OUT_PSI), psi_o, prec)
        for a in range(3):
            _report(f"grad[{a}]", p.get(sf.SF_OUT_GRAD, a), grad_o[a], prec)
        sf.sf_solve(p.plan)
        _report("psi(solve after gradient)", p.get(sf.SF_OUT_PSI), psi_o, prec)


# ------------------------------------------------------------------------------- config 5
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_cfg5_vortex_ring_curl(prec):
    n = 32
    v = W.vortex_ring(n, sigma_h=2.0)
    om = rounded(v["omega"], prec)
    eps = 2.0 * v["h"][0]
    gh = O.unbounded_green(v["n"], v["h"], eps)
    u_o = O.unbounded_solve(om.astype(np.float64), v["h"], gh, rhs_sign=-1.0, want_curl=True)
    psi_o = O.unbounded_solve(om.astype(np.float64), v["h"], gh, rhs_sign=-1.0)
    with Plan(om.shape[1:], v["h"], sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec=prec, ncomp=3,
              rhs_sign=-1.0) as p:
        p.set_source(om)
        sf.sf_curl(p.plan)
        for c in range(3):
            _report(f"u[{c}]", p.get(sf.SF_OUT_CURL, c), u_o[c], prec)
        assert sf.sf_last_launch_count(p.plan) == 5
        with pytest.raises(sf.SailffishError):
            p.get(sf.SF_OUT_PSI, 0)
        sf.sf_solve(p.plan)  # vector solve = three scalar solves
        for c in range(3):
            _report(f"psi[{c}]", p.get(sf.SF_OUT_PSI, c), psi_o[c], prec)


def test_cfg5_noncubic_white_noise_curl():
    shape = (8, 32, 16)
    om = _rand((3,) + shape, 61)
    h = (0.1, 0.05, 0.2)
    eps = 2.0 * max(h)
    gh = O.unbounded_green(tuple(reversed(shape)), h, eps)
    u_o = O.unbounded_solve(om, h, gh, rhs_sign=-1.0, want_curl=True)
    with Plan(shape, h, sf.SF_BC_UNBOUNDED, op=sf.SF_OP_GREEN_GAUSS2, prec="f64", ncomp=3, rhs_sign=-1.0) as p:
        p.set_source(om)
        sf.sf_curl(p.plan)
        for c in range(3):
            _report(f"u[{c}]", p.get(sf.SF_OUT_CURL, c), u_o[c], "f64")


# ------------------------------------------------------------------------------- ABI behaviour on a device
def test_error_paths():
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_plan_create([64, 64, 64], [1, 1, 1], [sf.SF_BC_PERIODIC, sf.SF_BC_DIRICHLET, sf.SF_BC_PERIODIC])
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED  # mixed BCs
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_plan_create([48, 64, 64], [1, 1, 1], sf.SF_BC_PERIODIC)
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_plan_create([64, 64, 64], [1, 1, 1], sf.SF_BC_UNBOUNDED, op=sf.SF_OP_FD2)
    assert ei.value.status == sf.SF_ERR_UNSUPPORTED
    with pytest.raises(sf.SailffishError) as ei:
        sf.sf_plan_create([64, 64, 0], [1, 1, 1], sf.SF_BC_PERIODIC)
    assert ei.value.status == sf.SF_ERR_INVALID_ARG
    with Plan((16, 16, 16), (1, 1, 1), sf.SF_BC_PERIODIC, prec="f32") as p:
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_solve(p.plan)
        assert ei.value.status == sf.SF_ERR_STATE  # no source yet
        with pytest.raises(sf.SailffishError) as ei:
            sf.sf_curl(p.plan)
        assert ei.value.status == sf.SF_ERR_UNSUPPORTED
        assert sf.sf_device_bytes(p.plan) > 0


def test_user_stream_and_step_timing():
    import torch
    n = 32
    w = W.periodic3d_spectrum(n, kmax=8)
    f = rounded(w["f"], "f32")
    psi_o = O.periodic(f.astype(np.float64), w["L"], O.OP_PS)
    s = torch.cuda.Stream()
    with Plan(f.shape, tuple(L / n for L in w["L"]), sf.SF_BC_PERIODIC, prec="f32", stream=s.cuda_stream) as p:
        p.set_source(f)
        torch.cuda.synchronize()
        sf.sf_enable_step_timing(p.plan, 1)
        sf.sf_solve(p.plan)
        ms = sf.sf_step_times_ms(p.plan)
        assert len(ms) == 5 and all(t > 0 for t in ms)
        _report("psi", p.get(sf.SF_OUT_PSI), psi_o, "f32")
