"""Test-side helpers that drive the CUDA path through the C ABI (via the thin binding) and return
numpy arrays.  Argument marshalling only; torch supplies device memory.  Arrays are [z, y, x]."""
import numpy as np
import torch

import paper_2301_01145_b200 as sf

TOL = {"f64": 1e-12, "f32": 2e-5}  # BASELINE.json north_star: relative L2 vs the fp64 oracle


def np_dtype(prec):
    return np.float32 if prec == "f32" else np.float64


def sf_prec(prec):
    return sf.SF_F32 if prec == "f32" else sf.SF_F64


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def rounded(f, prec):
    """input as the plan sees it (reading A23: fp32 plans consume fp32-rounded inputs; the oracle gets
    the same rounded values widened to double)"""
    return np.ascontiguousarray(np.asarray(f, dtype=np_dtype(prec)))


class Plan:
    """context manager around sf_plan_create / sf_plan_destroy"""

    def __init__(self, shape_zyx, h_xyz, bc, grid=sf.SF_GRID_CELL_CENTRE, op=sf.SF_OP_PSEUDO_SPECTRAL, prec="f64",
                 ncomp=1, rhs_sign=1.0, eps_over_h=0.0, stream=None):
        self.shape = tuple(shape_zyx)
        self.prec = prec
        self.ncomp = ncomp
        n = list(reversed(self.shape))
        self.plan = sf.sf_plan_create(n, list(h_xyz)[: len(n)], bc, grid, op, sf_prec(prec), ncomp=ncomp,
                                      rhs_sign=rhs_sign, eps_over_h=eps_over_h, stream=stream)
        self.keep = []

    def __enter__(self):
        return self

    def __exit__(self, *a):
        sf.sf_synchronize(self.plan)
        sf.sf_plan_destroy(self.plan)
        self.plan = None

    def set_source(self, f, device=True):
        f = rounded(f, self.prec)
        if device:
            t = torch.from_numpy(f).cuda()
            self.keep.append(t)
            sf.sf_set_source(self.plan, t)
        else:
            sf.sf_set_source(self.plan, f)
            sf.sf_synchronize(self.plan)

    def set_faces(self, faces, device=True):
        for (axis, side), g in faces.items():
            g = rounded(g, self.prec)
            if device:
                t = torch.from_numpy(g).cuda()
                self.keep.append(t)
                sf.sf_set_bc_values(self.plan, axis, side, t)
            else:
                sf.sf_set_bc_values(self.plan, axis, side, g)
        sf.sf_synchronize(self.plan)

    def get(self, field, comp=0, device=False):
        if device:
            t = torch.empty(self.shape, dtype=torch.float32 if self.prec == "f32" else torch.float64, device="cuda")
            sf.sf_get_output(self.plan, field, comp, t)
            sf.sf_synchronize(self.plan)
            return t.cpu().numpy()
        out = np.empty(self.shape, dtype=np_dtype(self.prec))
        sf.sf_get_output(self.plan, field, comp, out)
        return out
