"""sf_probe_dft16_stage (include/sailffish.h): the one stage of the pencil transforms that could run as
a matrix product, on the fp32 pipe (variant 0) and on the tensor cores (variants 1, 2).  All three must compute the same
16-point DFTs; the timing comparison is in profiles/ and DESIGN.md section 6."""
import numpy as np
import pytest
import torch

import paper_2301_01145_b200 as sf
import workloads as W

pytestmark = pytest.mark.gpu


def _expected(x, reps):
    """x [T, 16 q, 16 o, 32 lane] complex: thread (o, lane) holds value q; after the exchange thread q holds the values
    of all o and transforms over o: out[T, k, q, lane] = 1/4 sum_o x[T, q, o, lane] exp(-2 pi i k o / 16)"""
    y = x
    for _ in range(reps):
        y = 0.25 * np.fft.fft(y, axis=2)        # [T, q, k, lane]
        y = np.transpose(y, (0, 2, 1, 3))       # [T, k, q, lane]: value index k, thread index q
    return y


@pytest.mark.parametrize("variant,tol", [(0, 2e-6), (1, 5e-6), (2, 5e-3)])
def test_probe_variants_compute_the_dft(variant, tol):
    T, reps = 37, 3
    r = W.Rng(777).normal(2 * T * 16 * 512).reshape(T, 16, 512, 2)
    x = (r[..., 0] + 1j * r[..., 1]).astype(np.complex64)
    src = torch.from_numpy(x).cuda()
    dst = torch.zeros_like(src)
    ms = sf.sf_probe_dft16_stage(variant, reps, T, src, dst)
    assert ms > 0.0
    got = dst.cpu().numpy().astype(np.complex128).reshape(T, 16, 16, 32)
    ref = _expected(x.astype(np.complex128).reshape(T, 16, 16, 32), reps)
    err = np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel())
    print(f"probe variant {variant}: rel-L2 {err:.3e} ({ms * 1e3:.1f} us for {T} tiles x {reps} stages)")
    assert err <= tol
