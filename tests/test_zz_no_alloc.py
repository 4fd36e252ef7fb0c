"""arche_fft3d_static: the 3D transform for callers that cannot allocate (scratch in a file-scope device array of the
library image, include/arche.h).  Collected last on purpose (pytest -x): a failure here hides nothing.

Checked against the existing path, arche_fft3d with caller scratch, on the same inputs: the same kernels run in the
same order, so the outputs must be bit-identical (the FFT parity tolerance against the oracle, 1e-13 * max * log2 N,
is asserted as well, against the existing path's result).  Two calls in a row with different inputs: the array keeps
the first call's contents and the second must not see them.  torch's allocator statistics bracket the calls: the
output tensors are made before, so no device allocation may happen in between.
"""
import numpy as np
import pytest

import arche_inputs as ai

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test run without a CUDA device")
    return torch


def _gpu(cfg, **kw):
    from paper_2606_13283_b200 import Arche
    return Arche(cfg, **kw)


@pytest.mark.parametrize("shape", [(64, 64, 64), (16, 24, 36), (9, 12, 18)])
def test_fft3d_static_matches_fft3d_twice_in_a_row(torch_cuda, shape):
    torch = torch_cuda
    nz, ny, nx = shape
    g = _gpu(ai.make_small(grid=(nx, ny, nz)))
    rng = np.random.default_rng(4242 + nx)
    a1 = torch.as_tensor(rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).cuda()
    a2 = torch.as_tensor(rng.standard_normal(shape) * 3.0 - 2j * rng.standard_normal(shape)).cuda()
    ref1 = g.fft3d(a1, -1)
    ref2 = g.fft3d(a2, +1)
    out1, out2 = torch.empty_like(a1), torch.empty_like(a2)
    torch.cuda.synchronize()
    n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]
    g.fft3d_static(a1, -1, out=out1)           # first call
    g.fft3d_static(a2, +1, out=out2)           # second call, straight after, on the array the first one left behind
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc
    for got, ref in ((out1, ref1), (out2, ref2)):
        got, ref = got.cpu().numpy(), ref.cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max() * np.log2(ref.size)
        assert np.array_equal(got, ref)
    # in place, and the forward-inverse round trip through the static path alone
    buf = a1.clone()
    g.fft3d_static(buf, -1, out=buf)
    g.fft3d_static(buf, +1, out=buf)
    torch.cuda.synchronize()
    back = buf.cpu().numpy() / a1.numel()
    assert np.abs(back - a1.cpu().numpy()).max() < 1e-13 * np.log2(a1.numel()) * float(a1.abs().max())


def test_fft3d_static_rejects_grids_beyond_its_maximum(torch_cuda):
    from paper_2606_13283_b200 import ArcheError
    torch = torch_cuda
    g = _gpu(ai.make_small(grid=(96, 64, 64)))   # 393 216 points > 64^3
    a = torch.zeros((64, 64, 96), dtype=torch.complex128, device="cuda")
    with pytest.raises(ArcheError, match="ARCHE_FFT3D_STATIC_MAX_POINTS"):
        g.fft3d_static(a, -1)
    g.fft3d(a, -1)   # the existing path still serves that grid
