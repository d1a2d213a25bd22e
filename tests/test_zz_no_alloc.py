"""holo_normalize_static (include/holo.h): the allocation-free entry point, against the existing path (holo_normalize on a
handle) and the oracle, on two calls in a row.  Named test_zz_* so that pytest collects it LAST: the suite runs with
`pytest -x`, and a failure here must not hide the parity tests.  Passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import oracle
from tests.util import rel_l2

pytestmark = pytest.mark.gpu

TOL = 2e-7          # the bound tests/test_gpu_parity.py::test_normalize_and_fftshift uses: one rounding of the scale, one of the product


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    return torch


def _image(rng, ny, nx):
    return (rng.random((ny, nx)) * 1e9 + 1e7).astype(np.float32)            # the magnitude of a real PCA image


def _existing_path(torch, M):
    """holo_normalize on a handle (in place): the path that exists since round 2."""
    from paper_2004_00923_b200 import Holo
    ny, nx = M.shape
    h = Holo(nx, ny, 2, 785e-9, 20e-6, 0.2, 1, 2)
    d = torch.from_numpy(M).cuda()
    h.normalize(d)
    torch.cuda.synchronize()
    out = d.cpu().numpy()
    h.close()
    return out


def test_normalize_static_matches_existing_path_two_calls_in_a_row(torch_cuda):
    torch = torch_cuda
    from paper_2004_00923_b200 import normalize_static
    rng = np.random.default_rng(20040923)
    # first a large image (1024 x 1024: 256 partial sums in the static scratch), then a small one (64 x 32, the existing path
    # needs power-of-two frames: ONE incomplete chunk): the second call finds 255 stale partials of the first behind its own and
    # must not read them; then the first image again, in place.  (Ragged sizes: the next test, against the oracle.)
    A, B = _image(rng, 1024, 1024), _image(rng, 32, 64) * 3.0
    refA, refB = _existing_path(torch, A), _existing_path(torch, B)
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    oA, oB = torch.empty_like(dA), torch.empty_like(dB)
    normalize_static(dA, oA, 1024, 1024)                     # (the first call on the device also resolves the scratch address)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    normalize_static(dA, oA, 1024, 1024)                     # two calls in a row on one stream, no synchronisation between them
    normalize_static(dB, oB, 64, 32)
    normalize_static(dA, dA, 1024, 1024)                     # in place
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the call took device memory"
    gA, gB, gA2 = oA.cpu().numpy(), oB.cpu().numpy(), dA.cpu().numpy()
    for got, ref, src in ((gA, refA, A), (gB, refB, B), (gA2, refA, A)):
        assert rel_l2(got, ref) <= TOL                                       # the existing CUDA path
        assert rel_l2(got, oracle.normalize(src.astype(np.float64))) <= TOL  # and the oracle
        assert abs(got.astype(np.float64).mean() - 1.0) <= 1e-6
    assert np.array_equal(gA, gA2)                           # fixed-order reduction: bit-reproducible, in place or not
    # a zero image stays zero (as holo_normalize), whatever the previous call left in the scratch
    Z0 = torch.zeros((64, 48), dtype=torch.float32, device="cuda")
    normalize_static(Z0, Z0, 48, 64)
    torch.cuda.synchronize()
    assert not bool(Z0.any())


def test_normalize_static_other_stream_and_sizes(torch_cuda):
    torch = torch_cuda
    from paper_2004_00923_b200 import normalize_static
    rng = np.random.default_rng(7)
    st = torch.cuda.Stream()
    for ny, nx in ((1, 1), (3, 4097), (16, 256), (2048, 2048)):
        M = _image(rng, ny, nx)
        d = torch.from_numpy(M).cuda()
        o = torch.empty_like(d)
        torch.cuda.synchronize()
        normalize_static(d, o, nx, ny, st)
        st.synchronize()
        assert rel_l2(o.cpu().numpy(), oracle.normalize(M.astype(np.float64))) <= TOL, (ny, nx)


def test_normalize_static_rejects_what_it_cannot_hold(torch_cuda):
    torch = torch_cuda
    from paper_2004_00923_b200 import normalize_static, HoloError, HOLO_ERR_ARG
    d = torch.ones((16, 16), dtype=torch.float32, device="cuda")
    o = torch.full((16, 16), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(HoloError) as e:                     # 4096 x 4097 pixels: one row more than the static scratch covers
        normalize_static(d, o, 4097, 4096)
    assert e.value.code == HOLO_ERR_ARG and "HOLO_STATIC_MAX_PIXELS" in str(e.value)
    for nx, ny in ((0, 16), (16, -1)):
        with pytest.raises(HoloError) as e:
            normalize_static(d, o, nx, ny)
        assert e.value.code == HOLO_ERR_ARG
    with pytest.raises(HoloError):
        normalize_static(0, o, 16, 16)
    torch.cuda.synchronize()
    assert bool((o == 7.0).all())                           # nothing was launched on an error return
    normalize_static(d, o, 16, 16)                          # and the entry point still works afterwards
    torch.cuda.synchronize()
    assert bool((o == 1.0).all())
