"""jp_gauss3d_static: the resolution-model smoothing for callers that cannot allocate device memory.

Some users of the library run where cudaMalloc / cudaMallocAsync are not an option: every byte of the GPU was
handed out when the reconstruction service started, or the calling thread sits in an acquisition loop that may
not stall on the allocator's lock, or the stream has no memory pool behind it.  For them jp_gauss3d_static keeps
the intermediate image of the three separable passes in a fixed 16 MiB array inside the library instead of
asking the allocator for it.  This file checks that entry point against the allocating one (jp_gauss3d, itself
compared with the float64 oracle in test_gpu_parity.py::test_resolution_model) and against the oracle directly.

The file is named so that pytest collects it LAST: with `pytest -x` a failure here cannot hide another test.
It must pass when run alone in a fresh process (the first call does the per-device set-up) and after the rest
of the suite (set-up possibly done, scratch full of an earlier call's values).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp

pytestmark = pytest.mark.gpu

GAUSS_MAX_ABS = 2e-6   # x max|oracle|: the bound test_resolution_model holds jp_gauss3d to


def test_static_scratch_matches_the_allocating_call_twice_in_a_row(cuda_device):
    """Two calls back to back, different images and shapes, both code paths of the smoothing (three generic passes;
    the fused two-kernel path for n2 % 4 == 0).  The second call finds the first one's intermediate in the shared
    scratch -- it is larger than the second image -- and must not be influenced by it."""
    sig = oracle.fwhm_to_sigma(4.5)
    vox = (2.0, 1.5, 2.78)
    rng = np.random.default_rng(2212)
    shapes = [(37, 70, 44), (19, 21, 45)]          # fused path first (113,960 voxels), then generic (17,955 voxels)
    for rep, shape in enumerate(shapes):
        x = rng.random(shape).astype(np.float32) * (1.0 + 99.0 * rep)   # second image on another scale
        xd = torch.as_tensor(x).to(cuda_device)
        want = jp.jp_gauss3d(xd, vox, sig)                               # existing path: cudaMallocAsync scratch
        got = torch.full_like(xd, float("nan"))                           # output buffer supplied by the caller
        ret = jp.jp_gauss3d_static(xd, vox, sig, 3.0, out=got)
        assert ret is got
        torch.cuda.synchronize(cuda_device)
        ref = oracle.gauss3d(x, vox, sig)
        g = got.cpu().numpy()
        assert np.isfinite(g).all()
        assert np.abs(g - want.cpu().numpy()).max() <= GAUSS_MAX_ABS * np.abs(ref).max(), f"call {rep}: differs from jp_gauss3d"
        assert torch.equal(got, want), f"call {rep}: same kernels, same order of operations: expected bit-identical"
        assert np.abs(g - ref).max() <= GAUSS_MAX_ABS * np.abs(ref).max(), f"call {rep}: differs from the oracle"
        # in place (in == out), the way the OSEM loop applies the model
        xi = xd.clone()
        jp.jp_gauss3d_static(xi, vox, sig, 3.0, out=xi)
        assert torch.equal(xi, want), f"call {rep}: in-place result differs"


def test_static_scratch_same_image_twice_gives_the_same_result(cuda_device):
    """the array keeps the last call's contents; a repeat of the same call on the same stream must not see them"""
    sig = oracle.fwhm_to_sigma(4.5)
    x = torch.rand((40, 40, 24), device=cuda_device, generator=torch.Generator(device=cuda_device).manual_seed(5))
    a, b = torch.empty_like(x), torch.empty_like(x)
    jp.jp_gauss3d_static(x, (2.0, 2.0, 2.0), sig, 3.0, out=a)
    jp.jp_gauss3d_static(x, (2.0, 2.0, 2.0), sig, 3.0, out=b)
    assert torch.equal(a, b)
    assert torch.equal(a, jp.jp_gauss3d(x, (2.0, 2.0, 2.0), sig))


def test_static_scratch_refuses_images_beyond_its_limit(cuda_device):
    """one voxel over JP_GAUSS3D_STATIC_MAX_VOXELS: a clear error before anything is enqueued, `out` untouched;
    exactly at the limit the call goes through"""
    assert jp.GAUSS3D_STATIC_MAX_VOXELS == 4194304
    sig = oracle.fwhm_to_sigma(4.5)
    big = torch.ones((4097, 32, 32), device=cuda_device)                 # 4,195,328 voxels > 4,194,304
    out = torch.full_like(big, -1.0)
    with pytest.raises(jp.JosephError, match="exceeds the built-in scratch"):
        jp.jp_gauss3d_static(big, (2.0, 2.0, 2.0), sig, 3.0, out=out)
    torch.cuda.synchronize(cuda_device)
    assert bool((out == -1.0).all())
    full = torch.ones((4096, 32, 32), device=cuda_device)                # == the limit
    o2 = torch.empty_like(full)
    jp.jp_gauss3d_static(full, (2.0, 2.0, 2.0), sig, 3.0, out=o2)
    assert torch.equal(o2, jp.jp_gauss3d(full, (2.0, 2.0, 2.0), sig))
    centre = float(o2[2048, 16, 16])
    assert abs(centre - 1.0) < 2e-6                                       # normalised taps: interior of a constant image


def test_static_scratch_at_the_papers_image_size(cuda_device):
    """200 x 200 x 96 (PAPER.md:94 geometry of configs[1]-[4]) fits the built-in scratch; sampled voxels against
    the oracle's definition evaluated only where needed would be slow, so compare with jp_gauss3d (oracle-checked)
    on the whole image"""
    sig = oracle.fwhm_to_sigma(4.5)
    x = torch.rand((200, 200, 96), device=cuda_device, generator=torch.Generator(device=cuda_device).manual_seed(7))
    out = torch.empty_like(x)
    jp.jp_gauss3d_static(x, (2.0, 2.0, 2.0), sig, 3.0, out=out)
    assert torch.equal(out, jp.jp_gauss3d(x, (2.0, 2.0, 2.0), sig))
