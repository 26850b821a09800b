"""Hybrid (host-buffer) mode: every pointer is a HOST pointer, the LOR list is streamed through the
GPU in chunks on two streams.  Parity against the oracle on the same seeded inputs (north_star tolerances), including
a list longer than one chunk boundary pattern (several chunks + ragged tail is forced with a scanner slice) and
the ACCUMULATE semantics of the back projections."""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs
from test_gpu_parity import assert_back, assert_fwd

pytestmark = pytest.mark.gpu


def test_host_nontof_and_tof_small(cuda_device):
    n = 7_013
    c = inputs.config0(n_lors=n)
    g = c["geom"]
    xs, xe = torch.from_numpy(c["xstart"]), torch.from_numpy(c["xend"])
    img, y = torch.from_numpy(c["img"]), torch.from_numpy(c["y"])
    targs = (9.0, 7.0, 3.0, 27)
    tof = jp.make_tof(*targs)
    # non-TOF
    p = jp.jp_fwd_host(xs, xe, img, g.origin, g.voxsize)
    assert_fwd(p, oracle.fwd(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize))
    start = np.random.default_rng(1).random(g.n).astype(np.float32)
    b = jp.jp_back_host(xs, xe, y, torch.from_numpy(start.copy()), g.origin, g.voxsize)
    assert_back(b, start + oracle.back(c["xstart"], c["xend"], c["y"], g.n, g.origin, g.voxsize))   # accumulates
    # TOF sinogram
    ps = jp.jp_fwd_tof_sino_host(xs, xe, img, g.origin, g.voxsize, tof)
    assert_fwd(ps, oracle.fwd_tof_sino(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize, *targs))
    ys = np.random.default_rng(2).random((n, 27)).astype(np.float32)
    bs = jp.jp_back_tof_sino_host(xs, xe, torch.from_numpy(ys), torch.from_numpy(start.copy()), g.origin, g.voxsize, tof)
    assert_back(bs, start + oracle.back_tof_sino(c["xstart"], c["xend"], ys, g.n, g.origin, g.voxsize, *targs))
    # TOF listmode
    tb = np.random.default_rng(3).integers(-6, 7, n).astype(np.int16)
    pl = jp.jp_fwd_tof_lm_host(xs, xe, torch.from_numpy(tb), img, g.origin, g.voxsize, tof)
    assert_fwd(pl, oracle.fwd_tof_lm(c["xstart"], c["xend"], tb, c["img"], g.origin, g.voxsize, *targs[:3]))
    bl = jp.jp_back_tof_lm_host(xs, xe, torch.from_numpy(tb), y, torch.from_numpy(start.copy()), g.origin, g.voxsize, tof)
    assert_back(bl, start + oracle.back_tof_lm(c["xstart"], c["xend"], tb, c["y"], g.n, g.origin, g.voxsize, *targs[:3]))


def test_host_tof_sino_several_chunks(cuda_device):
    """2.4 M scanner LORs x 29 bins = three chunks of the TOF sinogram pipeline (1,048,320 LORs each) with a ragged
    tail; host result == device-pointer call bit for bit on the forward side, within tolerance on the adjoint"""
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    tof = jp.make_tof(tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    xs, xe = inputs.sinogram_lors(views=[5, 64, 100, 201], radial=range(-60, 61, 2))
    xs, xe = xs[:, :2_400_011].contiguous(), xe[:, :2_400_011].contiguous()
    n = xs.shape[1]
    ph = torch.from_numpy(inputs.phantom())
    p_host = jp.jp_fwd_tof_sino_host(xs, xe, ph, g.origin, g.voxsize, tof)
    p_dev = jp.jp_fwd_tof_sino(xs.to(cuda_device), xe.to(cuda_device), ph.to(cuda_device), g.origin, g.voxsize, tof)
    assert torch.equal(p_host, p_dev.cpu())
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=77)
    b_host = jp.jp_back_tof_sino_host(xs, xe, y, torch.zeros(g.n), g.origin, g.voxsize, tof)
    b_dev = jp.jp_back_tof_sino(xs.to(cuda_device), xe.to(cuda_device), y.to(cuda_device), g.n, g.origin, g.voxsize, tof)
    assert float((b_host - b_dev.cpu()).abs().max()) <= 1e-4 * float(b_dev.abs().max())


def test_host_errors(cuda_device):
    c = inputs.config0(n_lors=16)
    g = c["geom"]
    xs, xe = torch.from_numpy(c["xstart"]), torch.from_numpy(c["xend"])
    tof = jp.make_tof(9.0, 7.0, 3.0, 27)
    with pytest.raises(jp.JosephError):          # device tensor where a host tensor is required
        jp.jp_fwd_tof_sino_host(xs.to(cuda_device), xe.to(cuda_device), torch.from_numpy(c["img"]), g.origin, g.voxsize, tof)
    with pytest.raises(jp.JosephError):          # wrong TOF bin dtype
        jp.jp_fwd_tof_lm_host(xs, xe, torch.zeros(16, dtype=torch.int32), torch.from_numpy(c["img"]), g.origin, g.voxsize, tof)
