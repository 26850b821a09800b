"""Hybrid (host-buffer) mode: every pointer is a HOST pointer; a jp_hybrid handle splits the LOR list
over its workers (one per device; several workers on ONE GPU exercise the fan-out and the summation of the partial
images on a single-GPU box), keeps the shards resident and sums the back projections on the host.  Parity against the
oracle on the same seeded inputs (north_star tolerances), forward results bit-equal between 1 and several workers,
ragged shards, more workers than work, and the ACCUMULATE semantics of the back projections."""
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


@pytest.mark.parametrize("ragged", [False, True])
def test_host_tof_sino_scanner(cuda_device, ragged):
    """562 k scanner LORs x 29 bins through the one-shot host calls.  Whole tracks: the shard is a regular sinogram and
    the host result equals the PLANNED device call bit for bit (same track-tile kernel); with a ragged tail the list is
    not regular and the host result equals the unplanned device call bit for bit.  Adjoint within tolerance."""
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    tof = jp.make_tof(tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    xs, xe = inputs.sinogram_lors(views=[5, 64, 100, 201], radial=range(-60, 61, 2))
    if ragged:
        xs, xe = xs[:, :400_011].contiguous(), xe[:, :400_011].contiguous()
    n = xs.shape[1]
    ph = torch.from_numpy(inputs.phantom())
    xsd, xed, phd = xs.to(cuda_device), xe.to(cuda_device), ph.to(cuda_device)
    p_host = jp.jp_fwd_tof_sino_host(xs, xe, ph, g.origin, g.voxsize, tof)
    if ragged:
        p_dev = jp.jp_fwd_tof_sino(xsd, xed, phd, g.origin, g.voxsize, tof)
    else:
        plan = jp.SinoPlan(xsd, xed)
        assert plan.regular
        p_dev = jp.jp_fwd_tof_sino_planned(plan, phd, g.origin, g.voxsize, tof)
    assert torch.equal(p_host, p_dev.cpu())
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=77)
    b_host = jp.jp_back_tof_sino_host(xs, xe, y, torch.zeros(g.n), g.origin, g.voxsize, tof)
    b_dev = jp.jp_back_tof_sino(xsd, xed, y.to(cuda_device), g.n, g.origin, g.voxsize, tof)
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


def _devices_variants():
    nd = torch.cuda.device_count()
    v = [[0], [0, 0, 0]]
    if nd > 1:
        v.append(list(range(nd)))
    return v


def test_hybrid_handle_nontof_workers(cuda_device):
    """jp_hybrid over 1 worker, 3 workers on device 0 and (when present) all visible devices: 14 tracks of 2304 scanner
    LORs (shards cut at track boundaries: 5 + 5 + 4 tracks) -- forward bit-equal between the variants and equal to
    the device call, back within tolerance of the oracle, accumulate semantics; then a ragged irregular list"""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    xs, xe = inputs.sinogram_lors(views=[3, 64], radial=[-30, -9, 0, 1, 17, 40, 70])
    n = xs.shape[1]
    img = torch.from_numpy(ph)
    y = inputs.uniform_values(n, 0.0, 1.0, seed=5)
    ref = oracle.fwd(xs.numpy(), xe.numpy(), ph, g.origin, g.voxsize)
    bref = oracle.back(xs.numpy(), xe.numpy(), y.numpy(), g.n, g.origin, g.voxsize)
    plan = jp.SinoPlan(xs.to(cuda_device), xe.to(cuda_device))
    p_dev = jp.jp_fwd_planned(plan, img.to(cuda_device), g.origin, g.voxsize).cpu()   # shards are whole tracks: same kernel
    for devs in _devices_variants():
        h = jp.Hybrid(devs)
        assert h.workers == len(devs)
        h.set_lors(xs, xe)
        p = h.fwd(img, g.origin, g.voxsize)
        assert torch.equal(p, p_dev)
        assert_fwd(p, ref)
        start = torch.full(g.n, 2.0)
        b = h.back(y, start, g.origin, g.voxsize)
        assert_back(b - 2.0, bref)
        # the list can be replaced; a ragged list is not a regular sinogram
        h.set_lors(xs[:, :9_001].contiguous(), xe[:, :9_001].contiguous())
        p2 = h.fwd(img, g.origin, g.voxsize)
        assert_fwd(p2, ref[:9_001])
        if len(devs) == 1:    # one shard: the same tiles as the device call on that list (the ragged tail goes per LOR)
            assert torch.equal(p2, jp.jp_fwd(xs[:, :9_001].contiguous().to(cuda_device), xe[:, :9_001].contiguous().to(cuda_device),
                                             img.to(cuda_device), g.origin, g.voxsize).cpu())
        h.destroy()
    # more workers than work
    h = jp.Hybrid([0] * 5)
    h.set_lors(xs[:, :700].contiguous(), xe[:, :700].contiguous())
    assert_fwd(h.fwd(img, g.origin, g.voxsize), ref[:700])
    h.set_lors(xs[:, :0].contiguous(), xe[:, :0].contiguous())
    assert h.fwd(img, g.origin, g.voxsize).numel() == 0
    h.destroy()


def test_hybrid_handle_tof(cuda_device):
    """TOF sinogram (regular shards: track tiles) and TOF listmode (a listmode plan per shard) on the handle, 1 and 3
    workers, against the oracle"""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    tp = inputs.TofParams()
    targs = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    tof = jp.make_tof(*targs)
    xs, xe = inputs.sinogram_lors(views=[64, 130], radial=[-20, 0, 7, 33])
    n = xs.shape[1]
    sel = np.arange(0, n, 7)
    img = torch.from_numpy(ph)
    ref = oracle.fwd_tof_sino(xs.numpy()[:, sel], xe.numpy()[:, sel], ph, g.origin, g.voxsize, *targs)
    y = torch.zeros((n, 29))
    y[sel] = inputs.uniform_values((sel.size, 29), 0.0, 1.0, seed=6)
    bref = oracle.back_tof_sino(xs.numpy()[:, sel], xe.numpy()[:, sel], y[sel].numpy(), g.n, g.origin, g.voxsize, *targs)
    ex, ee, tb = inputs.listmode_events(60_000, seed=9, img=ph, chunk=200_000)
    lref = oracle.fwd_tof_lm(ex.numpy(), ee.numpy(), tb.numpy(), ph, g.origin, g.voxsize, *targs[:3])
    yl = inputs.uniform_values(60_000, 0.5, 2.0, seed=7)
    lbref = oracle.back_tof_lm(ex.numpy(), ee.numpy(), tb.numpy(), yl.numpy(), g.n, g.origin, g.voxsize, *targs[:3])
    first = None
    for devs in _devices_variants():
        h = jp.Hybrid(devs)
        h.set_lors(xs, xe)
        p = h.fwd_tof_sino(img, g.origin, g.voxsize, tof)
        assert_fwd(p[sel], ref)
        if first is None:
            first = p
        assert torch.equal(p, first)                       # forward: independent of the number of workers
        b = h.back_tof_sino(y, torch.zeros(g.n), g.origin, g.voxsize, tof)
        assert_back(b, bref)
        h.set_lors(ex, ee, tb, g.n, g.origin, g.voxsize, tof)
        assert_fwd(h.fwd_tof_lm(img), lref)
        assert_back(h.back_tof_lm(yl, torch.zeros(g.n)), lbref)
        with pytest.raises(jp.JosephError):
            jp.Hybrid(devs).fwd(img, g.origin, g.voxsize)   # no list set
        h.destroy()


def test_hybrid_tof_listmode_unsnapped_events(cuda_device):
    """TOF listmode on the handle with end points that are NOT crystal centres (seeded jitter of a few mm, so no two
    events share a line): every shard's plan is sparse and takes the image-brick kernels, whose > 48 KB dynamic
    shared memory has to be enabled on EACH device that launches them.  Runs over 1 worker, 3 workers on device 0
    and, where more than one GPU is visible, one worker per GPU."""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    tp = inputs.TofParams()
    targs = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas)
    tof = jp.make_tof(*targs, tp.n_tofbins)
    n = 40_003
    ex, ee, tb = inputs.listmode_events(n, seed=inputs.BASE_SEED + 57, img=ph, chunk=200_000)
    rng = np.random.default_rng(57)
    ex = (ex + torch.from_numpy(rng.uniform(-2.0, 2.0, size=tuple(ex.shape)).astype(np.float32))).contiguous()
    ee = (ee + torch.from_numpy(rng.uniform(-2.0, 2.0, size=tuple(ee.shape)).astype(np.float32))).contiguous()
    img = torch.from_numpy(ph)
    yl = inputs.uniform_values(n, 0.5, 2.0, seed=58)
    lref = oracle.fwd_tof_lm(ex.numpy(), ee.numpy(), tb.numpy(), ph, g.origin, g.voxsize, *targs)
    lbref = oracle.back_tof_lm(ex.numpy(), ee.numpy(), tb.numpy(), yl.numpy(), g.n, g.origin, g.voxsize, *targs)
    for devs in _devices_variants():
        h = jp.Hybrid(devs)
        h.set_lors(ex, ee, tb, g.n, g.origin, g.voxsize, tof)
        assert_fwd(h.fwd_tof_lm(img), lref)
        assert_back(h.back_tof_lm(yl, torch.zeros(g.n)), lbref)
        assert_back(h.back_tof_lm(yl, torch.full(g.n, 1.0)) - 1.0, lbref)     # accumulates
        h.destroy()
