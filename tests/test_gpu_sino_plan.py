"""Sinogram plan (jp_sino_plan_create) and the planned TOF sinogram calls: parity against the float64 oracle through the
C ABI, element by element, plus the plan's own decisions (track length, regularity) which are integers: bit exact.

A regular list is K tracks (identical transaxial end points) x T LORs with one axial pattern; the track-tile kernels
factor the q1 half of Joseph's interpolation through shared-memory rows and stage the adjoint in shared memory
(PAPER.md:33, :35, :43, :44 / :46).  Tolerances are BASELINE.json north_star's (test_gpu_parity.py).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs
from test_gpu_parity import ADJ_GAP, adj_gap, assert_back, assert_fwd, dev

pytestmark = pytest.mark.gpu


def mini_sinogram(n_tracks, zs_vals, ze_vals, radius=150.0, seed=0, extra_tracks=()):
    """K tracks with random transaxial end points on a circle (plus `extra_tracks`: explicit (xs, ys, xe, ye)), each
    with the axial pattern zs_vals x ze_vals (zs slow, ze fast, like ring pairs).  float32 (3, K*T) arrays."""
    rng = np.random.default_rng(seed)
    a, b = rng.uniform(0, 2 * np.pi, n_tracks), rng.uniform(0, 2 * np.pi, n_tracks)
    tr = np.stack([radius * np.cos(a), radius * np.sin(a), radius * np.cos(b), radius * np.sin(b)], 1)
    if len(extra_tracks):
        tr = np.concatenate([tr, np.asarray(extra_tracks, dtype=np.float64)], 0)
    tr = tr.astype(np.float32)
    zs, ze = np.meshgrid(np.asarray(zs_vals, dtype=np.float32), np.asarray(ze_vals, dtype=np.float32), indexing="ij")
    zs, ze = zs.ravel(), ze.ravel()
    K, T = tr.shape[0], zs.size
    xs = np.empty((3, K * T), dtype=np.float32)
    xe = np.empty((3, K * T), dtype=np.float32)
    xs[0], xs[1], xs[2] = np.repeat(tr[:, 0], T), np.repeat(tr[:, 1], T), np.tile(zs, K)
    xe[0], xe[1], xe[2] = np.repeat(tr[:, 2], T), np.repeat(tr[:, 3], T), np.tile(ze, K)
    return xs, xe, K, T


@pytest.mark.parametrize("width,nbins,coff,nz", [(20.0, 13, 0.0, 20), (9.0, 27, 2.5, 23), (6.0, 41, 0.0, 20),
                                                (4.0, 61, -1.0, 12), (2.5, 63, 0.0, 8)])
def test_planned_tof_sino_small(cuda_device, width, nbins, coff, nz):
    """every compiled window size (4, 6, 8, 12) and the too-wide fallback; T = nz^2 (400, 529: slices of 384 + a
    ragged one); tracks along both transaxial axes, an exact 45 degree tie, a track that misses, a zero-length one"""
    g = inputs.GEOM_SMALL
    zv = np.linspace(-38.0, 38.0, nz)
    extra = [(-150.0, -150.0, 150.0, 150.0), (-150.0, 20.0, 150.0, 20.0), (7.0, -150.0, 7.0, 150.0),
             (-150.0, 140.0, 150.0, 149.0), (30.0, 40.0, 30.0, 40.0)]
    xs, xe, K, T = mini_sinogram(11, zv, zv, seed=nbins, extra_tracks=extra)
    n = K * T
    img = np.random.default_rng(1).uniform(0, 1, g.n).astype(np.float32)
    sigma, nsig = 7.0, 3.0
    tof = jp.make_tof(width, sigma, nsig, nbins, coff)
    xsd, xed, imgd = dev(xs, cuda_device), dev(xe, cuda_device), dev(img, cuda_device)
    plan = jp.SinoPlan(xsd, xed)
    assert plan.regular and plan.track_length == T and plan.n_tracks == K and plan.n == n   # integers: bit exact
    p = jp.jp_fwd_tof_sino_planned(plan, imgd, g.origin, g.voxsize, tof)
    ref = oracle.fwd_tof_sino(xs, xe, img, g.origin, g.voxsize, width, sigma, nsig, nbins, center_offset=coff)
    assert (ref > 0).mean() > 0.05
    assert_fwd(p, ref)
    y = np.random.default_rng(int(width * 10)).uniform(-0.5, 1, (n, nbins)).astype(np.float32)
    b = jp.jp_back_tof_sino_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(xs, xe, y, g.n, g.origin, g.voxsize, width, sigma, nsig, nbins,
                                        center_offset=coff))
    assert adj_gap(p, dev(y, cuda_device), imgd, b) <= ADJ_GAP
    # ACCUMULATE semantics
    b2 = jp.jp_back_tof_sino_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof, img=torch.full_like(b, 2.0))
    assert torch.allclose(b2 - 2.0, b, rtol=1e-4, atol=1e-3)
    plan.destroy()


def test_planned_steep_pattern_takes_the_per_lor_path(cuda_device):
    """an axial pattern steeper than some tracks are long transaxially: on those tracks a LOR may have principal
    axis z, so the whole track takes the per-LOR path inside the tile kernel (all three principal axes occur)"""
    g = inputs.GEOM_SMALL
    zv = np.linspace(-60.0, 60.0, 20)
    extra = [(-20.0, 3.0, 25.0, 5.0), (1.0, -30.0, 2.0, 31.0), (-150.0, 0.5, 150.0, -0.5)]
    xs, xe, K, T = mini_sinogram(5, zv, zv, seed=3, extra_tracks=extra)
    ax = oracle.classify(xs, xe, g.n, g.origin, g.voxsize)
    assert set(np.unique(ax)) == {0, 1, 2}
    img = np.random.default_rng(2).uniform(0, 1, g.n).astype(np.float32)
    args = (9.0, 7.0, 3.0, 27)
    tof = jp.make_tof(*args)
    xsd, xed, imgd = dev(xs, cuda_device), dev(xe, cuda_device), dev(img, cuda_device)
    plan = jp.SinoPlan(xsd, xed)
    assert plan.regular
    p = jp.jp_fwd_tof_sino_planned(plan, imgd, g.origin, g.voxsize, tof)
    assert_fwd(p, oracle.fwd_tof_sino(xs, xe, img, g.origin, g.voxsize, *args))
    y = np.random.default_rng(4).uniform(0, 1, (K * T, 27)).astype(np.float32)
    b = jp.jp_back_tof_sino_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(xs, xe, y, g.n, g.origin, g.voxsize, *args))


def test_plan_of_an_irregular_list(cuda_device):
    """random chords are not tracks: the plan keeps a copy and the planned calls equal the unplanned ones bit for bit
    (forward; the adjoint within the atomics' rounding); near-regular lists must be rejected too"""
    c = inputs.config0(n_lors=9_000)
    g = c["geom"]
    args = (9.0, 7.0, 3.0, 27)
    tof = jp.make_tof(*args)
    xsd, xed, imgd = dev(c["xstart"], cuda_device), dev(c["xend"], cuda_device), dev(c["img"], cuda_device)
    plan = jp.SinoPlan(xsd, xed)
    assert not plan.regular and plan.n == 9_000
    p = jp.jp_fwd_tof_sino_planned(plan, imgd, g.origin, g.voxsize, tof)
    assert torch.equal(p, jp.jp_fwd_tof_sino(xsd, xed, imgd, g.origin, g.voxsize, tof))
    y = np.random.default_rng(0).uniform(0, 1, (9_000, 27)).astype(np.float32)
    b = jp.jp_back_tof_sino_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(c["xstart"], c["xend"], y, g.n, g.origin, g.voxsize, *args))
    plan.destroy()
    # a regular list with ONE axial value changed, and one with a short last track, are not regular
    zv = np.linspace(-30.0, 30.0, 10)
    xs, xe, K, T = mini_sinogram(6, zv, zv, seed=9)
    xs2 = xs.copy()
    xs2[2, 3 * T + 17] += 0.5
    assert not jp.SinoPlan(dev(xs2, cuda_device), dev(xe, cuda_device)).regular
    assert not jp.SinoPlan(dev(xs[:, :-5], cuda_device), dev(xe[:, :-5], cuda_device)).regular
    assert jp.SinoPlan(dev(xs, cuda_device), dev(xe, cuda_device)).regular


def test_planned_adjoint_dynamic_range_and_nonfinite(cuda_device):
    """the fixed-point staging of the tile adjoint: y spanning 6 decades and both signs inside one slice stays within
    the tolerance (error <= 1.2e-7 x slice max per contribution); a slice whose y holds Inf / NaN takes the per-LOR
    float path, so the non-finite values land exactly where the oracle puts them and every other voxel stays right"""
    g = inputs.GEOM_SMALL
    zv = np.linspace(-38.0, 38.0, 20)
    xs, xe, K, T = mini_sinogram(6, zv, zv, seed=21, extra_tracks=[(-150.0, 10.0, 150.0, -14.0)])
    n = K * T
    args = (9.0, 7.0, 3.0, 27)
    tof = jp.make_tof(*args)
    plan = jp.SinoPlan(dev(xs, cuda_device), dev(xe, cuda_device))
    rng = np.random.default_rng(8)
    y = (10.0 ** rng.uniform(-6, 0, (n, 27)) * rng.choice([-1.0, 1.0], (n, 27))).astype(np.float32)
    b = jp.jp_back_tof_sino_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(xs, xe, y, g.n, g.origin, g.voxsize, *args))
    # non-finite: one Inf and one NaN on LORs of the last track that cross the image
    y2 = rng.uniform(0, 1, (n, 27)).astype(np.float32)
    j = (K - 1) * T + np.array([T // 2, T // 2 + 7])
    y2[j[0], 13] = np.inf
    y2[j[1], 12] = np.nan
    b2 = jp.jp_back_tof_sino_planned(plan, dev(y2, cuda_device), g.n, g.origin, g.voxsize, tof).cpu().numpy()
    # the oracle sums y x weight over ALL bins, so its Inf x 0 poisons every plane of the LOR; the CUDA paths only
    # visit the bins inside the truncated kernel (weights outside are exactly zero), so they poison the planes on which
    # the bad bin has weight: a subset of the oracle's set, identical between the tile path and the per-LOR path
    ref_bad = ~np.isfinite(oracle.back_tof_sino(xs, xe, y2, g.n, g.origin, g.voxsize, *args))
    bu = jp.jp_back_tof_sino(dev(xs, cuda_device), dev(xe, cuda_device), dev(y2, cuda_device), g.n, g.origin, g.voxsize,
                             tof).cpu().numpy()
    bad = ~np.isfinite(b2)
    assert bad.any() and not bad.all()
    assert np.array_equal(bad, ~np.isfinite(bu)) and not (bad & ~ref_bad).any()
    y0 = y2.copy()
    y0[~np.isfinite(y0)] = 0.0
    ref0 = oracle.back_tof_sino(xs, xe, y0, g.n, g.origin, g.voxsize, *args)
    assert np.abs(b2[~bad] - ref0[~bad]).max() <= 1e-4 * np.abs(ref0).max()           # nothing finite was dropped


def test_planned_tof_sino_scanner_views(cuda_device):
    """configs[2] structure: two views (incl. the 45 degree tie view 64) x 9 radial bins x all 2304 ring pairs of the
    48-ring scanner on the 200x200x96 phantom; the oracle on every 5th LOR; planned == unplanned elsewhere"""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    tofp = inputs.TofParams()
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    tof = jp.make_tof(*args)
    xs, xe = inputs.sinogram_lors(views=[64, 240], radial=[-128, -64, -40, -3, 0, 25, 63, 64, 65])
    n = xs.shape[1]
    xsd, xed, imgd = xs.to(cuda_device), xe.to(cuda_device), dev(ph, cuda_device)
    plan = jp.SinoPlan(xsd, xed)
    assert plan.regular and plan.track_length == 2304 and plan.n_tracks == 18
    p = jp.jp_fwd_tof_sino_planned(plan, imgd, g.origin, g.voxsize, tof)
    sel = np.arange(0, n, 5)
    hxs, hxe = xs.numpy()[:, sel], xe.numpy()[:, sel]
    sel = torch.from_numpy(sel).to(cuda_device)
    assert_fwd(p[sel], oracle.fwd_tof_sino(hxs, hxe, ph, g.origin, g.voxsize, *args))
    pu = jp.jp_fwd_tof_sino(xsd, xed, imgd, g.origin, g.voxsize, tof)
    assert float((p - pu).abs().max()) <= 2e-5 * float(pu.abs().max())
    # T1 on the planned result: bins sum to erf(3/sqrt2) x non-TOF
    pn = jp.jp_fwd(xsd, xed, imgd, g.origin, g.voxsize)
    assert torch.allclose(p.sum(1), 0.99730020393674 * pn, rtol=2e-5, atol=1e-3)
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=12, device=cuda_device)
    ys = torch.zeros_like(y)
    ys[sel] = y[sel]
    b = jp.jp_back_tof_sino_planned(plan, ys, g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(hxs, hxe, ys[sel].cpu().numpy(), g.n, g.origin, g.voxsize, *args))
    bd = jp.jp_back_tof_sino_planned(plan, y, g.n, g.origin, g.voxsize, tof)
    assert adj_gap(p, y, imgd, bd) <= ADJ_GAP
    bu = jp.jp_back_tof_sino(xsd, xed, y, g.n, g.origin, g.voxsize, tof)
    assert float((bd - bu).abs().max()) <= 1e-4 * float(bu.abs().max())


def test_planned_sino_osem(cuda_device):
    """jp_sino_sens_tof_planned / jp_sino_osem_tof_planned (fused forward + ratio + back per track slice) against the
    oracle's numpy OSEM (readings S1-S3): 3 subsets of whole tracks, mult and contam, 2 iterations; and a subset
    boundary that cuts a track (unplanned kernels on the expanded list) gives the same image"""
    g = inputs.GEOM_SMALL
    zv = np.linspace(-38.0, 38.0, 10)
    xs, xe, K, T = mini_sinogram(90, zv, zv, seed=31)
    n = K * T
    args = (9.0, 7.0, 3.0, 27)
    tof = jp.make_tof(*args)
    rng = np.random.default_rng(6)
    y = rng.uniform(0, 2, (n, 27)).astype(np.float32)
    mult = rng.uniform(0.2, 1.0, n).astype(np.float32)
    contam = rng.uniform(0.01, 0.1, (n, 27)).astype(np.float32)
    off = [0, 30 * T, 55 * T, n]
    x0 = rng.uniform(0.5, 1.5, g.n).astype(np.float32)
    plan = jp.SinoPlan(dev(xs, cuda_device), dev(xe, cuda_device))
    d = lambda a: dev(a, cuda_device)
    sens = jp.jp_sino_sens_tof_planned(plan, off, d(mult), g.n, g.origin, g.voxsize, tof)
    sens_o = oracle.sino_sens_tof(xs, xe, off, mult, g.n, g.origin, g.voxsize, *args)
    for m in range(3):
        assert_back(sens[m], sens_o[m])
    x = d(x0.copy())
    jp.jp_sino_osem_tof_planned(plan, off, d(y), d(mult), d(contam), sens, x, g.origin, g.voxsize, tof, n_iter=2)
    # the update divides by sens and zeroes x where sens == 0: both sides get the SAME sensitivity images (the CUDA
    # ones, checked against the oracle's just above), so that the zero sets cannot differ by a rounding
    sens_g = sens.cpu().numpy().astype(np.float64)
    ref = oracle.sino_osem_tof(xs, xe, off, y, mult, contam, sens_g, x0, g.origin, g.voxsize, *args, n_iter=2)
    got = x.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all() and np.linalg.norm(ref) > 1.0
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-4
    assert np.abs(got - ref).max() <= 1e-3 * np.abs(ref).max()
    # no factors at all (mult = 1, contam = 0), and a subset boundary inside a track.  Without contamination the ratio
    # y / ybar is only well conditioned for consistent data: y = A (1.3 x0) computed by the (checked) forward projector
    off2 = [0, 40 * T + 11, n]
    y2 = jp.jp_fwd_tof_sino_planned(plan, d(1.3 * x0), g.origin, g.voxsize, tof)
    sens2 = jp.jp_sino_sens_tof_planned(plan, off2, None, g.n, g.origin, g.voxsize, tof,
                                        workspace=torch.empty(4 * n * 27, dtype=torch.uint8, device=cuda_device))
    x2 = d(x0.copy())
    jp.jp_sino_osem_tof_planned(plan, off2, y2, None, None, sens2, x2, g.origin, g.voxsize, tof, n_iter=1)
    sens2_o = oracle.sino_sens_tof(xs, xe, off2, np.ones(n), g.n, g.origin, g.voxsize, *args)
    for m in range(2):
        assert_back(sens2[m], sens2_o[m])
    ref2 = oracle.sino_osem_tof(xs, xe, off2, y2.cpu().numpy(), np.ones(n), np.zeros((n, 27)),
                                sens2.cpu().numpy().astype(np.float64), x0, g.origin, g.voxsize, *args, n_iter=1)
    got2 = x2.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(ref2) > 1.0
    assert np.linalg.norm(got2 - ref2) / np.linalg.norm(ref2) <= 1e-4
    assert np.abs(got2 - ref2).max() <= 1e-3 * np.abs(ref2).max()


# ---- non-TOF projections of a sinogram plan (per-track tiles, no end-point arrays read) --------------------------------
def test_planned_nontof_scanner_views(cuda_device):
    """configs[1] structure: views 0, 64 (exact 45 degree ties) and 100 x 14 radial bins (incl. the degenerate
    r = +-128 and misses) x 2304 ring pairs: planned forward (one CTA per track) against the unplanned forward (tiles
    of 768 LORs: the same arithmetic per LOR up to the rounding of the plane coordinate, which depends on where a
    chunk of planes starts), both against the oracle; planned adjoint against the oracle; accumulate semantics"""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    radial = [-128, -70, -64, -33, -20, -1, 0, 1, 7, 31, 50, 64, 65, 128]
    xs, xe = inputs.sinogram_lors(views=[0, 64, 100], radial=radial)
    n = xs.shape[1]
    xsd, xed, imgd = xs.to(cuda_device), xe.to(cuda_device), dev(ph, cuda_device)
    plan = jp.SinoPlan(xsd, xed)
    assert plan.regular and plan.track_length == 2304 and plan.n_tracks == 3 * len(radial)
    p = jp.jp_fwd_planned(plan, imgd, g.origin, g.voxsize)
    pu = jp.jp_fwd(xsd, xed, imgd, g.origin, g.voxsize)
    assert float((p - pu).abs().max()) <= 2e-6 * float(pu.abs().max())
    assert torch.equal(p == 0, pu == 0)       # LORs that miss the image: exactly zero in both
    ref = oracle.fwd(xs.numpy(), xe.numpy(), ph, g.origin, g.voxsize)
    assert (ref > 0).mean() > 0.3
    assert_fwd(p, ref)
    y = inputs.uniform_values(n, 0.0, 1.0, seed=11)
    b = jp.jp_back_planned(plan, y.to(cuda_device), g.n, g.origin, g.voxsize)
    assert_back(b, oracle.back(xs.numpy(), xe.numpy(), y.numpy(), g.n, g.origin, g.voxsize))
    assert adj_gap(p, y.to(cuda_device), imgd, b) <= ADJ_GAP
    b2 = jp.jp_back_planned(plan, y.to(cuda_device), g.n, g.origin, g.voxsize, img=torch.full_like(b, 5.0))
    assert torch.allclose(b2 - 5.0, b, rtol=1e-4, atol=1e-2)


def test_planned_nontof_tracks_not_a_multiple_of_the_tile(cuda_device):
    """36-ring sub-scanner: tracks of 1296 ring pairs = one tile of 768 + one of 528 per track; and the small
    image with a mini sinogram whose tracks are shorter than a tile and partly steeper than they are long"""
    g, ph = inputs.GEOM_SCANNER, inputs.phantom()
    xs, xe = inputs.sinogram_lors(views=[5, 64, 130], radial=range(-40, 41, 8))
    idx = np.arange(xs.shape[1])
    keep = ((idx // 48) % 48 < 36) & (idx % 48 < 36)
    hxs, hxe = np.ascontiguousarray(xs.numpy()[:, keep]), np.ascontiguousarray(xe.numpy()[:, keep])
    n = hxs.shape[1]
    plan = jp.SinoPlan(dev(hxs, cuda_device), dev(hxe, cuda_device))
    assert plan.regular and plan.track_length == 1296
    p = jp.jp_fwd_planned(plan, dev(ph, cuda_device), g.origin, g.voxsize)
    assert_fwd(p, oracle.fwd(hxs, hxe, ph, g.origin, g.voxsize))
    y = np.random.default_rng(3).uniform(0, 1, n).astype(np.float32)
    b = jp.jp_back_planned(plan, dev(y, cuda_device), g.n, g.origin, g.voxsize)
    assert_back(b, oracle.back(hxs, hxe, y, g.n, g.origin, g.voxsize))
    # small image, T = 400 < 768, steep pattern (some tracks take the per-LOR path), image 32 x 32 x 16
    gs = inputs.GEOM_SMALL
    zv = np.linspace(-60.0, 60.0, 20)
    extra = [(-20.0, 3.0, 25.0, 5.0), (1.0, -30.0, 2.0, 31.0), (-150.0, 0.5, 150.0, -0.5), (-150.0, -150.0, 150.0, 150.0)]
    sxs, sxe, K, T = mini_sinogram(7, zv, zv, seed=13, extra_tracks=extra)
    img = np.random.default_rng(1).uniform(0, 1, gs.n).astype(np.float32)
    plan2 = jp.SinoPlan(dev(sxs, cuda_device), dev(sxe, cuda_device))
    assert plan2.regular and plan2.track_length == 400
    p2 = jp.jp_fwd_planned(plan2, dev(img, cuda_device), gs.origin, gs.voxsize)
    assert_fwd(p2, oracle.fwd(sxs, sxe, img, gs.origin, gs.voxsize))
    y2 = np.random.default_rng(2).uniform(-1, 1, K * T).astype(np.float32)
    b2 = jp.jp_back_planned(plan2, dev(y2, cuda_device), gs.n, gs.origin, gs.voxsize)
    assert_back(b2, oracle.back(sxs, sxe, y2, gs.n, gs.origin, gs.voxsize))


@pytest.mark.parametrize("nzs,nze", [(60, 60), (1, 2500), (53, 47)])
def test_planned_nontof_long_tracks(cuda_device, nzs, nze):
    """tracks longer than one CTA takes (3600 = 2 pieces of 1800; 2500 LORs with ONE axial start point: no grid, 2
    pieces of 1250; 2491 = 53 x 47: 2 ragged pieces that cut the grid rows) on the small image, wide axial range
    (part of every track misses the image, the extra tracks are steep or degenerate)"""
    gs = inputs.GEOM_SMALL
    extra = [(-20.0, 3.0, 25.0, 5.0), (-150.0, 0.5, 150.0, -0.5), (-150.0, -150.0, 150.0, 150.0), (30.0, 40.0, 30.0, 40.0)]
    sxs, sxe, K, T = mini_sinogram(5, np.linspace(-45.0, 45.0, nzs) if nzs > 1 else [3.0], np.linspace(-50.0, 41.0, nze),
                                   seed=nzs, extra_tracks=extra)
    img = np.random.default_rng(1).uniform(0, 1, gs.n).astype(np.float32)
    plan = jp.SinoPlan(dev(sxs, cuda_device), dev(sxe, cuda_device))
    assert plan.regular and plan.track_length == nzs * nze and T > 2304
    p = jp.jp_fwd_planned(plan, dev(img, cuda_device), gs.origin, gs.voxsize)
    ref = oracle.fwd(sxs, sxe, img, gs.origin, gs.voxsize)
    assert (ref > 0).mean() > 0.3
    assert_fwd(p, ref)
    y = np.random.default_rng(2).uniform(-1, 1, K * T).astype(np.float32)
    b = jp.jp_back_planned(plan, dev(y, cuda_device), gs.n, gs.origin, gs.voxsize)
    assert_back(b, oracle.back(sxs, sxe, y, gs.n, gs.origin, gs.voxsize))
    assert adj_gap(p, dev(y, cuda_device), dev(img, cuda_device), b) <= ADJ_GAP


@pytest.mark.parametrize("planned", [False, True])
def test_nontof_adjoint_dynamic_range_and_nonfinite(cuda_device, planned):
    """k_back_tile's fixed-point staging at full configs[1] tile density (every LOR of 6 tracks carries a value):
    y spanning 6 decades with both signs inside every 768-LOR tile stays within the tolerance; a tile whose y holds
    Inf / NaN takes the per-LOR float path: the non-finite voxels are exactly the oracle's, all others stay right"""
    g = inputs.GEOM_SCANNER
    xs, xe = inputs.sinogram_lors(views=[17, 100], radial=[-20, 0, 33])
    n = xs.shape[1]
    xsd, xed = xs.to(cuda_device), xe.to(cuda_device)
    plan = jp.SinoPlan(xsd, xed) if planned else None
    back = (lambda yy: jp.jp_back_planned(plan, yy, g.n, g.origin, g.voxsize)) if planned else \
           (lambda yy: jp.jp_back(xsd, xed, yy, g.n, g.origin, g.voxsize))
    rng = np.random.default_rng(77)
    y = (10.0 ** rng.uniform(-6, 0, n) * rng.choice([-1.0, 1.0], n)).astype(np.float32)
    assert_back(back(dev(y, cuda_device)), oracle.back(xs.numpy(), xe.numpy(), y, g.n, g.origin, g.voxsize))
    y2 = rng.uniform(0, 1, n).astype(np.float32)
    y2[2304 + 1000] = np.inf            # second track, second tile
    y2[4 * 2304 + 5] = np.nan           # fifth track, first tile
    got = back(dev(y2, cuda_device)).cpu().numpy()
    ref = oracle.back(xs.numpy(), xe.numpy(), y2, g.n, g.origin, g.voxsize)
    bad, gbad = ~np.isfinite(ref), ~np.isfinite(got)
    assert bad.any() and not bad.all()
    # the poisoned voxels are the oracle's, up to the zero-weight neighbours of crossing points that float32 and float64
    # put on different sides of a voxel centre (Inf x 0 = NaN reaches a neighbour only where the weight is exactly 0)
    assert np.logical_xor(gbad, bad).sum() <= 0.01 * bad.sum()
    ok = ~bad & ~gbad
    assert np.abs(got[ok] - ref[ok]).max() <= 1e-4 * np.abs(ref[ok]).max()
