"""Parity of the CUDA path (through the C ABI, via the thin binding) against the float64 oracle,
element by element, on the same seeded inputs.  Tolerances are BASELINE.json north_star's:

  forward      rel-L2 <= 1e-5  and  max abs <= 1e-4 * max|oracle|
  back         per-voxel max abs <= 1e-4 * max|oracle|   (atomic summation order)
  adjointness  GPU relative gap <= 1e-4
  principal axis / counts: bit-exact
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs

pytestmark = pytest.mark.gpu

FWD_REL_L2 = 1e-5
MAX_ABS = 1e-4
ADJ_GAP = 1e-4


def assert_fwd(gpu: torch.Tensor, ref: np.ndarray):
    g = gpu.detach().cpu().numpy().astype(np.float64).reshape(ref.shape)
    assert np.isfinite(g).all()
    den = np.linalg.norm(ref)
    rel = np.linalg.norm(g - ref) / den if den > 0 else np.linalg.norm(g)
    mx = np.abs(g - ref).max() if ref.size else 0.0
    scale = np.abs(ref).max() if ref.size else 1.0
    assert rel <= FWD_REL_L2, f"forward rel-L2 {rel:.3e}"
    assert mx <= MAX_ABS * scale, f"forward max abs {mx:.3e} vs {MAX_ABS * scale:.3e}"
    return rel, mx / scale


def assert_back(gpu: torch.Tensor, ref: np.ndarray):
    g = gpu.detach().cpu().numpy().astype(np.float64)
    assert np.isfinite(g).all()
    mx = np.abs(g - ref).max()
    scale = np.abs(ref).max()
    assert mx <= MAX_ABS * scale, f"back max abs {mx:.3e} vs {MAX_ABS * scale:.3e}"
    return mx / scale


def adj_gap(Ax, y, x, Aty):
    a = float((Ax.double() * y.double()).sum())
    b = float((x.double() * Aty.double()).sum())
    return abs(a - b) / abs(a)


def dev(a, device):
    return torch.as_tensor(a).to(device).contiguous()


# ---- config 0: the full small case ---------------------------------------------------------------------
def test_config0_nontof(cuda_device):
    c = inputs.config0()
    g = c["geom"]
    xs, xe = dev(c["xstart"], cuda_device), dev(c["xend"], cuda_device)
    img, y = dev(c["img"], cuda_device), dev(c["y"], cuda_device)
    # principal axis: bit exact
    ax = jp.jp_classify(xs, xe).cpu().numpy()
    assert np.array_equal(ax, oracle.classify(c["xstart"], c["xend"], g.n, g.origin, g.voxsize))
    p = jp.jp_fwd(xs, xe, img, g.origin, g.voxsize)
    assert p.shape == (50_000,)
    assert_fwd(p, oracle.fwd(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize))
    b = jp.jp_back(xs, xe, y, g.n, g.origin, g.voxsize)
    assert_back(b, oracle.back(c["xstart"], c["xend"], c["y"], g.n, g.origin, g.voxsize))
    assert adj_gap(p, y, img, b) <= ADJ_GAP
    # ACCUMULATE semantics
    b2 = jp.jp_back(xs, xe, y, g.n, g.origin, g.voxsize, img=torch.full_like(b, 3.0))
    assert torch.allclose(b2 - 3.0, b, rtol=1e-4, atol=1e-3)


def test_config0_tof(cuda_device):
    """config-0 LORs with a TOF model scaled to the 128 mm image (all three principal axes occur)"""
    c = inputs.config0(n_lors=20_000)
    g = c["geom"]
    rng = np.random.default_rng(5)
    tofp = inputs.TofParams(tofbin_width=9.0, sigma_tof=7.0, n_sigmas=3.0, n_tofbins=27)
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    xs, xe = dev(c["xstart"], cuda_device), dev(c["xend"], cuda_device)
    img = dev(c["img"], cuda_device)
    # sinogram
    p = jp.jp_fwd_tof_sino(xs, xe, img, g.origin, g.voxsize, tof)
    assert_fwd(p, oracle.fwd_tof_sino(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize, *args))
    y = rng.uniform(0, 1, (20_000, 27)).astype(np.float32)
    b = jp.jp_back_tof_sino(xs, xe, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(c["xstart"], c["xend"], y, g.n, g.origin, g.voxsize, *args))
    assert adj_gap(p, dev(y, cuda_device), img, b) <= ADJ_GAP
    # listmode
    it = rng.integers(-13, 14, 20_000).astype(np.int16)
    pl = jp.jp_fwd_tof_lm(xs, xe, dev(it, cuda_device), img, g.origin, g.voxsize, tof)
    assert_fwd(pl, oracle.fwd_tof_lm(c["xstart"], c["xend"], it, c["img"], g.origin, g.voxsize, *args[:3]))
    yl = rng.uniform(0.5, 2, 20_000).astype(np.float32)
    bl = jp.jp_back_tof_lm(xs, xe, dev(it, cuda_device), dev(yl, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(bl, oracle.back_tof_lm(c["xstart"], c["xend"], it, yl, g.n, g.origin, g.voxsize, *args[:3]))
    assert adj_gap(pl, dev(yl, cuda_device), img, bl) <= ADJ_GAP


@pytest.mark.parametrize("width,nbins,coff", [(20.0, 13, 0.0), (9.0, 27, 2.5), (6.0, 41, 0.0), (4.0, 61, -1.0),
                                              (2.5, 63, 0.0)])
def test_tof_sino_window_sizes(cuda_device, width, nbins, coff):
    """TOF sinogram kernels for every compiled register-window size (4, 6, 8, 12 bins) and the generic fallback
    (window of 18 bins), with a centre offset, all three principal axes and a ragged tail"""
    c = inputs.config0(n_lors=6_007)
    g = c["geom"]
    sigma, nsig = 7.0, 3.0
    tof = jp.make_tof(width, sigma, nsig, nbins, coff)
    xs, xe = dev(c["xstart"], cuda_device), dev(c["xend"], cuda_device)
    img = dev(c["img"], cuda_device)
    p = jp.jp_fwd_tof_sino(xs, xe, img, g.origin, g.voxsize, tof)
    ref = oracle.fwd_tof_sino(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize, width, sigma, nsig, nbins,
                              center_offset=coff)
    assert_fwd(p, ref)
    y = np.random.default_rng(int(width * 10)).uniform(-0.5, 1, (6_007, nbins)).astype(np.float32)
    b = jp.jp_back_tof_sino(xs, xe, dev(y, cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(c["xstart"], c["xend"], y, g.n, g.origin, g.voxsize, width, sigma, nsig, nbins,
                                        center_offset=coff))
    assert adj_gap(p, dev(y, cuda_device), img, b) <= ADJ_GAP


# ---- slices of configs 1-3 on the scanner geometry (several tiles + ragged tail) ----------------------
@pytest.fixture(scope="module")
def scanner():
    g = inputs.GEOM_SCANNER
    return g, inputs.phantom()


def _sino_slice(views, radial):
    xs, xe = inputs.sinogram_lors(views=views, radial=radial)
    return xs, xe


def test_config1_slice_nontof(cuda_device, scanner):
    """views 0, 64 (exact 45 degree ties) and 100, radial offsets incl. the degenerate r=+-128 and a miss"""
    g, ph = scanner
    radial = [-128, -70, -64, -33, -20, -1, 0, 1, 7, 31, 50, 64, 65, 128]
    xs, xe = _sino_slice([0, 64, 100], radial)
    n = xs.shape[1]
    assert n == 3 * len(radial) * 2304
    # ragged tail: drop a few LORs so n is not a multiple of the block size
    xs, xe = xs[:, : n - 37].contiguous(), xe[:, : n - 37].contiguous()
    n -= 37
    xsd, xed, imgd = xs.to(cuda_device), xe.to(cuda_device), dev(ph, cuda_device)
    ax = jp.jp_classify(xsd, xed).cpu().numpy()
    ax_ref = oracle.classify(xs.numpy(), xe.numpy(), g.n, g.origin, g.voxsize)
    assert np.array_equal(ax, ax_ref)
    p = jp.jp_fwd(xsd, xed, imgd, g.origin, g.voxsize)
    ref = oracle.fwd(xs.numpy(), xe.numpy(), ph, g.origin, g.voxsize)
    assert (ref > 0).mean() > 0.3
    assert_fwd(p, ref)
    y = inputs.uniform_values(n, 0.0, 1.0, seed=11)
    b = jp.jp_back(xsd, xed, y.to(cuda_device), g.n, g.origin, g.voxsize)
    assert_back(b, oracle.back(xs.numpy(), xe.numpy(), y.numpy(), g.n, g.origin, g.voxsize))
    assert adj_gap(p, y.to(cuda_device), imgd, b) <= ADJ_GAP


def test_tracks_not_a_multiple_of_the_tile(cuda_device, scanner):
    """36-ring sub-scanner: tracks of 36 x 36 = 1296 ring pairs, not a multiple of the 768-LOR tile -> the kernels
    deal tiles per track (768 + 528); a second list whose track lengths vary (tile_is_track must fall back)"""
    g, ph = scanner
    xs, xe = inputs.sinogram_lors(views=[5, 64, 130], radial=range(-40, 41, 4))
    idx = np.arange(xs.shape[1])
    keep = ((idx // 48) % 48 < 36) & (idx % 48 < 36)
    for variant in (0, 1):
        k = keep.copy()
        if variant == 1:
            k[1296 * 3 + 100:1296 * 3 + 150] = False        # one track is 50 LORs shorter: the assumed grid slips
        hxs, hxe = np.ascontiguousarray(xs.numpy()[:, k]), np.ascontiguousarray(xe.numpy()[:, k])
        n = hxs.shape[1]
        assert n > 8 * 768
        dxs, dxe = dev(hxs, cuda_device), dev(hxe, cuda_device)
        p = jp.jp_fwd(dxs, dxe, dev(ph, cuda_device), g.origin, g.voxsize)
        assert_fwd(p, oracle.fwd(hxs, hxe, ph, g.origin, g.voxsize))
        y = np.random.default_rng(variant).uniform(0, 1, n).astype(np.float32)
        b = jp.jp_back(dxs, dxe, dev(y, cuda_device), g.n, g.origin, g.voxsize)
        assert_back(b, oracle.back(hxs, hxe, y, g.n, g.origin, g.voxsize))
        assert adj_gap(p, dev(y, cuda_device), dev(ph, cuda_device), b) <= ADJ_GAP


def test_config2_slice_tof_sino(cuda_device, scanner):
    g, ph = scanner
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    xs, xe = _sino_slice([64, 240], [-40, -3, 0, 25, 64])
    # every 7th ring pair keeps the oracle fast while spanning many blocks
    xs, xe = xs[:, ::7].contiguous(), xe[:, ::7].contiguous()
    n = xs.shape[1]
    xsd, xed, imgd = xs.to(cuda_device), xe.to(cuda_device), dev(ph, cuda_device)
    p = jp.jp_fwd_tof_sino(xsd, xed, imgd, g.origin, g.voxsize, tof)
    ref = oracle.fwd_tof_sino(xs.numpy(), xe.numpy(), ph, g.origin, g.voxsize, *args)
    assert_fwd(p, ref)
    # T1 on the GPU result: bins sum to erf(3/sqrt2) x non-TOF
    pn = jp.jp_fwd(xsd, xed, imgd, g.origin, g.voxsize)
    assert torch.allclose(p.sum(1), 0.99730020393674 * pn, rtol=2e-5, atol=1e-3)
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=12)
    b = jp.jp_back_tof_sino(xsd, xed, y.to(cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(xs.numpy(), xe.numpy(), y.numpy(), g.n, g.origin, g.voxsize, *args))
    assert adj_gap(p, y.to(cuda_device), imgd, b) <= ADJ_GAP


@pytest.fixture(scope="module")
def events(scanner):
    g, ph = scanner
    xs, xe, tb = inputs.listmode_events(300_011, seed=inputs.BASE_SEED + 3, img=ph, chunk=1_000_000)
    return xs, xe, tb


def test_config3_slice_tof_lm(cuda_device, scanner, events):
    g, ph = scanner
    xs, xe, tb = events
    n = xs.shape[1]
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    xsd, xed, tbd, imgd = xs.to(cuda_device), xe.to(cuda_device), tb.to(cuda_device), dev(ph, cuda_device)
    p = jp.jp_fwd_tof_lm(xsd, xed, tbd, imgd, g.origin, g.voxsize, tof)
    ref = oracle.fwd_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), ph, g.origin, g.voxsize, *args)
    assert (ref > 0).mean() > 0.95
    assert_fwd(p, ref)
    y = inputs.uniform_values(n, 0.5, 2.0, seed=13)
    b = jp.jp_back_tof_lm(xsd, xed, tbd, y.to(cuda_device), g.n, g.origin, g.voxsize, tof)
    assert_back(b, oracle.back_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), y.numpy(), g.n, g.origin, g.voxsize, *args))
    assert adj_gap(p, y.to(cuda_device), imgd, b) <= ADJ_GAP
    # T3 on the GPU: listmode == sinogram column
    sub = slice(0, 5000)
    ps = jp.jp_fwd_tof_sino(xsd[:, sub].contiguous(), xed[:, sub].contiguous(), imgd, g.origin, g.voxsize, tof)
    col = ps[torch.arange(5000, device=cuda_device), (tbd[sub].long() + 14)]
    assert torch.allclose(col, p[sub], rtol=2e-5, atol=1e-4)


def test_config4_small_osem(cuda_device, scanner, events):
    """listmode OSEM on a reduced problem: 300k events, 5 subsets, 2 iterations, vs the float64 oracle"""
    g, ph = scanner
    xs, xe, tb = events
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    # sensitivity: non-TOF back projection of ones over a coarse set of sinogram LORs
    sx, se = inputs.sinogram_lors(views=range(0, 256, 8), radial=range(-64, 65, 4))
    sx, se = sx[:, ::5].contiguous(), se[:, ::5].contiguous()
    sens64 = oracle.back(sx.numpy(), se.numpy(), np.ones(sx.shape[1]), g.n, g.origin, g.voxsize)
    sens32 = sens64.astype(np.float32)
    x0 = np.ones(g.n, dtype=np.float32)
    ref = oracle.lm_osem(xs.numpy(), xe.numpy(), tb.numpy(), sens32.astype(np.float64), x0, g.origin, g.voxsize,
                         *args, n_subsets=5, n_iter=2)
    img = dev(x0, cuda_device).clone()
    jp.jp_lm_osem(xs.to(cuda_device), xe.to(cuda_device), tb.to(cuda_device), dev(sens32, cuda_device), img,
                  g.origin, g.voxsize, tof, n_subsets=5, n_iter=2)
    got = img.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    assert rel <= 1e-4, f"OSEM rel-L2 {rel:.3e}"
    assert mx <= 1e-3, f"OSEM max abs / max {mx:.3e}"


def test_config3_plan_sorted_events(cuda_device, scanner, events):
    """the listmode plan (sorted events) computes what the unplanned calls compute, in caller order"""
    g, ph = scanner
    xs, xe, tb = events
    n = xs.shape[1]
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    xsd, xed, tbd, imgd = xs.to(cuda_device), xe.to(cuda_device), tb.to(cuda_device), dev(ph, cuda_device)
    plan = jp.LmPlan(xsd, xed, tbd, g.n, g.origin, g.voxsize, tof, n_subsets=7)
    # counts: bit exact
    counts = [plan.subset_count(m) for m in range(7)]
    assert counts == [len(range(m, n, 7)) for m in range(7)] and plan.subset_count(-1) == n
    p_ref = jp.jp_fwd_tof_lm(xsd, xed, tbd, imgd, g.origin, g.voxsize, tof)
    mask = torch.zeros(n, dtype=torch.bool, device=cuda_device)
    mask[3::7] = True
    # the plan's own choice for this list (sparsely populated lines: image bricks, another TOF table and summation
    # order than the per-event kernels): equal within float32 rounding
    p_all = jp.jp_fwd_tof_lm_planned(plan, imgd)
    assert float((p_all - p_ref).abs().max()) <= 1e-5 * float(p_ref.max())
    p_sub = jp.jp_fwd_tof_lm_planned(plan, imgd, subset=3, out=torch.full((n,), -1.0, device=cuda_device))
    assert float((p_sub[mask] - p_ref[mask]).abs().max()) <= 1e-5 * float(p_ref.max()) and bool((p_sub[~mask] == -1.0).all())
    # quad image: same arithmetic per event as the unplanned kernels, only the order differs -> bit for bit
    plan.set_path(2)
    assert torch.equal(jp.jp_fwd_tof_lm_planned(plan, imgd), p_ref)
    p_sub = jp.jp_fwd_tof_lm_planned(plan, imgd, subset=3, out=torch.full((n,), -1.0, device=cuda_device))
    assert torch.equal(p_sub[mask], p_ref[mask]) and bool((p_sub[~mask] == -1.0).all())
    plan.set_path(0)
    # adjoint: subsets add up to the whole, and the whole matches the oracle
    y = inputs.uniform_values(n, 0.5, 2.0, seed=13).to(cuda_device)
    b_all = jp.jp_back_tof_lm_planned(plan, y)
    b_sum = torch.zeros_like(b_all)
    for m in range(7):
        jp.jp_back_tof_lm_planned(plan, y, subset=m, img=b_sum)
    ref = oracle.back_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), y.cpu().numpy(), g.n, g.origin, g.voxsize, *args)
    assert_back(b_all, ref)
    assert_back(b_sum, ref)
    assert adj_gap(p_all, y, imgd, b_all) <= ADJ_GAP
    plan.destroy()


def _line_events(seed=21):
    """events that share few transaxial lines (long runs for the line tiles): all 2304 ring pairs of 22 sinogram
    bins, a third of them given as (e, s) instead of (s, e), random TOF bins, shuffled"""
    xs, xe = inputs.sinogram_lors(views=[3, 64, 100, 192, 200], radial=[-30, -5, 0, 17])
    xs2, xe2 = inputs.sinogram_lors(views=[77], radial=[-64, 31])     # grazing / partly outside
    xs, xe = torch.cat([xs, xs2], 1), torch.cat([xe, xe2], 1)
    n = xs.shape[1]
    rng = np.random.default_rng(seed)
    keep = rng.permutation(n)[: n - 101]                                # ragged
    xs, xe = xs[:, keep].numpy().copy(), xe[:, keep].numpy().copy()
    n = xs.shape[1]
    swap = rng.random(n) < 0.33
    xs[:, swap], xe[:, swap] = xe[:, swap].copy(), xs[:, swap].copy()
    tb = rng.integers(-12, 13, n).astype(np.int16)
    return xs, xe, tb


@pytest.mark.parametrize("n_subsets", [1, 3])
def test_lm_line_tiles(cuda_device, scanner, n_subsets):
    """planned TOF listmode projectors on line tiles (runs of events sharing a transaxial line) vs the oracle; then a
    y with Inf / NaN: the runs that hold them take the per-LOR float path, nothing finite is lost"""
    g, ph = scanner
    xs, xe, tb = _line_events()
    n = xs.shape[1]
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins, 1.5)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    xsd, xed, tbd, imgd = dev(xs, cuda_device), dev(xe, cuda_device), dev(tb, cuda_device), dev(ph, cuda_device)
    plan = jp.LmPlan(xsd, xed, tbd, g.n, g.origin, g.voxsize, tof, n_subsets=n_subsets).set_path(1)
    p = jp.jp_fwd_tof_lm_planned(plan, imgd)
    ref = oracle.fwd_tof_lm(xs, xe, tb, ph, g.origin, g.voxsize, *args, center_offset=1.5)
    assert (ref > 0).mean() > 0.5
    assert_fwd(p, ref)
    y = inputs.uniform_values(n, 0.5, 2.0, seed=14).to(cuda_device)
    b = jp.jp_back_tof_lm_planned(plan, y)
    assert_back(b, oracle.back_tof_lm(xs, xe, tb, y.cpu().numpy(), g.n, g.origin, g.voxsize, *args, center_offset=1.5))
    assert adj_gap(p, y, imgd, b) <= ADJ_GAP
    # non-finite values on events that cross the image (chosen among the large forward values)
    hit = np.argsort(ref)[-2000:]
    y2 = y.cpu().numpy().copy()
    y2[hit[0]], y2[hit[1000]] = np.inf, np.nan
    got = jp.jp_back_tof_lm_planned(plan, dev(y2, cuda_device)).cpu().numpy()
    y0 = y2.copy()
    y0[~np.isfinite(y0)] = 0.0
    ref0 = oracle.back_tof_lm(xs, xe, tb, y0, g.n, g.origin, g.voxsize, *args, center_offset=1.5)
    refb = ~np.isfinite(oracle.back_tof_lm(xs, xe, tb, y2, g.n, g.origin, g.voxsize, *args, center_offset=1.5))
    bad = ~np.isfinite(got)
    assert bad.any() and not bad.all() and not (bad & ~refb).sum() > 0.01 * refb.sum()
    assert np.abs(got[~bad] - ref0[~bad]).max() <= 1e-4 * np.abs(ref0).max()
    plan.destroy()


@pytest.mark.parametrize("path", [0, 2, 3])
def test_config4_small_osem_planned(cuda_device, scanner, events, path):
    """listmode OSEM on a plan: 0 = the plan's own choice, 2 = quad image, 3 = image bricks (jp_brick.cu)"""
    g, ph = scanner
    xs, xe, tb = events
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    sx, se = inputs.sinogram_lors(views=range(0, 256, 8), radial=range(-64, 65, 4))
    sx, se = sx[:, ::5].contiguous(), se[:, ::5].contiguous()
    sens32 = oracle.back(sx.numpy(), se.numpy(), np.ones(sx.shape[1]), g.n, g.origin, g.voxsize).astype(np.float32)
    x0 = np.ones(g.n, dtype=np.float32)
    ref = oracle.lm_osem(xs.numpy(), xe.numpy(), tb.numpy(), sens32.astype(np.float64), x0, g.origin, g.voxsize,
                         *args, n_subsets=5, n_iter=2)
    plan = jp.LmPlan(xs.to(cuda_device), xe.to(cuda_device), tb.to(cuda_device), g.n, g.origin, g.voxsize, tof,
                     n_subsets=5).set_path(path)
    img = dev(x0, cuda_device).clone()
    jp.jp_lm_osem_planned(plan, dev(sens32, cuda_device), img, n_iter=2)
    got = img.cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    assert rel <= 1e-4, f"OSEM rel-L2 {rel:.3e}"
    assert mx <= 1e-3, f"OSEM max abs / max {mx:.3e}"
    plan.destroy()


def test_osem_over_event_shards(cuda_device, scanner, events):
    """the multi-GPU OSEM driver (multi_gpu.lm_osem_sharded) on ONE GPU: the event list is cut into
    the shards two and three ranks would hold (multi_gpu.shard_events), each shard gets its own plan, the per-shard
    images b are summed where the all-reduce would sum them (sequentially, nothing waits on anything), and the
    result must be the oracle's OSEM over the whole list.  world_size-2 gloo runs of the same driver: tests/
    test_sharding_gloo.py."""
    from paper_2212_12519_b200 import multi_gpu
    g, ph = scanner
    xs, xe, tb = events
    n = xs.shape[1]
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    ns = 5
    sx, se = inputs.sinogram_lors(views=range(0, 256, 8), radial=range(-64, 65, 4))
    sx, se = sx[:, ::5].contiguous(), se[:, ::5].contiguous()
    sens32 = oracle.back(sx.numpy(), se.numpy(), np.ones(sx.shape[1]), g.n, g.origin, g.voxsize).astype(np.float32)
    x0 = np.ones(g.n, dtype=np.float32)
    ref = oracle.lm_osem(xs.numpy(), xe.numpy(), tb.numpy(), sens32.astype(np.float64), x0, g.origin, g.voxsize,
                         *args, n_subsets=ns, n_iter=2)
    sens = dev(sens32, cuda_device)
    for world in (1, 2, 3):
        plans = []
        for r in range(world):
            lo, hi = multi_gpu.shard_events(n, r, world, ns)
            plans.append(jp.LmPlan(xs[:, lo:hi].contiguous().to(cuda_device), xe[:, lo:hi].contiguous().to(cuda_device),
                                   tb[lo:hi].contiguous().to(cuda_device), g.n, g.origin, g.voxsize, tof, n_subsets=ns))
        shard_ops = [multi_gpu.CudaOps(jp, plan=pl) for pl in plans]

        class AllRanks:      # what the ranks + the all-reduce compute together, one rank after the other
            def backratio(self, m, x, b):
                b.zero_()
                part = torch.empty_like(b)
                for o in shard_ops:
                    o.backratio(m, x, part)
                    b += part            # the all-reduce(sum) of the driver, stood in for on one device

            def update(self, x, b, sens_, scale):
                shard_ops[0].update(x, b, sens_, scale)

        x = dev(x0, cuda_device).clone()
        multi_gpu.lm_osem_sharded(AllRanks(), sens, x, ns, 2)
        got = x.cpu().numpy().astype(np.float64)
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mx = np.abs(got - ref).max() / np.abs(ref).max()
        assert rel <= 1e-4 and mx <= 1e-3, (world, rel, mx)
        for pl in plans:
            pl.destroy()


@pytest.mark.parametrize("tile", ["1", "0"])
def test_nontof_listmode_planned(cuda_device, scanner, events, tile):
    """non-TOF projections of listmode events: unsorted through jp_fwd /
    jp_back, and through the plan (line tiles forced on / off) -- all against the oracle, in caller order"""
    g, ph = scanner
    if tile == "1":
        xs, xe, tb = _line_events(seed=22)
    else:
        xs, xe, tb = (t.numpy() for t in events)
        xs, xe, tb = xs[:, :100_003], xe[:, :100_003], tb[:100_003]
    n = xs.shape[1]
    tof = jp.make_tof(17.0, 13.6, 3.0, 29)
    xsd, xed, imgd = dev(xs, cuda_device), dev(xe, cuda_device), dev(ph, cuda_device)
    ref = oracle.fwd(xs, xe, ph, g.origin, g.voxsize)
    assert_fwd(jp.jp_fwd(xsd, xed, imgd, g.origin, g.voxsize), ref)
    plan = jp.LmPlan(xsd, xed, dev(tb, cuda_device), g.n, g.origin, g.voxsize, tof, n_subsets=2)
    plan.set_path(1 if tile == "1" else 2)
    p = jp.jp_fwd_lm_planned(plan, imgd)
    assert_fwd(p, ref)
    y = inputs.uniform_values(n, 0.5, 2.0, seed=15).to(cuda_device)
    bref = oracle.back(xs, xe, y.cpu().numpy(), g.n, g.origin, g.voxsize)
    b = jp.jp_back_lm_planned(plan, y)
    assert_back(b, bref)
    b2 = jp.jp_back_lm_planned(plan, y, subset=0)
    jp.jp_back_lm_planned(plan, y, subset=1, img=b2)
    assert_back(b2, bref)
    assert adj_gap(p, y, imgd, b) <= ADJ_GAP
    plan.destroy()


def test_resolution_model(cuda_device, scanner, events):
    """image-based resolution model: jp_gauss3d vs the oracle's plain 3-D sum, and OSEM with it"""
    g, ph = scanner
    sig = oracle.fwhm_to_sigma(4.5)
    # anisotropic voxels, odd sizes (several blocks + ragged tail), in-place call
    rng = np.random.default_rng(8)
    x = rng.random((37, 21, 45)).astype(np.float32)
    vox = (2.0, 1.5, 2.78)
    ref = oracle.gauss3d(x, vox, sig)
    got = jp.jp_gauss3d(dev(x, cuda_device), vox, sig)
    assert np.abs(got.cpu().numpy() - ref).max() <= 2e-6 * np.abs(ref).max()
    xi = dev(x, cuda_device).clone()
    jp.jp_gauss3d(xi, vox, sig, out=xi)
    assert torch.equal(xi, got)
    # fused two-kernel path (n2 a multiple of 4): several row tiles with a ragged last one, also in place
    x4 = rng.random((19, 70, 44)).astype(np.float32)
    ref4 = oracle.gauss3d(x4, vox, sig)
    got4 = jp.jp_gauss3d(dev(x4, cuda_device), vox, sig)
    assert np.abs(got4.cpu().numpy() - ref4).max() <= 2e-6 * np.abs(ref4).max()
    x4i = dev(x4, cuda_device).clone()
    jp.jp_gauss3d(x4i, vox, sig, out=x4i)
    assert torch.equal(x4i, got4)
    # OSEM with the model: 5 subsets x 1 iteration on the scanner geometry
    xs, xe, tb = events
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    args = (tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas)
    sx, se = inputs.sinogram_lors(views=range(0, 256, 8), radial=range(-64, 65, 4))
    sx, se = sx[:, ::5].contiguous(), se[:, ::5].contiguous()
    sens = oracle.gauss3d(oracle.back(sx.numpy(), se.numpy(), np.ones(sx.shape[1]), g.n, g.origin, g.voxsize),
                          g.voxsize, sig).astype(np.float32)
    x0 = np.ones(g.n, dtype=np.float32)
    ref = oracle.lm_osem_res(xs.numpy(), xe.numpy(), tb.numpy(), sens.astype(np.float64), x0, g.origin, g.voxsize,
                             *args, n_subsets=5, n_iter=1, res_sigma_mm=sig)
    plan = jp.LmPlan(xs.to(cuda_device), xe.to(cuda_device), tb.to(cuda_device), g.n, g.origin, g.voxsize, tof,
                     n_subsets=5)
    img = dev(x0, cuda_device).clone()
    jp.jp_lm_osem_planned_res(plan, dev(sens, cuda_device), img, n_iter=1, res_sigma_mm=sig)
    gotx = img.cpu().numpy().astype(np.float64)
    assert np.isfinite(gotx).all()
    assert np.linalg.norm(gotx - ref) / np.linalg.norm(ref) <= 1e-4
    assert np.abs(gotx - ref).max() <= 1e-3 * np.abs(ref).max()
    plan.destroy()


# ---- edge cases ----------------------------------------------------------------------------------------
def test_edge_cases(cuda_device):
    g = inputs.GEOM_SMALL
    img = torch.rand(g.n, device=cuda_device)
    empty = torch.zeros((3, 0), device=cuda_device)
    assert jp.jp_fwd(empty, empty, img, g.origin, g.voxsize).numel() == 0
    b = jp.jp_back(empty, empty, torch.zeros(0, device=cuda_device), g.n, g.origin, g.voxsize)
    assert float(b.abs().max()) == 0.0
    # zero-length LOR, LOR missing the image, LOR ending inside the image
    xs = torch.tensor([[1.0, 500.0, 3.0], [1.0, 500.0, 2.0], [1.0, 500.0, 1.0]], device=cuda_device)
    xe = torch.tensor([[1.0, 600.0, 90.0], [1.0, 510.0, 5.0], [1.0, 505.0, 2.0]], device=cuda_device)
    p = jp.jp_fwd(xs, xe, img, g.origin, g.voxsize)
    ref = oracle.fwd(xs.cpu().numpy(), xe.cpu().numpy(), img.cpu().numpy(), g.origin, g.voxsize)
    assert p[0] == 0 and p[1] == 0 and torch.isfinite(p).all()
    assert abs(float(p[2]) - ref[2]) <= 1e-5 * abs(ref[2])
    # error codes: bad sizes raise
    with pytest.raises(jp.JosephError):
        jp.jp_fwd(xs, xe, img, g.origin, (0.0, 1.0, 1.0))
    with pytest.raises(jp.JosephError):
        jp.jp_fwd_tof_sino(xs, xe, img, g.origin, g.voxsize, jp.make_tof(17.0, -1.0, 3.0, 29))
    with pytest.raises(jp.JosephError):
        jp.jp_fwd(xs.cpu(), xe.cpu(), img, g.origin, g.voxsize)   # no CPU fallback


def test_forward_projections_are_deterministic(cuda_device, scanner, events, monkeypatch):
    """no atomics on the forward side: every forward kernel (track tiles, per-track tiles, TOF sinogram window,
    listmode line tiles and quad gathers) must give bit-identical results from run to run -- a cheap detector of
    shared-memory races between the phases of a tile (compute-sanitizer is not available on the test pool)"""
    g, ph = scanner
    img = dev(ph, cuda_device)
    tofp = inputs.TofParams()
    tof = jp.make_tof(tofp.tofbin_width, tofp.sigma_tof, tofp.n_sigmas, tofp.n_tofbins)
    xs, xe = inputs.sinogram_lors(views=[5, 64, 130], radial=range(-40, 41, 8))
    idx = np.arange(xs.shape[1])
    keep = torch.from_numpy(((idx // 48) % 48 < 36) & (idx % 48 < 36))
    lists = [(xs.to(cuda_device), xe.to(cuda_device)), (xs[:, keep].contiguous().to(cuda_device), xe[:, keep].contiguous().to(cuda_device))]
    for a, b in lists:
        ref = jp.jp_fwd(a, b, img, g.origin, g.voxsize).clone()
        for _ in range(3):
            assert torch.equal(jp.jp_fwd(a, b, img, g.origin, g.voxsize), ref)
    a, b = lists[0][0][:, :20_000].contiguous(), lists[0][1][:, :20_000].contiguous()
    ref = jp.jp_fwd_tof_sino(a, b, img, g.origin, g.voxsize, tof).clone()
    for _ in range(3):
        assert torch.equal(jp.jp_fwd_tof_sino(a, b, img, g.origin, g.voxsize, tof), ref)
    ex, ee, tb = (t.to(cuda_device) for t in events)
    for path in (1, 2):
        plan = jp.LmPlan(ex, ee, tb, g.n, g.origin, g.voxsize, tof, n_subsets=1).set_path(path)
        ref = jp.jp_fwd_tof_lm_planned(plan, img).clone()
        refn = jp.jp_fwd_lm_planned(plan, img).clone()
        for _ in range(3):
            assert torch.equal(jp.jp_fwd_tof_lm_planned(plan, img), ref)
            assert torch.equal(jp.jp_fwd_lm_planned(plan, img), refn)
        plan.destroy()
    # image bricks (path 3): an event's pieces are summed with float atomics, so repeats agree up to the order of a
    # handful of additions (a race in the TMA-loaded brick would show as a difference orders of magnitude larger)
    plan = jp.LmPlan(ex, ee, tb, g.n, g.origin, g.voxsize, tof, n_subsets=3).set_path(3)
    ref = jp.jp_fwd_tof_lm_planned(plan, img).clone()
    for _ in range(3):
        assert float((jp.jp_fwd_tof_lm_planned(plan, img) - ref).abs().max()) <= 1e-6 * float(ref.max())
    plan.destroy()


@pytest.mark.parametrize("case", ["wide_image", "wide_tof_kernel"])
def test_planned_listmode_when_the_line_tiles_cannot_hold_the_problem(cuda_device, case):
    """an image longer than the line tiles' widest shared row (n2 > 256), and a TOF kernel whose weight table does not
    fit in shared memory: the planned TOF and non-TOF calls must take the quad / per-event path even when line tiles
    are asked for (they used to fail with 'operation not supported'), and agree with the oracle"""
    c = inputs.config0(n_lors=4_000)
    if case == "wide_image":
        g = inputs.Geometry((24, 24, 270), (4.0, 4.0, 1.0))
        width, sigma = 9.0, 7.0
    else:
        g = c["geom"]
        width, sigma = 1.0, 40.0
    rng = np.random.default_rng(3)
    img = rng.uniform(0, 1, g.n).astype(np.float32)
    tb = rng.integers(-4, 5, 4_000).astype(np.int16)
    tof = jp.make_tof(width, sigma, 3.0, 29)
    xs, xe = c["xstart"], c["xend"]
    xsd, xed, imgd = dev(xs, cuda_device), dev(xe, cuda_device), dev(img, cuda_device)
    plan = jp.LmPlan(xsd, xed, dev(tb, cuda_device), g.n, g.origin, g.voxsize, tof, n_subsets=2).set_path(1)
    p = jp.jp_fwd_tof_lm_planned(plan, imgd)
    assert_fwd(p, oracle.fwd_tof_lm(xs, xe, tb, img, g.origin, g.voxsize, width, sigma, 3.0))
    y = rng.uniform(0.5, 2, 4_000).astype(np.float32)
    b = jp.jp_back_tof_lm_planned(plan, dev(y, cuda_device))
    assert_back(b, oracle.back_tof_lm(xs, xe, tb, y, g.n, g.origin, g.voxsize, width, sigma, 3.0))
    pn = jp.jp_fwd_lm_planned(plan, imgd)
    assert_fwd(pn, oracle.fwd(xs, xe, img, g.origin, g.voxsize))
    bn = jp.jp_back_lm_planned(plan, dev(y, cuda_device))
    assert_back(bn, oracle.back(xs, xe, y, g.n, g.origin, g.voxsize))
    plan.destroy()


@pytest.mark.parametrize("path", [1, 2])
def test_planned_listmode_in_plan_order(cuda_device, scanner, events, path):
    """jp_*_tof_lm_planned_sorted take / return per-event arrays in PLAN order: forward == the caller-order result
    moved to plan order by jp_lm_plan_permute, bit for bit; the adjoint of a permuted y == the caller-order adjoint;
    the permutation round-trips; per subset as well"""
    g, ph = scanner
    if path == 1:
        xs, xe, tb = _line_events(seed=31)
    else:
        xs, xe, tb = (t.numpy()[..., :80_007] for t in events)
    n = xs.shape[1]
    tof = jp.make_tof(17.0, 13.6, 3.0, 29)
    imgd = dev(ph, cuda_device)
    plan = jp.LmPlan(dev(xs, cuda_device), dev(xe, cuda_device), dev(tb, cuda_device), g.n, g.origin, g.voxsize, tof,
                     n_subsets=3).set_path(path)
    p = jp.jp_fwd_tof_lm_planned(plan, imgd)
    ps = jp.jp_fwd_tof_lm_planned_sorted(plan, imgd)
    assert torch.equal(ps, jp.jp_lm_plan_permute(plan, p, True))
    assert torch.equal(jp.jp_lm_plan_permute(plan, ps, False), p)
    assert_fwd(p, oracle.fwd_tof_lm(xs, xe, tb, ph, g.origin, g.voxsize, 17.0, 13.6, 3.0))
    y = inputs.uniform_values(n, 0.5, 2.0, seed=19).to(cuda_device)
    ys = jp.jp_lm_plan_permute(plan, y, True)
    b = jp.jp_back_tof_lm_planned(plan, y)
    bs = jp.jp_back_tof_lm_planned_sorted(plan, ys)
    assert float((b - bs).abs().max()) <= 1e-5 * float(b.abs().max())
    assert_back(bs, oracle.back_tof_lm(xs, xe, tb, y.cpu().numpy(), g.n, g.origin, g.voxsize, 17.0, 13.6, 3.0))
    b1 = jp.jp_back_tof_lm_planned_sorted(plan, ys, subset=1)
    assert float((b1 - jp.jp_back_tof_lm_planned(plan, y, subset=1)).abs().max()) <= 1e-5 * float(b.abs().max())
    plan.destroy()
