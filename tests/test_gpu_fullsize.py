"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot run 151.6 M LORs / 40 M events in seconds, so (task statement, parity bar):
  forward   the full-size launch is compared with the oracle on SAMPLED outputs (seeded random LORs plus
            whole tracks that contain the 45 degree tie views and the degenerate r = +-128 LORs);
  back      the full-size launch gets a sinogram that is zero outside a sampled subset S of the LORs, so
            its result is the oracle's back projection of the LORs of S alone -- compared voxel by voxel;
            plus a property that holds at any size: <A x, y> = <x, A^T y> with the dense y;
  counts    LOR / event / subset counts and the principal axis of every sampled LOR: bit exact.
Tolerances are BASELINE.json north_star's (see test_gpu_parity.py).
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs
from test_gpu_parity import ADJ_GAP, adj_gap, assert_back, assert_fwd

pytestmark = pytest.mark.gpu

G = inputs.GEOM_SCANNER
TOFP = inputs.TofParams()
TOF_ARGS = (TOFP.tofbin_width, TOFP.sigma_tof, TOFP.n_sigmas, TOFP.n_tofbins)


def _tof():
    return jp.make_tof(TOFP.tofbin_width, TOFP.sigma_tof, TOFP.n_sigmas, TOFP.n_tofbins)


def _sample(n, k, seed, extra=()):
    rng = np.random.default_rng(seed)
    idx = np.unique(np.concatenate([rng.integers(0, n, k)] + [np.asarray(e, dtype=np.int64) for e in extra]))
    return torch.from_numpy(idx)


def _track(v_index, r, n_views_total=inputs.N_VIEWS):
    """all 2304 ring pairs of sinogram bin (view position v_index in the list, radial offset r)"""
    base = (v_index * inputs.N_RADIAL + (r + 128)) * 2304
    return np.arange(base, base + 2304)


@pytest.fixture(scope="module")
def phantom_dev(cuda_device):
    ph = inputs.phantom()
    return ph, torch.from_numpy(ph).to(cuda_device)


def test_config1_full_nontof(cuda_device, phantom_dev):
    ph, imgd = phantom_dev
    xs, xe = inputs.sinogram_lors(device=cuda_device)
    n = xs.shape[1]
    assert n == 151_584_768                                               # LOR count: bit exact
    # sample: 150k random LORs + tie view 64 (r = 0, 17), view 192 (r = -5), rim (r = 64), degenerate r = 128
    extra = [_track(64, 0), _track(64, 17), _track(192, -5), _track(10, 64), _track(3, 128), _track(255, -128)]
    idx = _sample(n, 150_000, 1, extra).to(cuda_device)
    sxs, sxe = xs[:, idx].contiguous(), xe[:, idx].contiguous()
    hxs, hxe = sxs.cpu().numpy(), sxe.cpu().numpy()

    ax = jp.jp_classify(xs, xe)
    assert np.array_equal(ax[idx].cpu().numpy(), oracle.classify(hxs, hxe, G.n, G.origin, G.voxsize))
    del ax
    p = jp.jp_fwd(xs, xe, imgd, G.origin, G.voxsize)
    ref = oracle.fwd(hxs, hxe, ph, G.origin, G.voxsize)
    assert (ref > 0).mean() > 0.2          # 44 % of configs[1] LORs reach the image, fewer the phantom
    assert_fwd(p[idx], ref)

    # back: the full launch with y supported on the sample only
    y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 101, device=cuda_device)
    ys = torch.zeros_like(y)
    ys[idx] = y[idx]
    b = jp.jp_back(xs, xe, ys, G.n, G.origin, G.voxsize)
    assert_back(b, oracle.back(hxs, hxe, ys[idx].cpu().numpy(), G.n, G.origin, G.voxsize))
    del ys, b
    # adjointness of the full-size pair with the dense y
    bd = jp.jp_back(xs, xe, y, G.n, G.origin, G.voxsize)
    assert adj_gap(p, y, imgd, bd) <= ADJ_GAP
    # the sensitivity image of configs[4] is this operator applied to ones: sum(A^T 1) = sum(A 1)
    ones_img = torch.ones_like(imgd)
    p1 = jp.jp_fwd(xs, xe, ones_img, G.origin, G.voxsize)
    sens = jp.jp_back(xs, xe, torch.ones_like(y), G.n, G.origin, G.voxsize)
    gap = abs(float(p1.double().sum()) - float(sens.double().sum())) / float(p1.double().sum())
    assert gap <= ADJ_GAP


def test_config1_full_nontof_planned(cuda_device, phantom_dev):
    """configs[1] in the launch configuration bench.py times: a sinogram plan over all 151,584,768 LORs (65,792 tracks
    of 2304 ring pairs) and the whole-track kernels k_fwd_track / k_back_track on a grid of 65,792 x pieces CTAs, with
    the 64-bit output offsets and the skipping of the tracks that miss the image (56 % of them) that only this size
    exercises.  Forward: sampled outputs against the oracle (incl. the tie, rim and degenerate tracks) and EVERY
    output against the unplanned call (itself oracle-checked in test_config1_full_nontof); back: masked y against
    the oracle voxel by voxel, dense y through the adjoint identity."""
    ph, imgd = phantom_dev
    xs, xe = inputs.sinogram_lors(device=cuda_device)
    n = xs.shape[1]
    plan = jp.SinoPlan(xs, xe)
    assert plan.regular and plan.n == n
    extra = [_track(64, 0), _track(64, 17), _track(192, -5), _track(10, 64), _track(3, 128), _track(255, -128),
             _track(0, -128), _track(255, 128)]                             # first and last track of the list
    idx = _sample(n, 150_000, 2, extra).to(cuda_device)
    hxs, hxe = xs[:, idx].cpu().numpy(), xe[:, idx].cpu().numpy()
    p = torch.full((n,), float("nan"), dtype=torch.float32, device=cuda_device)   # every output must be written
    jp.jp_fwd_planned(plan, imgd, G.origin, G.voxsize, out=p)
    ref = oracle.fwd(hxs, hxe, ph, G.origin, G.voxsize)
    assert_fwd(p[idx], ref)
    pu = jp.jp_fwd(xs, xe, imgd, G.origin, G.voxsize)
    assert bool(torch.isfinite(p).all())
    assert float((p - pu).abs().max()) <= 2e-5 * float(pu.abs().max())      # all 151.6 M outputs: track path == tile path
    del pu, xs, xe                # the planned calls read the plan's track table, not the 3.6 GB of end points
    y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 101, device=cuda_device)
    ys = torch.zeros_like(y)
    ys[idx] = y[idx]
    b = jp.jp_back_planned(plan, ys, G.n, G.origin, G.voxsize)
    assert_back(b, oracle.back(hxs, hxe, ys[idx].cpu().numpy(), G.n, G.origin, G.voxsize))
    del ys, b
    bd = jp.jp_back_planned(plan, y, G.n, G.origin, G.voxsize)
    assert adj_gap(p, y, imgd, bd) <= ADJ_GAP
    # accumulate semantics at full size: a second pass into the same image doubles it
    bd2 = jp.jp_back_planned(plan, y, G.n, G.origin, G.voxsize, img=bd.clone())
    assert float((bd2 - 2 * bd).abs().max()) <= 1e-4 * float(bd.abs().max())
    plan.destroy()


def test_config2_full_tof_sino(cuda_device, phantom_dev):
    ph, imgd = phantom_dev
    xs, xe = inputs.sinogram_lors(views=inputs.SUBSET_VIEWS, device=cuda_device)
    n = xs.shape[1]
    assert n == 9_474_048
    # view 64 is the 5th view of the subset (tie view), view 192 the 13th
    extra = [_track(4, 0)[::9], _track(12, 30)[::9], _track(0, 64)[::9]]
    idx = _sample(n, 12_000, 2, extra).to(cuda_device)
    hxs, hxe = xs[:, idx].cpu().numpy(), xe[:, idx].cpu().numpy()
    tof = _tof()
    p = jp.jp_fwd_tof_sino(xs, xe, imgd, G.origin, G.voxsize, tof)
    assert p.shape == (n, 29)
    ref = oracle.fwd_tof_sino(hxs, hxe, ph, G.origin, G.voxsize, *TOF_ARGS)
    assert_fwd(p[idx], ref)
    # T1 at full size: bins sum to erf(3/sqrt2) x non-TOF for every LOR (phantom radius 150 mm < 205 mm)
    pn = jp.jp_fwd(xs, xe, imgd, G.origin, G.voxsize)
    assert torch.allclose(p.sum(1), 0.99730020393674 * pn, rtol=3e-5, atol=2e-3)
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=inputs.BASE_SEED + 102, device=cuda_device)
    ys = torch.zeros_like(y)
    ys[idx] = y[idx]
    b = jp.jp_back_tof_sino(xs, xe, ys, G.n, G.origin, G.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(hxs, hxe, ys[idx].cpu().numpy(), G.n, G.origin, G.voxsize, *TOF_ARGS))
    bd = jp.jp_back_tof_sino(xs, xe, y, G.n, G.origin, G.voxsize, tof)
    assert adj_gap(p, y, imgd, bd) <= ADJ_GAP
    # the planned calls (track tiles of the sinogram plan: the configuration bench.py times), same checks
    plan = jp.SinoPlan(xs, xe)
    assert plan.regular and plan.track_length == 2304 and plan.n_tracks == 16 * 257 and plan.n == n
    pp = jp.jp_fwd_tof_sino_planned(plan, imgd, G.origin, G.voxsize, tof)
    assert_fwd(pp[idx], ref)
    assert torch.allclose(pp.sum(1), 0.99730020393674 * pn, rtol=3e-5, atol=2e-3)
    assert float((pp - p).abs().max()) <= 2e-5 * float(p.abs().max())
    del p, pn
    b = jp.jp_back_tof_sino_planned(plan, ys, G.n, G.origin, G.voxsize, tof)
    assert_back(b, oracle.back_tof_sino(hxs, hxe, ys[idx].cpu().numpy(), G.n, G.origin, G.voxsize, *TOF_ARGS))
    bp = jp.jp_back_tof_sino_planned(plan, y, G.n, G.origin, G.voxsize, tof)
    assert adj_gap(pp, y, imgd, bp) <= ADJ_GAP
    assert float((bp - bd).abs().max()) <= 1e-4 * float(bd.abs().max())    # dense y: tile path == per-LOR path
    plan.destroy()


@pytest.fixture(scope="module")
def events_full(cuda_device):
    xs, xe, tb = inputs.listmode_events(40_000_000, device=cuda_device, img=inputs.phantom())
    return xs, xe, tb


def test_config3_full_tof_lm(cuda_device, phantom_dev, events_full):
    ph, imgd = phantom_dev
    xs, xe, tb = events_full
    n = xs.shape[1]
    assert n == 40_000_000 and tb.dtype == torch.int16
    idx = _sample(n, 120_000, 3).to(cuda_device)
    hxs, hxe, htb = xs[:, idx].cpu().numpy(), xe[:, idx].cpu().numpy(), tb[idx].cpu().numpy()
    tof = _tof()
    ref = oracle.fwd_tof_lm(hxs, hxe, htb, ph, G.origin, G.voxsize, *TOF_ARGS[:3])
    y = inputs.uniform_values(n, 0.5, 2.0, seed=inputs.BASE_SEED + 103, device=cuda_device)
    ys = torch.zeros_like(y)
    ys[idx] = y[idx]
    bref = oracle.back_tof_lm(hxs, hxe, htb, ys[idx].cpu().numpy(), G.n, G.origin, G.voxsize, *TOF_ARGS[:3])
    # unplanned calls (acquisition order)
    p = jp.jp_fwd_tof_lm(xs, xe, tb, imgd, G.origin, G.voxsize, tof)
    assert_fwd(p[idx], ref)
    assert_back(jp.jp_back_tof_lm(xs, xe, tb, ys, G.n, G.origin, G.voxsize, tof), bref)
    # planned calls (sorted events, the configuration bench.py times), results in caller order
    plan = jp.LmPlan(xs, xe, tb, G.n, G.origin, G.voxsize, tof, n_subsets=20)
    assert [plan.subset_count(m) for m in range(20)] == [2_000_000] * 20 and plan.subset_count(-1) == n
    pp = jp.jp_fwd_tof_lm_planned(plan, imgd)
    assert_fwd(pp[idx], ref)
    assert_back(jp.jp_back_tof_lm_planned(plan, ys), bref)
    bd = jp.jp_back_tof_lm_planned(plan, y)
    assert adj_gap(pp, y, imgd, bd) <= ADJ_GAP
    # the other kernel paths of the same plan at full size: quad image (2), image bricks forward + float adjoint (3)
    for path in (2, 3):
        plan.set_path(path)
        assert_fwd(jp.jp_fwd_tof_lm_planned(plan, imgd)[idx], ref)
        assert_back(jp.jp_back_tof_lm_planned(plan, ys), bref)
        assert adj_gap(pp, y, imgd, jp.jp_back_tof_lm_planned(plan, y)) <= ADJ_GAP
    plan.destroy()


def test_config4_osem_full_image(cuda_device, phantom_dev, events_full):
    """configs[4] geometry (200x200x96 image, 20 subsets, 3 iterations, sens = non-TOF A^T 1 over all 151.6 M
    configs[1] LORs) on the first JP_OSEM_EVENTS events (default 4 M; 40000000 = the full config, about
    ten minutes of oracle time on 16 cores) against the float64 oracle OSEM."""
    ph, imgd = phantom_dev
    nev = int(os.environ.get("JP_OSEM_EVENTS", "4000000"))
    xs, xe, tb = (t[..., :nev].contiguous() for t in events_full)
    sx, se = inputs.sinogram_lors(device=cuda_device)
    sens = jp.jp_back(sx, se, torch.ones(sx.shape[1], device=cuda_device), G.n, G.origin, G.voxsize)
    del sx, se
    tof = _tof()
    x = torch.ones(G.n, device=cuda_device)
    plan = jp.LmPlan(xs, xe, tb, G.n, G.origin, G.voxsize, tof, n_subsets=20)
    jp.jp_lm_osem_planned(plan, sens, x, n_iter=3)             # the plan's choice: image bricks forward, float adjoint
    x2 = torch.ones(G.n, device=cuda_device)
    jp.jp_lm_osem(xs, xe, tb, sens, x2, G.origin, G.voxsize, tof, n_subsets=20, n_iter=3)
    sens32 = sens.cpu().numpy()
    ref = oracle.lm_osem(xs.cpu().numpy(), xe.cpu().numpy(), tb.cpu().numpy(), sens32.astype(np.float64),
                         np.ones(G.n, dtype=np.float32), G.origin, G.voxsize, *TOF_ARGS[:3], n_subsets=20, n_iter=3)
    for got in (x, x2):
        g = got.cpu().numpy().astype(np.float64)
        assert np.isfinite(g).all()
        rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
        mx = np.abs(g - ref).max() / np.abs(ref).max()
        assert rel <= 1e-4, f"OSEM rel-L2 {rel:.3e}"
        assert mx <= 1e-3, f"OSEM max abs / max {mx:.3e}"
    plan.destroy()


def test_config4_full_density_subset(cuda_device, phantom_dev, events_full):
    """configs[4] at the event density bench.py times (a plan over all 40 M events x 20 subsets: 2 M events per subset,
    about 20 events per line and subset -- the regime in which the plan picks the image bricks): ONE subset's
    projection half of the OSEM update, b = A_m^T (1 / A_m x), against the oracle's forward -> ratio -> back over
    the same 2 M events, every voxel, for each kernel path the plan can pick by itself (0 = its own choice, 1 line
    tiles, 2 quad image, 3 bricks forward + float adjoint)."""
    ph, imgd = phantom_dev
    xs, xe, tb = events_full
    tof = _tof()
    m = 7
    x_h = (ph + 0.25).astype(np.float32)                 # positive everywhere: every event's expectation is > 1e-9
    x = torch.from_numpy(x_h).to(cuda_device)
    sub = torch.arange(m, xs.shape[1], 20, device=cuda_device)      # reading A14: subset m = events e with e mod 20 == m
    hxs, hxe, htb = xs[:, sub].cpu().numpy(), xe[:, sub].cpu().numpy(), tb[sub].cpu().numpy()
    assert hxs.shape[1] == 2_000_000
    ybar = oracle.fwd_tof_lm(hxs, hxe, htb, x_h, G.origin, G.voxsize, *TOF_ARGS[:3])
    r = np.where(ybar > 1e-9, 1.0 / np.maximum(ybar, 1e-300), 0.0)
    assert (ybar > 1e-3).all()
    bref = oracle.back_tof_lm(hxs, hxe, htb, r, G.n, G.origin, G.voxsize, *TOF_ARGS[:3])
    plan = jp.LmPlan(xs, xe, tb, G.n, G.origin, G.voxsize, tof, n_subsets=20)
    assert plan.subset_count(m) == 2_000_000
    for path in (0, 1, 2, 3):
        plan.set_path(path)
        out = torch.full(G.n, float("nan"), dtype=torch.float32, device=cuda_device)    # the call overwrites b
        b = jp.jp_lm_osem_planned_backratio(plan, m, x, out=out)
        err = assert_back(b, bref)
        assert err <= 1e-4, f"path {path}"
    plan.destroy()


def test_sino_osem_full_subset(cuda_device, phantom_dev):
    """SURVEY.md 8(f) row 3 at the size and launch configuration bench.py --config 5 times per subset (9,474,048 LORs
    x 29 bins, fused ratio epilogue): the emission sinogram is zero outside a sampled set S of LORs, so the ratio is
    zero there and the update is the oracle's update over the LORs of S alone (mult and contam are dense)."""
    ph, imgd = phantom_dev
    xs, xe = inputs.sinogram_lors(views=inputs.SUBSET_VIEWS, device=cuda_device)
    n = xs.shape[1]
    extra = [_track(4, 0)[::9], _track(12, 30)[::9]]
    idx = _sample(n, 10_000, 5, extra).to(cuda_device)
    hxs, hxe = xs[:, idx].cpu().numpy(), xe[:, idx].cpu().numpy()
    tof = _tof()
    y = torch.zeros((n, 29), dtype=torch.float32, device=cuda_device)
    y[idx] = inputs.uniform_values((idx.numel(), 29), 0.0, 3.0, seed=inputs.BASE_SEED + 305, device=cuda_device)
    mult = inputs.uniform_values(n, 0.2, 1.0, seed=inputs.BASE_SEED + 306, device=cuda_device)
    contam = inputs.uniform_values((n, 29), 0.01, 0.1, seed=inputs.BASE_SEED + 307, device=cuda_device)
    sens = torch.ones((1,) + tuple(G.n), dtype=torch.float32, device=cuda_device)
    x0 = ph + np.float32(0.1)
    x = torch.from_numpy(x0).to(cuda_device)
    jp.jp_sino_osem_tof(xs, xe, [0, n], y, mult, contam, sens, x, G.origin, G.voxsize, tof, n_iter=1)
    k = idx.numel()
    ref = oracle.sino_osem_tof(hxs, hxe, [0, k], y[idx].cpu().numpy(), mult[idx].cpu().numpy(),
                               contam[idx].cpu().numpy(), np.ones((1,) + tuple(G.n)), x0, G.origin, G.voxsize,
                               *TOF_ARGS, n_iter=1)
    assert_back(x, ref)
    plan = jp.SinoPlan(xs, xe)
    xp = torch.from_numpy(x0).to(cuda_device)
    jp.jp_sino_osem_tof_planned(plan, [0, n], y, mult, contam, sens, xp, G.origin, G.voxsize, tof, n_iter=1)
    assert_back(xp, ref)
    # and a dense run: finite, non-negative, zero where the start image is zero; planned == unplanned
    y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=inputs.BASE_SEED + 308, device=cuda_device)
    x = imgd.clone()
    jp.jp_sino_osem_tof(xs, xe, [0, n], y, mult, contam, sens, x, G.origin, G.voxsize, tof, n_iter=1)
    assert torch.isfinite(x).all() and float(x.min()) >= 0.0
    assert float(x[imgd == 0].abs().max()) == 0.0
    xp = imgd.clone()
    jp.jp_sino_osem_tof_planned(plan, [0, n], y, mult, contam, sens, xp, G.origin, G.voxsize, tof, n_iter=1)
    assert float((xp - x).abs().max()) <= 1e-4 * float(x.abs().max())
    plan.destroy()
