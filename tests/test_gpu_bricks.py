"""Parity of the listmode BRICK kernels (csrc/jp_brick.cu: path 3 of a listmode plan) against the float64 oracle.

path 3 = forward projection on shared-memory image bricks (TMA tile loads), adjoint with float atomics (quad image),
both reading one TOF table.  (Rounds 1-2 had a path 4, the adjoint staged in the bricks in int32 fixed point with one
scale per chunk; it could not hold the 1e-3 OSEM bound on low-count data and was removed: set_path(4) is an error.)
Tolerances: BASELINE.json north_star (forward rel-L2 <= 1e-5, max abs <= 1e-4 max; back max abs <= 1e-4 max; adjoint gap
<= 1e-4); OSEM images: DESIGN.md A14 (rel-L2 <= 1e-4, max abs <= 1e-3 max).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs

pytestmark = pytest.mark.gpu


def _cmp_fwd(got, ref):
    g = got.detach().cpu().numpy().astype(np.float64)
    assert np.isfinite(g).all()
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    mx = np.abs(g - ref).max() / np.abs(ref).max()
    assert rel <= 1e-5, f"forward rel-L2 {rel:.3e}"
    assert mx <= 1e-4, f"forward max abs / max {mx:.3e}"


def _cmp_back(got, ref, tol=1e-4):
    g = got.detach().cpu().numpy().astype(np.float64)
    assert np.isfinite(g).all()
    mx = np.abs(g - ref).max() / np.abs(ref).max()
    assert mx <= tol, f"back max abs / max {mx:.3e}"


@pytest.fixture(scope="module")
def scanner_events():
    ph = inputs.phantom()
    xs, xe, tb = inputs.listmode_events(200_003, seed=inputs.BASE_SEED + 31, img=ph, chunk=1_000_000)
    return ph, xs, xe, tb


@pytest.mark.parametrize("path", [3])
def test_scanner_events_on_bricks(cuda_device, scanner_events, path):
    """crystal-snapped events of the ring scanner, 3 subsets (ragged: 200003 events), both index orders"""
    ph, xs, xe, tb = scanner_events
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    tof = jp.make_tof(tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    args = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas)
    n = xs.shape[1]
    d = cuda_device
    img = torch.from_numpy(ph).to(d)
    y = inputs.uniform_values(n, 0.5, 2.0, seed=77)
    plan = jp.LmPlan(xs.to(d), xe.to(d), tb.to(d), g.n, g.origin, g.voxsize, tof, n_subsets=3).set_path(path)
    ref = oracle.fwd_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), ph, g.origin, g.voxsize, *args)
    bref = oracle.back_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), y.numpy(), g.n, g.origin, g.voxsize, *args)
    p = jp.jp_fwd_tof_lm_planned(plan, img)
    _cmp_fwd(p, ref)
    b = jp.jp_back_tof_lm_planned(plan, y.to(d))
    _cmp_back(b, bref)
    a = float((p.double() * y.to(d).double()).sum())
    assert abs(a - float((img.double() * b.double()).sum())) <= 1e-4 * abs(a)
    # one subset only: the other events' entries stay untouched
    p1 = torch.full((n,), -1.0, device=d)
    jp.jp_fwd_tof_lm_planned(plan, img, subset=1, out=p1)
    sel = np.arange(1, n, 3)
    _cmp_fwd(p1[torch.from_numpy(sel).to(d)], ref[sel])
    rest = np.setdiff1d(np.arange(n), sel)
    assert float(p1[torch.from_numpy(rest).to(d)].max()) == -1.0
    # plan order
    ps = jp.jp_fwd_tof_lm_planned_sorted(plan, img)
    # (an event's pieces are summed with float atomics: equal up to the order of <= ~6 additions, not bit for bit)
    assert float((jp.jp_lm_plan_permute(plan, ps, False) - p).abs().max()) <= 2e-6 * float(p.max())
    bs = jp.jp_back_tof_lm_planned_sorted(plan, jp.jp_lm_plan_permute(plan, y.to(d), True))
    _cmp_back(bs, bref)
    plan.destroy()


@pytest.mark.parametrize("shape,vox", [((32, 32, 16), (4.0, 4.0, 4.0)), ((45, 37, 18), (3.0, 3.5, 2.5)), ((70, 33, 40), (2.0, 4.0, 3.0))])
@pytest.mark.parametrize("path", [3])
def test_random_chords_on_bricks(cuda_device, shape, vox, path):
    """random chords of a cylinder (all three principal axes, misses, ties), images whose sizes are not multiples of
    the brick, an axial size that is not a multiple of 4 (no TMA box: plain loads), anisotropic voxels, a centre offset"""
    rng = np.random.default_rng(5 + shape[0])
    n = 60_001
    g = inputs.Geometry(shape, vox)
    R = 0.8 * max(s * v for s, v in zip(shape, vox))
    ph0, ph1 = rng.uniform(0, 2 * np.pi, n), rng.uniform(0, 2 * np.pi, n)
    zr = 0.6 * shape[2] * vox[2]
    xs = np.stack([R * np.cos(ph0), R * np.sin(ph0), rng.uniform(-zr, zr, n)]).astype(np.float32)
    xe = np.stack([R * np.cos(ph1), R * np.sin(ph1), rng.uniform(-zr, zr, n)]).astype(np.float32)
    xs[:, :50] = np.float32(np.round(xs[:, :50]))          # a few exact ties / axis-parallel candidates
    xe[:, :50] = np.float32(np.round(xe[:, :50]))
    tb = rng.integers(-6, 7, n).astype(np.int16)
    img = rng.random(shape).astype(np.float32)
    y = rng.uniform(0.5, 2.0, n).astype(np.float32)
    W, sig, ns, coff = 11.0, 9.0, 3.0, 1.5
    tof = jp.make_tof(W, sig, ns, 27, center_offset=coff)
    d = cuda_device
    plan = jp.LmPlan(torch.from_numpy(xs).to(d), torch.from_numpy(xe).to(d), torch.from_numpy(tb).to(d), g.n, g.origin,
                     g.voxsize, tof, n_subsets=4).set_path(path)
    ref = oracle.fwd_tof_lm(xs, xe, tb, img, g.origin, g.voxsize, W, sig, ns, center_offset=coff)
    bref = oracle.back_tof_lm(xs, xe, tb, y, g.n, g.origin, g.voxsize, W, sig, ns, center_offset=coff)
    assert (ref > 0).mean() > 0.3
    _cmp_fwd(jp.jp_fwd_tof_lm_planned(plan, torch.from_numpy(img).to(d)), ref)
    _cmp_back(jp.jp_back_tof_lm_planned(plan, torch.from_numpy(y).to(d)), bref)
    plan.destroy()


def test_brick_plan_adjoint_value_range(cuda_device, scanner_events):
    """the adjoint of a brick plan (float atomics that read the brick kernels' TOF table): values spanning six decades,
    mixed signs, zeros, and Inf / NaN (which must propagate as on the per-event path)"""
    ph, xs, xe, tb = scanner_events
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    tof = jp.make_tof(tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    args = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas)
    n = xs.shape[1]
    d = cuda_device
    rng = np.random.default_rng(11)
    y = (10.0 ** rng.uniform(-3, 3, n) * rng.choice([-1.0, 1.0], n)).astype(np.float32)
    y[rng.random(n) < 0.1] = 0.0
    plan = jp.LmPlan(xs.to(d), xe.to(d), tb.to(d), g.n, g.origin, g.voxsize, tof, n_subsets=2).set_path(3)
    bref = oracle.back_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), y, g.n, g.origin, g.voxsize, *args)
    _cmp_back(jp.jp_back_tof_lm_planned(plan, torch.from_numpy(y).to(d)), bref)
    # non-finite values propagate into the voxels of the event's TOF window (the oracle, which also multiplies Inf by the
    # zero weights outside the window, marks the whole LOR: the GPU set is a subset of its set); all other voxels agree
    y2 = y.copy()
    bad_ev = rng.choice(n, 7, replace=False)
    y2[bad_ev[:4]] = np.inf
    y2[bad_ev[4:]] = np.nan
    ref2 = oracle.back_tof_lm(xs.numpy(), xe.numpy(), tb.numpy(), y2, g.n, g.origin, g.voxsize, *args)
    got2 = jp.jp_back_tof_lm_planned(plan, torch.from_numpy(y2).to(d)).cpu().numpy().astype(np.float64)
    refbad = ~np.isfinite(ref2)
    gotbad = ~np.isfinite(got2)
    assert gotbad.sum() >= 7 * 30 and (gotbad & ~refbad).sum() <= 0.01 * refbad.sum()
    ok = ~refbad & ~gotbad
    assert np.abs(got2[ok] - bref[ok]).max() <= 1e-4 * np.abs(bref).max()
    plan.destroy()


def test_osem_on_bricks_dense_sensitivity(cuda_device, scanner_events):
    """listmode OSEM on the brick path with a sensitivity image that is positive in the whole field of view (the sparse
    sensitivity with zeros inside the object is the case of test_config4_small_osem_planned)"""
    ph, xs, xe, tb = scanner_events
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    tof = jp.make_tof(tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    args = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas)
    d = cuda_device
    sx, se = inputs.sinogram_lors(views=range(0, 256, 2), radial=range(-128, 129, 1), device=d)
    sx, se = sx[:, ::7].contiguous(), se[:, ::7].contiguous()
    sens = jp.jp_back(sx, se, torch.ones(sx.shape[1], device=d), g.n, g.origin, g.voxsize)
    sens32 = sens.cpu().numpy()
    r = np.hypot(*np.meshgrid((np.arange(200) - 99.5) * 2, (np.arange(200) - 99.5) * 2, indexing="ij"))
    assert sens32[r < 190].min() > 0.0
    x0 = np.ones(g.n, dtype=np.float32)
    ref = oracle.lm_osem(xs.numpy(), xe.numpy(), tb.numpy(), sens32.astype(np.float64), x0, g.origin, g.voxsize, *args,
                         n_subsets=4, n_iter=2)
    for path in (3,):
        plan = jp.LmPlan(xs.to(d), xe.to(d), tb.to(d), g.n, g.origin, g.voxsize, tof, n_subsets=4).set_path(path)
        x = torch.from_numpy(x0).to(d)
        jp.jp_lm_osem_planned(plan, sens, x, n_iter=2)
        got = x.cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all()
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mx = np.abs(got - ref).max() / np.abs(ref).max()
        assert rel <= 1e-4, f"path {path}: OSEM rel-L2 {rel:.3e}"
        assert mx <= 1e-3, f"path {path}: OSEM max abs / max {mx:.3e}"
        plan.destroy()


def test_bricks_small_lists(cuda_device):
    """fewer events than subsets, and a plan whose events all miss the image"""
    g = inputs.Geometry((32, 32, 16), (4.0, 4.0, 4.0))
    d = cuda_device
    tof = jp.make_tof(9.0, 7.0, 3.0, 27)
    xs = torch.tensor([[-150.0, 0.0], [3.0, -150.0], [1.0, 2.0]], device=d)
    xe = torch.tensor([[150.0, 1.0], [2.0, 150.0], [-1.0, 0.5]], device=d)
    tb = torch.tensor([0, 1], dtype=torch.int16, device=d)
    img = torch.ones(g.n, device=d)
    for path in (3,):
        plan = jp.LmPlan(xs, xe, tb, g.n, g.origin, g.voxsize, tof, n_subsets=5).set_path(path)
        p = jp.jp_fwd_tof_lm_planned(plan, img)
        ref = oracle.fwd_tof_lm(xs.cpu().numpy(), xe.cpu().numpy(), tb.cpu().numpy(), np.ones(g.n, dtype=np.float32), g.origin,
                                g.voxsize, 9.0, 7.0, 3.0)
        assert np.abs(p.cpu().numpy() - ref).max() <= 1e-5 * ref.max()
        b = jp.jp_back_tof_lm_planned(plan, torch.ones(2, device=d))
        assert abs(float(b.double().sum()) - float(p.double().sum())) <= 1e-4 * float(p.double().sum())
        plan.destroy()
        far = jp.LmPlan(xs + 1000.0, xe + 1000.0, tb, g.n, g.origin, g.voxsize, tof, n_subsets=2).set_path(path)
        assert float(jp.jp_fwd_tof_lm_planned(far, img).abs().max()) == 0.0
        assert float(jp.jp_back_tof_lm_planned(far, torch.ones(2, device=d)).abs().max()) == 0.0
        far.destroy()


def test_removed_staged_path_is_rejected(cuda_device):
    """jp_lm_plan_set_path accepts 0..3 only: the fixed-point brick adjoint (former path 4) is gone from the ABI"""
    g = inputs.Geometry((32, 32, 16), (4.0, 4.0, 4.0))
    d = cuda_device
    tof = jp.make_tof(9.0, 7.0, 3.0, 27)
    xs = torch.tensor([[-150.0, 0.0], [3.0, -150.0], [1.0, 2.0]], device=d)
    xe = torch.tensor([[150.0, 1.0], [2.0, 150.0], [-1.0, 0.5]], device=d)
    tb = torch.tensor([0, 1], dtype=torch.int16, device=d)
    plan = jp.LmPlan(xs, xe, tb, g.n, g.origin, g.voxsize, tof, n_subsets=1)
    for bad in (4, 5, -1):
        with pytest.raises(jp.JosephError):
            plan.set_path(bad)
    plan.set_path(3).set_path(0)
    plan.destroy()
