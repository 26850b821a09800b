"""Parity of jp_sino_sens_tof / jp_sino_osem_tof against oracle.sino_sens_tof /
oracle.sino_osem_tof on the same seeded inputs, through the C ABI.

Tolerances: sensitivity images are back projections (max abs <= 1e-4 max|oracle|, north_star); the OSEM image
uses the tolerance of reading A14 (rel-L2 <= 1e-4, max abs <= 1e-3 max|oracle|: float32 atomics order compounds
through the multiplicative updates)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2212_12519_b200 import binding as jp
from paper_2212_12519_b200 import inputs

pytestmark = pytest.mark.gpu


def dev(a, device):
    return torch.as_tensor(a).to(device).contiguous()


def _check_img(gpu, ref, rel_tol=1e-4, abs_tol=1e-3):
    g = gpu.detach().cpu().numpy().astype(np.float64)
    assert np.isfinite(g).all()
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    mx = np.abs(g - ref).max() / np.abs(ref).max()
    assert rel <= rel_tol, f"rel-L2 {rel:.3e}"
    assert mx <= abs_tol, f"max abs / max {mx:.3e}"
    return rel, mx


def _run(cuda_device, xs, xe, off, geom, targs, img0, y, mult, contam, n_iter):
    tof = jp.make_tof(*targs)
    dxs, dxe = dev(xs, cuda_device), dev(xe, cuda_device)
    dmult = None if mult is None else dev(mult.astype(np.float32), cuda_device)
    dcont = None if contam is None else dev(contam.astype(np.float32), cuda_device)
    nl = xs.shape[1]
    ws = torch.empty(jp.jp_sino_osem_tof_workspace_bytes(off, nl, tof), dtype=torch.uint8, device=cuda_device)
    sens = jp.jp_sino_sens_tof(dxs, dxe, off, dmult, geom.n, geom.origin, geom.voxsize, tof, workspace=ws)
    m64 = np.ones(nl) if mult is None else mult.astype(np.float32).astype(np.float64)
    c64 = np.zeros((nl, targs[3])) if contam is None else contam.astype(np.float32).astype(np.float64)
    sens_o = oracle.sino_sens_tof(xs, xe, off, m64, geom.n, geom.origin, geom.voxsize, *targs)
    smax = np.abs(sens_o).max()
    assert np.abs(sens.cpu().numpy().astype(np.float64) - sens_o).max() <= 1e-4 * smax
    # the OSEM call gets the float32 sensitivity images the library produced; the oracle its own float64 ones
    x = dev(img0.astype(np.float32), cuda_device).clone()
    jp.jp_sino_osem_tof(dxs, dxe, off, dev(y.astype(np.float32), cuda_device), dmult, dcont, sens, x, geom.origin,
                        geom.voxsize, tof, n_iter=n_iter, workspace=ws)
    ref = oracle.sino_osem_tof(xs, xe, off, y.astype(np.float32), m64, c64, sens_o, img0.astype(np.float32),
                               geom.origin, geom.voxsize, *targs, n_iter=n_iter)
    return _check_img(x, ref)


@pytest.mark.parametrize("targs,with_factors", [((9.0, 7.0, 3.0, 27), True), ((9.0, 7.0, 3.0, 27), False),
                                                ((2.5, 7.0, 3.0, 63), True)])
def test_small_random_lors(cuda_device, targs, with_factors):
    """random chords (no tracks, all principal axes, ragged subset sizes); the third case has a
    TOF window of 18 bins = the unfused generic kernels"""
    n = 5_003
    c = inputs.config0(n_lors=n)
    g = c["geom"]
    rng = np.random.default_rng(21)
    off = [0, 1700, 3302, n]
    mult = rng.uniform(0.2, 1.0, n) if with_factors else None
    contam = rng.uniform(0.01, 0.3, (n, targs[3])) if with_factors else None
    xtrue = rng.uniform(0.2, 2.0, g.n)
    ytrue = oracle.fwd_tof_sino(c["xstart"], c["xend"], xtrue, g.origin, g.voxsize, *targs)
    if with_factors:
        ytrue = mult[:, None] * ytrue + contam
    y = rng.poisson(ytrue * 5.0) / 5.0
    _run(cuda_device, c["xstart"], c["xend"], off, g, targs, np.ones(g.n), y, mult, contam, n_iter=2)


def test_scanner_views(cuda_device):
    """eight views of the configs[2] structure in two subsets (one holds the 45 degree tie view), all radial bins, the
    12 x 12 ring pairs of the first 12 rings, 29 bins of 17 mm; phantom data with attenuation-like factors and a flat
    contamination.  As in practice the start image is a field-of-view mask, here the voxels every subset sees with at
    least 1 % of its peak sensitivity (from the oracle): elsewhere the update divides by sensitivities that are
    zero or nearly zero (a few views leave holes), `sens > 0` is decided by the last bit and nothing is comparable."""
    g = inputs.GEOM_SCANNER
    tp = inputs.TofParams()
    targs = (tp.tofbin_width, tp.sigma_tof, tp.n_sigmas, tp.n_tofbins)
    subsets = ([16, 48, 80, 112], [0, 32, 64, 96])
    xs, xe = inputs.sinogram_lors(views=list(subsets[0] + subsets[1]))
    xs, xe = xs.numpy(), xe.numpy()
    idx = np.arange(xs.shape[1])
    keep = ((idx // 48) % 48 < 12) & (idx % 48 < 12)
    xs, xe = np.ascontiguousarray(xs[:, keep]), np.ascontiguousarray(xe[:, keep])
    nl = xs.shape[1]
    off = [0, nl // 2, nl]
    rng = np.random.default_rng(22)
    mu = (inputs.phantom() > 0).astype(np.float64)
    mult = np.exp(-0.0096 * oracle.fwd(xs, xe, mu, g.origin, g.voxsize)).astype(np.float32).astype(np.float64)
    sens_o = oracle.sino_sens_tof(xs, xe, off, mult, g.n, g.origin, g.voxsize, *targs)
    fov = (sens_o >= 1e-2 * sens_o.max(axis=(1, 2, 3), keepdims=True)).all(axis=0)
    assert fov.sum() > 200_000
    ph = inputs.phantom().astype(np.float64) * fov
    proj = oracle.fwd_tof_sino(xs, xe, ph, g.origin, g.voxsize, *targs)
    contam = np.full(proj.shape, 0.2 * float((mult[:, None] * proj).mean()))
    y = rng.poisson((mult[:, None] * proj + contam) * 2.0) / 2.0
    rel, mx = _run(cuda_device, xs, xe, off, g, targs, fov.astype(np.float64), y, mult, contam, n_iter=2)
    print(f"sino OSEM scanner views: rel-L2 {rel:.2e}, max abs / max {mx:.2e}")


def test_errors(cuda_device):
    c = inputs.config0(n_lors=64)
    g = c["geom"]
    tof = jp.make_tof(9.0, 7.0, 3.0, 27)
    xs, xe = dev(c["xstart"], cuda_device), dev(c["xend"], cuda_device)
    y = torch.ones(64 * 27, device=cuda_device)
    sens = torch.ones((2,) + tuple(g.n), device=cuda_device)
    x = torch.ones(g.n, device=cuda_device)
    with pytest.raises(jp.JosephError):      # offsets beyond the list
        jp.jp_sino_osem_tof(xs, xe, [0, 32, 65], y, None, None, sens, x, g.origin, g.voxsize, tof, n_iter=1,
                            workspace=torch.empty(1 << 20, dtype=torch.uint8, device=cuda_device))
    with pytest.raises(jp.JosephError):      # decreasing offsets
        jp.jp_sino_osem_tof(xs, xe, [0, 40, 32], y, None, None, sens, x, g.origin, g.voxsize, tof, n_iter=1,
                            workspace=torch.empty(1 << 20, dtype=torch.uint8, device=cuda_device))
    # an empty subset has sens = 0: the update (S3) zeroes the image, as the oracle's does
    x0 = torch.ones(g.n, device=cuda_device)
    s3 = torch.ones((3,) + tuple(g.n), device=cuda_device)
    s3[1] = 0
    jp.jp_sino_osem_tof(xs, xe, [0, 32, 32, 64], y, None, None, s3, x0, g.origin, g.voxsize, tof, n_iter=1)
    assert float(x0.abs().max()) == 0.0
    # zero iterations: image untouched
    jp.jp_sino_osem_tof(xs, xe, [0, 32, 64], y, None, None, sens, x, g.origin, g.voxsize, tof, n_iter=0)
    assert float(x.min()) == 1.0 and float(x.max()) == 1.0
