"""Pins of the oracle's image-based resolution model (readings R1-R3)."""
import numpy as np
import scipy.ndimage as ndi

import oracle

SIG = oracle.fwhm_to_sigma(4.5)     # "3D isotropic Gaussian kernel of 4.5 mm FWHM"


def test_fwhm_definition():
    # a Gaussian of this sigma is at half maximum at +-FWHM/2 (closed form)
    assert abs(np.exp(-0.5 * (2.25 / SIG) ** 2) - 0.5) < 1e-15


def test_impulse_response_closed_form():
    """R1: impulse -> outer product of per-axis normalised truncated Gaussians (anisotropic voxels)"""
    v = (2.0, 1.5, 3.0)
    x = np.zeros((15, 17, 11)); x[7, 8, 5] = 1.0
    y = oracle.gauss3d(x, v, SIG, 3.0)
    taps = []
    for a in range(3):
        r = int(np.ceil(3.0 * SIG / v[a]))
        k = np.arange(-r, r + 1)
        g = np.exp(-0.5 * (k * v[a] / SIG) ** 2)
        taps.append((r, g / g.sum()))
    ref = np.zeros_like(x)
    (r0, g0), (r1, g1), (r2, g2) = taps
    ref[7 - r0:8 + r0, 8 - r1:9 + r1, 5 - r2:6 + r2] = g0[:, None, None] * g1[None, :, None] * g2[None, None, :]
    assert np.abs(y - ref).max() < 1e-16
    assert abs(y.sum() - 1.0) < 1e-14                      # interior impulse: mass preserved


def test_against_library_filter():
    """R1 + R2 == scipy.ndimage.gaussian_filter(mode='constant', explicit radius), random image"""
    rng = np.random.default_rng(3)
    x = rng.random((12, 9, 14))
    v = (2.0, 2.0, 2.78)
    radius = [int(np.ceil(3.0 * SIG / a)) for a in v]
    ref = ndi.gaussian_filter(x, sigma=[SIG / a for a in v], mode="constant", cval=0.0, radius=radius)
    assert np.abs(oracle.gauss3d(x, v, SIG, 3.0) - ref).max() < 1e-14


def test_symmetric_operator_and_boundary():
    """R2: zero boundary makes G self-adjoint; a constant image keeps its value only in the interior"""
    rng = np.random.default_rng(4)
    x, y = rng.random((8, 10, 6)), rng.random((8, 10, 6))
    v = (2.0, 2.0, 2.0)
    a = float((oracle.gauss3d(x, v, SIG) * y).sum()); b = float((x * oracle.gauss3d(y, v, SIG)).sum())
    assert abs(a - b) <= 1e-13 * abs(a)
    ones = oracle.gauss3d(np.ones((9, 9, 9)), v, SIG)
    assert abs(ones[4, 4, 4] - 1.0) < 1e-14 and ones[0, 0, 0] < 0.4 and ones[0, 4, 4] < ones[1, 4, 4] < 1.0


def test_osem_res_reduces_to_plain_osem_and_preserves_counts():
    """R3: a kernel narrower than half a voxel is the identity -> orc_lm_osem; with the model, one EM update
    with sens = G A^T 1 preserves the number of events (sum x_new sens / ... identity of EM with a symmetric G)"""
    from paper_2212_12519_b200 import inputs
    c = inputs.config0(n_lors=3000)
    g = c["geom"]
    tb = np.random.default_rng(1).integers(-4, 5, 3000).astype(np.int16)
    args = (9.0, 7.0, 3.0)
    ones = np.ones(3000)
    sens0 = oracle.back_tof_lm(c["xstart"], c["xend"], tb, ones, g.n, g.origin, g.voxsize, *args)
    x0 = np.ones(g.n)
    plain = oracle.lm_osem(c["xstart"], c["xend"], tb, sens0, x0, g.origin, g.voxsize, *args, n_subsets=3, n_iter=1)
    ident = oracle.lm_osem_res(c["xstart"], c["xend"], tb, sens0, x0, g.origin, g.voxsize, *args, n_subsets=3,
                               n_iter=1, res_sigma_mm=0.1, res_n_sigmas=3.0)
    assert np.abs(plain - ident).max() <= 1e-13 * np.abs(plain).max()
    # count preservation: with sens = G A^T 1 (one subset), sum_v x1 sens_raw... = <G x1', .> ; check via forward model
    sens = oracle.gauss3d(sens0, g.voxsize, SIG)
    x1 = oracle.lm_osem_res(c["xstart"], c["xend"], tb, sens, x0, g.origin, g.voxsize, *args, n_subsets=1, n_iter=1,
                            res_sigma_mm=SIG)
    ybar = oracle.fwd_tof_lm(c["xstart"], c["xend"], tb, oracle.gauss3d(x0, g.voxsize, SIG), g.origin, g.voxsize, *args)
    assert abs(float((x1 * sens).sum()) - float((ybar > 1e-9).sum())) < 1e-8 * 3000
