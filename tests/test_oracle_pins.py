"""Pins of the float64 oracle (oracle/joseph_oracle.c) against what the paper and the mathematics
fix -- never against itself and never against the CUDA path.  SURVEY.md section 8(c) pin names.

CPU only (``-m "not gpu"``).
"""
import math
import os

import numpy as np
import pytest
import torch
from scipy import integrate, ndimage

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")

# ---- the 4x4x4 test image of pin W ----------------------------------------------------------------
N4 = (4, 4, 4)
V4 = np.array([1.0, 1.5, 2.0])
O4 = -(np.array(N4) - 1) / 2.0 * V4
_i0, _i1, _i2 = np.meshgrid(*[np.arange(4)] * 3, indexing="ij")
F4 = 1.0 + _i0 + 4.0 * _i1 + 16.0 * _i2

TOF = dict(tofbin_width=17.0, sigma_tof=13.6, n_sigmas=3.0, n_tofbins=29)


def _col(*pts):
    return np.array(pts, dtype=np.float64).T


def _read_table(name):
    rows = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


def _random_lors(rng, n, radius=6.0, zmax=4.0):
    """chords of a cylinder around a small image, all three principal axes occur"""
    s = rng.uniform(-1, 1, (3, n))
    e = rng.uniform(-1, 1, (3, n))
    s /= np.linalg.norm(s, axis=0)
    e /= np.linalg.norm(e, axis=0)
    return s * radius, e * radius


# ---- W: worked examples, golden values --------------------------------------------------------------
@pytest.mark.parametrize("row", _read_table("worked_examples.txt"), ids=lambda r: r[0])
def test_W_worked_examples(row):
    name = row[0]
    s = _col([float(x) for x in row[1:4]])
    e = _col([float(x) for x in row[4:7]])
    img = np.ones(N4) if name == "C3" else F4
    p = oracle.fwd(s, e, img, O4, V4)[0]
    assert oracle.classify(s, e, N4, O4, V4)[0] == int(row[7])
    assert p == pytest.approx(float(row[9]), rel=2e-11)
    # cf is observable through the all-ones image when the ray stays inside the voxel-centre hull
    if name in ("W-A", "W-B", "C3"):
        ones = oracle.fwd(s, e, np.ones(N4), O4, V4)[0]
        assert ones == pytest.approx(4 * V4[int(row[7])] * float(row[8]) / V4[int(row[7])], rel=2e-11)


# ---- C1/C2/C3: chord closed forms -------------------------------------------------------------------
@pytest.mark.parametrize("p", [0, 1, 2])
def test_C1_axis_aligned_chord(p):
    n = (5, 6, 7)
    v = np.array([1.25, 2.0, 0.75])
    o = np.array([-3.0, 1.0, 10.0])
    q = [a for a in range(3) if a != p]
    s = np.zeros(3)
    e = np.zeros(3)
    s[p], e[p] = o[p] - 50.0, o[p] + 80.0
    for a, u in zip(q, (1.3, 2.6)):           # interior crossing point, in voxel units
        s[a] = e[a] = o[a] + u * v[a]
    val = oracle.fwd(_col(s), _col(e), np.ones(n), o, v)[0]
    assert val == pytest.approx(n[p] * v[p], rel=1e-13)
    # reversed direction gives the same
    assert oracle.fwd(_col(e), _col(s), np.ones(n), o, v)[0] == pytest.approx(n[p] * v[p], rel=1e-13)


@pytest.mark.parametrize("phi", [0.0, 0.25, 0.9])
def test_C2_rim_ramp(phi):
    """outer half-voxel shell: zero padding makes the value ramp linearly to 0"""
    n = (5, 6, 7)
    v = np.array([1.0, 2.0, 3.0])
    o = np.zeros(3)
    for (q, uq, expect) in [(1, n[1] - 1 + phi, 1 - phi), (1, -1.0 + phi, phi), (1, -1.0, 0.0),
                            (1, float(n[1]), 0.0), (2, n[2] - 1 + phi, 1 - phi), (2, -1.5, 0.0)]:
        s = np.array([-20.0, 2.2 * v[1], 3.1 * v[2]])
        s[q] = uq * v[q]
        e = s.copy()
        e[0] = 30.0
        val = oracle.fwd(_col(s), _col(e), np.ones(n), o, v)[0]
        assert val == pytest.approx(n[0] * v[0] * expect, abs=1e-12)


def test_C3_oblique_chord():
    """all-ones image, ray inside the voxel-centre hull on every plane: n_p v_p L / |d_p|"""
    rng = np.random.default_rng(1)
    n = (9, 8, 7)
    v = np.array([1.0, 1.5, 2.0])
    o = -(np.array(n) - 1) / 2.0 * v
    for p in range(3):
        q = [a for a in range(3) if a != p]
        for _ in range(20):
            s = np.zeros(3)
            e = np.zeros(3)
            s[p], e[p] = -40.0, 45.0
            half = (np.array(n) - 1) / 2.0 * v
            # entry/exit points of the hull faces of axis p, kept inside the hull in q
            a_in = rng.uniform(-0.9, 0.9, 2) * half[q]
            a_out = rng.uniform(-0.9, 0.9, 2) * half[q]
            # extend the line through (−half_p, a_in) and (+half_p, a_out) to s_p and e_p
            for k, a in enumerate(q):
                slope = (a_out[k] - a_in[k]) / (2 * half[p])
                s[a] = a_in[k] + slope * (s[p] + half[p])
                e[a] = a_in[k] + slope * (e[p] + half[p])
            d = e - s
            if np.argmax(np.abs(d)) != p:
                continue
            val = oracle.fwd(_col(s), _col(e), np.ones(n), o, v)[0]
            assert val == pytest.approx(n[p] * v[p] * np.linalg.norm(d) / abs(d[p]), rel=1e-12)


# ---- L: each plane is the zero-padded order-1 interpolant of the slice (library routines) -----------
def _fwd_via_library(s, e, img, o, v, interp):
    d = e - s
    p = int(np.argmax(np.abs(d)))
    q1, q2 = [a for a in range(3) if a != p]
    n = img.shape
    cf = v[p] * np.linalg.norm(d) / abs(d[p])
    total = 0.0
    for i in range(n[p]):
        t = (o[p] + i * v[p] - s[p]) / d[p]
        if t < 0 or t > 1:
            continue
        u1 = (s[q1] + t * d[q1] - o[q1]) / v[q1]
        u2 = (s[q2] + t * d[q2] - o[q2]) / v[q2]
        total += interp(np.take(img, i, axis=p), u1, u2)
    return cf * total


def _interp_scipy(sl, u1, u2):
    return float(ndimage.map_coordinates(sl, [[u1], [u2]], order=1, mode="grid-constant", cval=0.0)[0])


def _interp_torch(sl, u1, u2):
    h, w = sl.shape
    gx = 2.0 * u2 / (w - 1) - 1.0
    gy = 2.0 * u1 / (h - 1) - 1.0
    grid = torch.tensor([[[[gx, gy]]]], dtype=torch.float64)
    out = torch.nn.functional.grid_sample(torch.from_numpy(np.ascontiguousarray(sl))[None, None], grid,
                                          mode="bilinear", padding_mode="zeros", align_corners=True)
    return float(out[0, 0, 0, 0])


@pytest.mark.parametrize("interp", [_interp_scipy, _interp_torch], ids=["scipy", "torch"])
def test_L_library_interpolant(interp):
    rng = np.random.default_rng(2)
    n = (6, 5, 7)
    v = np.array([1.0, 1.5, 2.0])
    o = -(np.array(n) - 1) / 2.0 * v + np.array([0.3, -0.2, 0.1])
    img = rng.uniform(0, 1, n)
    s, e = _random_lors(rng, 60, radius=9.0)
    p = oracle.fwd(s, e, img, o, v)
    seen = set()
    for j in range(s.shape[1]):
        seen.add(int(np.argmax(np.abs(e[:, j] - s[:, j]))))
        ref = _fwd_via_library(s[:, j], e[:, j], img, o, v, interp)
        assert p[j] == pytest.approx(ref, rel=1e-11, abs=1e-12)
    assert seen == {0, 1, 2}


# ---- BF: brute-force exact intersection on 4x4x4 ----------------------------------------------------
def _exact_line_integral(s, e, img, o, v):
    """Siddon-type: exact integral of the piecewise-constant image along the segment s->e."""
    n = img.shape
    d = e - s
    ts = [0.0, 1.0]
    for a in range(3):
        if d[a] != 0:
            for k in range(n[a] + 1):
                t = (o[a] + (k - 0.5) * v[a] - s[a]) / d[a]
                if 0 < t < 1:
                    ts.append(t)
    ts = np.unique(ts)
    L = np.linalg.norm(d)
    total = 0.0
    for t0, t1 in zip(ts[:-1], ts[1:]):
        m = s + 0.5 * (t0 + t1) * d
        idx = np.floor((m - o) / v + 0.5).astype(int)
        if np.all(idx >= 0) and np.all(idx < n):
            total += img[tuple(idx)] * (t1 - t0) * L
    return total


def test_BF_exact_intersection():
    # (i) axis-aligned LORs through voxel centres: Joseph == exact integral
    for p in range(3):
        for a in range(4):
            for b in range(4):
                idx = [0, 0, 0]
                q = [x for x in range(3) if x != p]
                idx[q[0]], idx[q[1]] = a, b
                s = O4 + np.array(idx) * V4
                e = s.copy()
                s[p], e[p] = -30.0, 30.0
                jos = oracle.fwd(_col(s), _col(e), F4, O4, V4)[0]
                assert jos == pytest.approx(_exact_line_integral(s, e, F4, O4, V4), rel=1e-12)
    # (ii) uniform image, ray inside the voxel-centre hull: both give a chord; Joseph's chord is that
    # of the centre-to-centre slab extended by half a voxel at both ends (n_p v_p), the exact one the
    # box chord; they agree when the ray leaves through the two faces of axis p
    s = np.array([-20.0, -0.9, -1.3])
    e = np.array([20.0, 1.5, 2.1])
    jos = oracle.fwd(_col(s), _col(e), np.ones(N4), O4, V4)[0]
    assert jos == pytest.approx(_exact_line_integral(s, e, np.ones(N4), O4, V4), rel=1e-12)
    # (iii) generic rays: Joseph is a rectangle-rule approximation -> loose sanity bound only
    rng = np.random.default_rng(3)
    ss, ee = _random_lors(rng, 200, radius=8.0)
    jos = oracle.fwd(ss, ee, F4, O4, V4)
    ex = np.array([_exact_line_integral(ss[:, j], ee[:, j], F4, O4, V4) for j in range(200)])
    # (on a 4^3 image most rays graze the rim, where zero padding and the box differ by up to ~2 voxels)
    assert np.abs(jos - ex).max() < 2.0 * F4.max() * V4.max()
    assert abs(jos.sum() - ex.sum()) / ex.sum() < 0.03
    assert np.corrcoef(jos, ex)[0, 1] > 0.97


# ---- M / ADJ: exact adjoint --------------------------------------------------------------------------
def _dense_matrix(fwd_fn, n):
    nv = int(np.prod(n))
    cols = []
    for x in range(nv):
        unit = np.zeros(nv)
        unit[x] = 1.0
        cols.append(fwd_fn(unit.reshape(n)).ravel())
    return np.array(cols).T       # (n_out, nv)


def test_M_dense_matrix_transpose():
    rng = np.random.default_rng(4)
    s, e = _random_lors(rng, 40, radius=7.0)
    it = rng.integers(-2, 3, 40).astype(np.int16)
    tof = dict(tofbin_width=1.7, sigma_tof=1.36, n_sigmas=3.0)
    # non-TOF
    A = _dense_matrix(lambda f: oracle.fwd(s, e, f, O4, V4), N4)
    y = rng.uniform(0, 1, 40)
    bp = oracle.back(s, e, y, N4, O4, V4)
    assert np.abs(bp.ravel() - A.T @ y).max() < 1e-13 * max(1.0, np.abs(bp).max())
    # the matrix also reproduces the forward projection of F4 (linearity)
    assert np.allclose(A @ F4.ravel(), oracle.fwd(s, e, F4, O4, V4), rtol=1e-12)
    # TOF sinogram
    A = _dense_matrix(lambda f: oracle.fwd_tof_sino(s, e, f, O4, V4, n_tofbins=5, **tof), N4)
    y = rng.uniform(0, 1, (40, 5))
    bp = oracle.back_tof_sino(s, e, y, N4, O4, V4, n_tofbins=5, **tof)
    assert np.abs(bp.ravel() - A.T @ y.ravel()).max() < 1e-13 * max(1.0, np.abs(bp).max())
    # TOF listmode
    A = _dense_matrix(lambda f: oracle.fwd_tof_lm(s, e, it, f, O4, V4, **tof), N4)
    y = rng.uniform(0, 1, 40)
    bp = oracle.back_tof_lm(s, e, it, y, N4, O4, V4, **tof)
    assert np.abs(bp.ravel() - A.T @ y).max() < 1e-13 * max(1.0, np.abs(bp).max())


def test_M_autograd_of_library_interpolant():
    """back projection == gradient of <A x, y> w.r.t. x with A built from torch grid_sample"""
    rng = np.random.default_rng(5)
    n = (5, 4, 6)
    v = np.array([1.0, 1.5, 2.0])
    o = -(np.array(n) - 1) / 2.0 * v
    s, e = _random_lors(rng, 25, radius=8.0)
    y = rng.uniform(0, 1, 25)
    x = torch.from_numpy(rng.uniform(0, 1, n)).requires_grad_(True)
    total = torch.zeros((), dtype=torch.float64)
    for j in range(25):
        sj, ej = s[:, j], e[:, j]
        d = ej - sj
        p = int(np.argmax(np.abs(d)))
        q1, q2 = [a for a in range(3) if a != p]
        cf = v[p] * np.linalg.norm(d) / abs(d[p])
        for i in range(n[p]):
            t = (o[p] + i * v[p] - sj[p]) / d[p]
            if t < 0 or t > 1:
                continue
            u1 = (sj[q1] + t * d[q1] - o[q1]) / v[q1]
            u2 = (sj[q2] + t * d[q2] - o[q2]) / v[q2]
            sl = x.select(p, i)
            grid = torch.tensor([[[[2 * u2 / (sl.shape[1] - 1) - 1, 2 * u1 / (sl.shape[0] - 1) - 1]]]],
                                dtype=torch.float64)
            val = torch.nn.functional.grid_sample(sl[None, None], grid, mode="bilinear",
                                                  padding_mode="zeros", align_corners=True)[0, 0, 0, 0]
            total = total + y[j] * cf * val
    total.backward()
    bp = oracle.back(s, e, y, n, o, v)
    assert np.abs(bp - x.grad.numpy()).max() < 1e-12


def test_ADJ_all_operators():
    rng = np.random.default_rng(6)
    n = (12, 10, 8)
    v = np.array([2.0, 2.5, 3.0])
    o = -(np.array(n) - 1) / 2.0 * v
    s, e = _random_lors(rng, 500, radius=30.0)
    s = s.astype(np.float32)
    e = e.astype(np.float32)
    it = rng.integers(-3, 4, 500).astype(np.int16)
    tof = dict(tofbin_width=4.0, sigma_tof=3.1, n_sigmas=3.0)
    x = rng.uniform(0, 1, n)

    def gap(Ax, y, Aty):
        a, b = float((Ax * y).sum()), float((x * Aty).sum())
        return abs(a - b) / abs(a)

    y = rng.uniform(0, 1, 500)
    assert gap(oracle.fwd(s, e, x, o, v), y, oracle.back(s, e, y, n, o, v)) < 1e-13
    y = rng.uniform(0, 1, (500, 11))
    assert gap(oracle.fwd_tof_sino(s, e, x, o, v, n_tofbins=11, **tof), y,
               oracle.back_tof_sino(s, e, y, n, o, v, n_tofbins=11, **tof)) < 1e-13
    y = rng.uniform(0, 1, 500)
    assert gap(oracle.fwd_tof_lm(s, e, it, x, o, v, **tof), y,
               oracle.back_tof_lm(s, e, it, y, n, o, v, **tof)) < 1e-13
    # back projections ACCUMULATE into the given image
    img = np.full(n, 2.0)
    out = oracle.back(s, e, y, n, o, v, img=img)
    assert out is img
    assert np.allclose(img - 2.0, oracle.back(s, e, y, n, o, v), rtol=1e-12, atol=1e-12)


# ---- TOF pins ----------------------------------------------------------------------------------------
def _scanner_like(rng, n_lors):
    """LORs between points of a cylinder r=400, |z|<94 -- like configs 1-3"""
    phi = rng.uniform(0, 2 * np.pi, (2, n_lors))
    z = rng.uniform(-94, 94, (2, n_lors))
    s = np.stack([400 * np.cos(phi[0]), 400 * np.sin(phi[0]), z[0]]).astype(np.float32)
    e = np.stack([400 * np.cos(phi[1]), 400 * np.sin(phi[1]), z[1]]).astype(np.float32)
    return s, e


def test_T1_bin_sum_equals_truncated_nontof():
    """sum over the 29 bins = erf(3/sqrt 2) x non-TOF for activity within |tau| <= 205.7 mm"""
    rng = np.random.default_rng(7)
    n = (50, 50, 24)
    v = np.array([8.0, 8.0, 8.0])
    o = -(np.array(n) - 1) / 2.0 * v
    ax = [o[a] + np.arange(n[a]) * v[a] for a in range(3)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    img = ((X ** 2 + Y ** 2) <= 150.0 ** 2) * rng.uniform(0.5, 1.5, n)
    s, e = _scanner_like(rng, 300)
    nontof = oracle.fwd(s, e, img, o, v)
    tofp = oracle.fwd_tof_sino(s, e, img, o, v, **TOF)
    assert (nontof > 0).sum() > 50
    frac = math.erf(3.0 / math.sqrt(2.0))
    assert frac == pytest.approx(0.99730020393674, rel=1e-13)
    assert np.allclose(tofp.sum(1), frac * nontof, rtol=1e-12, atol=1e-12)


def _quad_weight(tau, centre, delta, sigma, nsig):
    """integral over the bin of the Gaussian truncated at nsig sigma -- by numerical quadrature"""
    def pdf(x):
        z = x - tau
        return math.exp(-0.5 * (z / sigma) ** 2) / (sigma * math.sqrt(2 * math.pi)) if abs(z) <= nsig * sigma else 0.0
    lo, hi = centre - delta / 2, centre + delta / 2
    pts = [p for p in (tau - nsig * sigma, tau + nsig * sigma) if lo < p < hi]
    val, _ = integrate.quad(pdf, lo, hi, points=pts or None, epsabs=1e-13, epsrel=1e-13, limit=200)
    return val


@pytest.mark.parametrize("p", [0, 1, 2])
@pytest.mark.parametrize("tau", [0.0, 5.0, -23.7, 61.3])
def test_T2_point_source_vs_quadrature(p, tau):
    n = [9, 9, 9]
    n[p] = 101
    v = np.array([2.0, 2.0, 2.0])
    o = -(np.array(n) - 1) / 2.0 * v
    # voxel on the LOR at distance tau from the midpoint (midpoint = 0): index along p
    ip = 50 + int(round(tau / v[p]))
    pos = o[p] + ip * v[p]
    img = np.zeros(n)
    idx = [4, 4, 4]
    idx[p] = ip
    img[tuple(idx)] = 1.0
    s = np.zeros(3)
    e = np.zeros(3)
    s[p], e[p] = -300.0, 300.0
    out = oracle.fwd_tof_sino(_col(s), _col(e), img, o, v, **TOF)[0]
    for k in range(29):
        ref = v[p] * _quad_weight(pos, (k - 14) * 17.0, 17.0, 13.6, 3.0)
        assert out[k] == pytest.approx(ref, abs=2e-11)
    # reversed LOR mirrors the bins (A9)
    out_r = oracle.fwd_tof_sino(_col(e), _col(s), img, o, v, **TOF)[0]
    assert np.allclose(out_r, out[::-1], atol=1e-14)


def test_T2_point_source_golden():
    n = (101, 3, 3)
    v = np.array([1.0, 2.0, 2.0])
    o = -(np.array(n) - 1) / 2.0 * v
    s, e = _col([-300.0, 0.0, 0.0]), _col([300.0, 0.0, 0.0])
    for row in _read_table("tof_point_source.txt"):
        tau, it, w = float(row[0]), int(row[1]), float(row[2])
        img = np.zeros(n)
        img[50 + int(tau), 1, 1] = 1.0
        lm = oracle.fwd_tof_lm(s, e, np.array([it], dtype=np.int16), img, o, v, 17.0, 13.6, 3.0)[0]
        assert lm == pytest.approx(v[0] * w, abs=2e-10)
    # bins further out are exactly zero (truncation)
    img = np.zeros(n)
    img[50, 1, 1] = 1.0
    for it in (-4, -3, 3, 4):
        assert oracle.fwd_tof_lm(s, e, np.array([it], dtype=np.int16), img, o, v, 17.0, 13.6, 3.0)[0] == 0.0


def test_T3_listmode_equals_sinogram_column():
    rng = np.random.default_rng(8)
    n = (40, 40, 20)
    v = np.array([10.0, 10.0, 10.0])
    o = -(np.array(n) - 1) / 2.0 * v
    img = rng.uniform(0, 1, n)
    s, e = _scanner_like(rng, 200)
    sino = oracle.fwd_tof_sino(s, e, img, o, v, **TOF)
    it = rng.integers(-14, 15, 200).astype(np.int16)
    lm = oracle.fwd_tof_lm(s, e, it, img, o, v, 17.0, 13.6, 3.0)
    assert np.allclose(lm, sino[np.arange(200), it + 14], rtol=1e-13, atol=1e-15)
    # adjoint: LM back projection == sinogram back projection of a one-hot y
    y = rng.uniform(0, 1, 200)
    onehot = np.zeros((200, 29))
    onehot[np.arange(200), it + 14] = y
    b1 = oracle.back_tof_lm(s, e, it, y, n, o, v, 17.0, 13.6, 3.0)
    b2 = oracle.back_tof_sino(s, e, onehot, n, o, v, **TOF)
    assert np.allclose(b1, b2, rtol=1e-12, atol=1e-14)
    # centre offset shifts tau (A8)
    lm_off = oracle.fwd_tof_lm(s, e, it, img, o, v, 17.0, 13.6, 3.0, center_offset=17.0)
    lm_m1 = oracle.fwd_tof_lm(s, e, (it + 1).astype(np.int16), img, o, v, 17.0, 13.6, 3.0)
    assert np.allclose(lm_off, lm_m1, rtol=1e-11, atol=1e-14)


# ---- S: symmetries -----------------------------------------------------------------------------------
def test_S_symmetries():
    rng = np.random.default_rng(9)
    n = (10, 9, 8)
    v = np.array([2.0, 2.5, 3.0])
    o = -(np.array(n) - 1) / 2.0 * v
    img = rng.uniform(0, 1, n)
    s, e = _random_lors(rng, 300, radius=25.0)
    it = rng.integers(-2, 3, 300).astype(np.int16)
    tof = dict(tofbin_width=4.0, sigma_tof=3.1, n_sigmas=3.0)
    p0 = oracle.fwd(s, e, img, o, v)
    # swap s <-> e: non-TOF unchanged, TOF bins mirrored
    assert np.allclose(oracle.fwd(e, s, img, o, v), p0, rtol=1e-12, atol=1e-14)
    t0 = oracle.fwd_tof_sino(s, e, img, o, v, n_tofbins=9, **tof)
    t1 = oracle.fwd_tof_sino(e, s, img, o, v, n_tofbins=9, **tof)
    assert np.allclose(t1, t0[:, ::-1], rtol=1e-12, atol=1e-14)
    l0 = oracle.fwd_tof_lm(s, e, it, img, o, v, **tof)
    l1 = oracle.fwd_tof_lm(e, s, (-it).astype(np.int16), img, o, v, **tof)
    assert np.allclose(l1, l0, rtol=1e-12, atol=1e-14)
    # translate image and LORs together
    sh = np.array([[12.5], [-7.25], [3.0]])
    assert np.allclose(oracle.fwd(s + sh, e + sh, img, o + sh[:, 0], v), p0, rtol=1e-11, atol=1e-13)
    # permute axes of image and coordinates consistently (exercises all three code paths)
    for perm in [(1, 2, 0), (2, 0, 1), (0, 2, 1)]:
        pp = oracle.fwd(s[list(perm)], e[list(perm)], np.ascontiguousarray(img.transpose(perm)),
                        o[list(perm)], v[list(perm)])
        assert np.allclose(pp, p0, rtol=1e-12, atol=1e-14)
        tt = oracle.fwd_tof_sino(s[list(perm)], e[list(perm)], np.ascontiguousarray(img.transpose(perm)),
                                 o[list(perm)], v[list(perm)], n_tofbins=9, **tof)
        assert np.allclose(tt, t0, rtol=1e-12, atol=1e-14)
    # scale all lengths by lambda: non-TOF result x lambda
    lam = 1.7
    assert np.allclose(oracle.fwd(lam * s, lam * e, img, lam * o, lam * v), lam * p0, rtol=1e-11)
    # linearity and non-negativity
    img2 = rng.uniform(0, 1, n)
    assert np.allclose(oracle.fwd(s, e, 2 * img + 3 * img2, o, v),
                       2 * p0 + 3 * oracle.fwd(s, e, img2, o, v), rtol=1e-12)
    assert (p0 >= 0).all() and (t0 >= 0).all() and (l0 >= 0).all()


def test_A3_tie_break_lowest_axis():
    """exact 45 degree LORs: the lowest axis index wins (convention, reading A3)"""
    s = _col([-10.0, -10.0, 0.0], [-10.0, 0.0, -10.0], [0.0, -10.0, -10.0], [-10.0, -10.0, -10.0])
    e = _col([10.0, 10.0, 0.0], [10.0, 0.0, 10.0], [0.0, 10.0, 10.0], [10.0, -30.0, 10.0])
    assert list(oracle.classify(s, e, N4, O4, V4)) == [0, 0, 1, 0]
    # float32 inputs are promoted exactly: a one-ulp difference decides
    a = np.float32(10.0)
    b = np.nextafter(a, np.float32(20.0))
    s32 = np.zeros((3, 2), dtype=np.float32)
    e32 = np.array([[a, a], [b, a], [0, 0]], dtype=np.float32)
    assert list(oracle.classify(s32, e32, N4, O4, V4)) == [1, 0]


# ---- D: degenerate -----------------------------------------------------------------------------------
def test_D_degenerate_and_missing():
    img = F4
    s = _col([1.0, 1.0, 1.0], [50.0, 50.0, 50.0], [-10.0, 30.0, 0.0])
    e = _col([1.0, 1.0, 1.0], [60.0, 55.0, 52.0], [10.0, 30.0, 0.0])
    p = oracle.fwd(s, e, img, O4, V4)
    assert np.all(p == 0.0) and np.all(np.isfinite(p))
    t = oracle.fwd_tof_sino(s, e, img, O4, V4, **TOF)
    assert np.all(t == 0.0)
    b = oracle.back(s, e, np.ones(3), N4, O4, V4)
    assert np.all(b == 0.0)
    # empty LOR list
    z = np.zeros((3, 0))
    assert oracle.fwd(z, z, img, O4, V4).shape == (0,)
    assert np.all(oracle.back(z, z, np.zeros(0), N4, O4, V4) == 0.0)


# ---- O: OSEM count preservation ----------------------------------------------------------------------
def test_O_osem_count_preservation():
    """one subset, one EM update: sum_voxels sens*x_new = #events with ybar > 0 when sens = A^T 1
    restricted to the event list itself (listmode likelihood)"""
    rng = np.random.default_rng(10)
    n = (40, 40, 12)
    v = np.array([8.0, 8.0, 8.0])
    o = -(np.array(n) - 1) / 2.0 * v
    s, e = _scanner_like(rng, 4000)
    s[2] *= 0.3
    e[2] *= 0.3
    it = rng.integers(-2, 3, 4000).astype(np.int16)
    sens = rng.uniform(0.5, 2.0, n)
    x0 = rng.uniform(0.5, 1.5, n)
    x1, ybar = oracle.lm_osem(s, e, it, sens, x0, o, v, 17.0, 13.6, 3.0, n_subsets=1, n_iter=1,
                              return_ybar=True)
    assert np.allclose(ybar, oracle.fwd_tof_lm(s, e, it, x0, o, v, 17.0, 13.6, 3.0), rtol=1e-13)
    n_pos = int((ybar > 1e-9).sum())
    assert n_pos > 1000
    assert float((sens * x1).sum()) == pytest.approx(n_pos, rel=1e-12)
    # subsets: e mod n_subsets, update uses b * n_subsets / sens
    x2 = oracle.lm_osem(s, e, it, sens, x0, o, v, 17.0, 13.6, 3.0, n_subsets=4, n_iter=1)
    x = x0.copy()
    for m in range(4):
        sel = np.arange(m, 4000, 4)
        yb = oracle.fwd_tof_lm(s[:, sel], e[:, sel], it[sel], x, o, v, 17.0, 13.6, 3.0)
        r = np.where(yb > 1e-9, 1.0 / np.where(yb > 1e-9, yb, 1.0), 0.0)
        b = oracle.back_tof_lm(s[:, sel], e[:, sel], it[sel], r, n, o, v, 17.0, 13.6, 3.0)
        x = x * b * 4 / sens
    assert np.allclose(x2, x, rtol=1e-11, atol=1e-14)
    # zero sensitivity -> zero image value
    sens0 = sens.copy()
    sens0[0, 0, 0] = 0.0
    x3 = oracle.lm_osem(s, e, it, sens0, x0, o, v, 17.0, 13.6, 3.0, n_subsets=2, n_iter=1)
    assert x3[0, 0, 0] == 0.0


def test_segment_rule_endpoint_inside_image():
    """A4: only planes between the two end points count (closed segment)"""
    n = (10, 3, 3)
    v = np.array([1.0, 1.0, 1.0])
    o = np.zeros(3)
    img = np.ones(n)
    # from x=2.0 (exactly on plane 2) to x=6.5: planes 2,3,4,5,6
    s, e = _col([2.0, 1.0, 1.0]), _col([6.5, 1.0, 1.0])
    assert oracle.fwd(s, e, img, o, v)[0] == pytest.approx(5.0, rel=1e-14)
    assert oracle.fwd(e, s, img, o, v)[0] == pytest.approx(5.0, rel=1e-14)
    s, e = _col([2.0001, 1.0, 1.0]), _col([6.0, 1.0, 1.0])
    assert oracle.fwd(s, e, img, o, v)[0] == pytest.approx(4.0, rel=1e-14)


def test_O2_osem_subsets_by_composition_of_single_subset_updates():
    """Pins what test_O only re-types: the subset rule, the order of the subsets and the x n_subsets factor of A14.
    An OSEM pass over two subsets is two EM updates in a row (Hudson & Larkin, PAPER.md:193 ref. 39).  Each update is
    computed here through the ONE-subset path -- pinned by the count identity above and by H (sinogram OSEM of the
    histogrammed list) -- on the events of that subset alone with the sensitivity sens / n_subsets, because
    x b n / sens = x b / (sens / n).  Interleaving two different event lists A, B makes subset 0 = A, subset 1 = B.
    Swapping the roles of A and B changes the result (the order is part of the convention); k identical copies of one
    list make OSEM with k subsets equal to k ML-EM iterations on that list."""
    rng = np.random.default_rng(12)
    n = (24, 24, 8)
    v = np.array([12.0, 12.0, 12.0])
    o = -(np.array(n) - 1) / 2.0 * v
    sa, ea = _scanner_like(rng, 1500)
    sb, eb = _scanner_like(rng, 1500)
    for a in (sa, ea, sb, eb):
        a[2] *= 0.25
    ta, tb = rng.integers(-2, 3, 1500).astype(np.int16), rng.integers(-2, 3, 1500).astype(np.int16)
    sens = rng.uniform(0.5, 2.0, n)
    x0 = rng.uniform(0.5, 1.5, n)
    T = (17.0, 13.6, 3.0)
    ileave = lambda p, q: np.stack([p, q], axis=-1).reshape(p.shape[:-1] + (-1,))
    s, e, it = ileave(sa, sb), ileave(ea, eb), ileave(ta, tb)
    assert np.array_equal(s[:, 0::2], sa) and np.array_equal(s[:, 1::2], sb) and np.array_equal(it[1::2], tb)
    got = oracle.lm_osem(s, e, it, sens, x0, o, v, *T, n_subsets=2, n_iter=1)
    step1 = oracle.lm_osem(sa, ea, ta, sens / 2.0, x0, o, v, *T, n_subsets=1, n_iter=1)
    step2 = oracle.lm_osem(sb, eb, tb, sens / 2.0, step1, o, v, *T, n_subsets=1, n_iter=1)
    assert np.allclose(got, step2, rtol=1e-12, atol=1e-15)
    other = oracle.lm_osem(sa, ea, ta, sens / 2.0, oracle.lm_osem(sb, eb, tb, sens / 2.0, x0, o, v, *T, n_subsets=1, n_iter=1),
                           o, v, *T, n_subsets=1, n_iter=1)
    assert np.abs(got - other).max() > 1e-6 * np.abs(got).max()          # B-then-A is a different image
    # two iterations = the same pass twice
    got2 = oracle.lm_osem(s, e, it, sens, x0, o, v, *T, n_subsets=2, n_iter=2)
    assert np.allclose(got2, oracle.lm_osem(s, e, it, sens, got, o, v, *T, n_subsets=2, n_iter=1), rtol=1e-12, atol=1e-15)
    # k interleaved copies of one list: OSEM with k subsets == k ML-EM iterations on the list with sens / k
    k = 3
    s3, e3, t3 = np.repeat(sa, k, axis=1), np.repeat(ea, k, axis=1), np.repeat(ta, k)
    osem = oracle.lm_osem(s3, e3, t3, sens, x0, o, v, *T, n_subsets=k, n_iter=1)
    mlem = oracle.lm_osem(sa, ea, ta, sens / k, x0, o, v, *T, n_subsets=1, n_iter=k)
    assert np.allclose(osem, mlem, rtol=1e-12, atol=1e-15)
