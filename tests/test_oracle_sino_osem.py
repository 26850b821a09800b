"""Pins of the oracle's TOF sinogram OSEM with multiplicative factors and additive contamination
(readings S1-S3 in DESIGN.md).  All `-m "not gpu"`.

What fixes the update (none of these re-type the loop of oracle.sino_osem_tof):
  F   fixed point: noiseless data y = mult A x* + contam leave x* unchanged by EVERY subset update;
  V   one voxel: with contam = 0 one ML-EM update lands on the closed form sum(y) / sum(mult a) from any start;
  C   count identity of an EM update: sum_i sens_i x_new_i = sum_jk y (ybar - contam) / ybar;
  L   ML-EM (one subset) never decreases the Poisson log-likelihood (Shepp & Vardi), and does so for contam > 0;
  M   textbook matrix form: x <- x / (A^T m) * A^T (m y / (m A x + s)) with a dense A and numpy matmul;
  H   histogrammed listmode: sinogram OSEM on the histogram of an event list == listmode OSEM on the events
      (a different oracle routine, orc_lm_osem), when both use the same subsets.
"""
import numpy as np

import oracle
from paper_2212_12519_b200 import inputs

TOF = dict(tofbin_width=9.0, sigma_tof=7.0, n_sigmas=3.0, n_tofbins=15)
TARGS = (TOF["tofbin_width"], TOF["sigma_tof"], TOF["n_sigmas"], TOF["n_tofbins"])


def _problem(n_lors=1200, n_subsets=3, seed=5):
    c = inputs.config0(n_lors=n_lors)
    g = c["geom"]
    rng = np.random.default_rng(seed)
    xs, xe = c["xstart"], c["xend"]
    off = np.linspace(0, n_lors, n_subsets + 1).astype(np.int64)
    off[1] += 7                                   # unequal subsets
    mult = rng.uniform(0.2, 1.0, n_lors)
    contam = rng.uniform(0.01, 0.2, (n_lors, TOF["n_tofbins"]))
    xtrue = rng.uniform(0.5, 2.0, g.n)
    return g, xs, xe, off, mult, contam, xtrue, rng


def test_F_noiseless_data_are_a_fixed_point():
    g, xs, xe, off, mult, contam, xtrue, _ = _problem()
    sens = oracle.sino_sens_tof(xs, xe, off, mult, g.n, g.origin, g.voxsize, *TARGS)
    seen = sens.min(axis=0) > 0                  # voxels every subset sees; the others hold no activity
    assert seen.sum() > 1000
    xtrue = np.where(seen, xtrue, 0.0)
    y = mult[:, None] * oracle.fwd_tof_sino(xs, xe, xtrue, g.origin, g.voxsize, *TARGS) + contam
    x1 = oracle.sino_osem_tof(xs, xe, off, y, mult, contam, sens, xtrue, g.origin, g.voxsize, *TARGS, n_iter=2)
    assert np.abs(x1 - xtrue).max() <= 1e-12 * xtrue.max()
    # a wrong ratio (mult forgotten) would move it: the fixed point is not trivial
    y_bad = oracle.fwd_tof_sino(xs, xe, xtrue, g.origin, g.voxsize, *TARGS) + contam
    x2 = oracle.sino_osem_tof(xs, xe, off, y_bad, mult, contam, sens, xtrue, g.origin, g.voxsize, *TARGS, n_iter=1)
    assert np.abs(x2 - xtrue).max() > 1e-2


def test_V_single_voxel_closed_form():
    rng = np.random.default_rng(2)
    n = 40
    # LORs through one 30 mm voxel at the origin, oblique in x/y
    ang = rng.uniform(0, 2 * np.pi, n)
    offs = rng.uniform(-8, 8, n)
    d = np.stack([np.cos(ang), np.sin(ang), 0.1 * rng.standard_normal(n)])
    nrm = np.stack([-np.sin(ang), np.cos(ang), np.zeros(n)])
    xs = (offs * nrm - 100.0 * d).astype(np.float32)
    xe = (offs * nrm + 100.0 * d).astype(np.float32)
    geom = ((1, 1, 1), (0.0, 0.0, 0.0), (30.0, 30.0, 30.0))
    a = oracle.fwd_tof_sino(xs, xe, np.ones(geom[0]), geom[1], geom[2], *TARGS)
    assert (a.sum(axis=1) > 0).sum() > n // 2
    mult = rng.uniform(0.3, 1.0, n)
    y = rng.poisson(5.0, a.shape).astype(np.float64)
    y[a <= 1e-9] = 0.0                           # bins the voxel cannot reach carry no signal when contam = 0
    off = np.array([0, n])
    sens = oracle.sino_sens_tof(xs, xe, off, mult, *geom, *TARGS)
    for start in (0.3, 7.0):
        x = oracle.sino_osem_tof(xs, xe, off, y, mult, np.zeros_like(y), sens, np.full(geom[0], start), geom[1],
                                 geom[2], *TARGS, n_iter=1)
        assert abs(x[0, 0, 0] - y.sum() / (mult[:, None] * a).sum()) <= 1e-12 * x[0, 0, 0]


def test_C_count_identity_and_L_likelihood():
    g, xs, xe, off, mult, contam, xtrue, rng = _problem(n_subsets=1)
    ytrue = mult[:, None] * oracle.fwd_tof_sino(xs, xe, xtrue, g.origin, g.voxsize, *TARGS) + contam
    y = rng.poisson(ytrue * 20.0) / 20.0
    sens = oracle.sino_sens_tof(xs, xe, off, mult, g.n, g.origin, g.voxsize, *TARGS)

    def ybar_of(x):
        return mult[:, None] * oracle.fwd_tof_sino(xs, xe, x, g.origin, g.voxsize, *TARGS) + contam

    def loglik(x):
        yb = ybar_of(x)
        return float((y * np.log(yb) - yb).sum())

    x = np.ones(g.n)
    ll = [loglik(x)]
    for it in range(4):
        yb = ybar_of(x)
        x_new = oracle.sino_osem_tof(xs, xe, off, y, mult, contam, sens, x, g.origin, g.voxsize, *TARGS, n_iter=1)
        lhs = float((sens[0] * x_new).sum())
        rhs = float((y * (yb - contam) / yb).sum())
        assert abs(lhs - rhs) <= 1e-11 * rhs     # C
        x = x_new
        ll.append(loglik(x))
    assert all(b > a for a, b in zip(ll, ll[1:])), ll   # L (strict: not yet converged)
    assert (x >= 0).all()


def test_M_dense_matrix_textbook_form():
    rng = np.random.default_rng(9)
    geom = inputs.Geometry((4, 5, 3), (6.0, 5.0, 7.0))
    n = 90
    ph = rng.uniform(0, 2 * np.pi, (2, n))
    xs = np.stack([60 * np.cos(ph[0]), 60 * np.sin(ph[0]), rng.uniform(-12, 12, n)]).astype(np.float32)
    xe = np.stack([60 * np.cos(ph[1]), 60 * np.sin(ph[1]), rng.uniform(-12, 12, n)]).astype(np.float32)
    nb = TOF["n_tofbins"]
    nv = int(np.prod(geom.n))
    A = np.zeros((n * nb, nv))
    for v in range(nv):                          # column v = projection of the unit image e_v
        e = np.zeros(nv); e[v] = 1.0
        A[:, v] = oracle.fwd_tof_sino(xs, xe, e.reshape(geom.n), geom.origin, geom.voxsize, *TARGS).ravel()
    mult = rng.uniform(0.2, 1.0, n)
    contam = rng.uniform(0.05, 0.3, (n, nb))
    y = rng.poisson(3.0, (n, nb)).astype(np.float64)
    off = np.array([0, 31, 60, 90])
    rows = [np.arange(off[m] * nb, off[m + 1] * nb) for m in range(3)]
    mrow = np.repeat(mult, nb)
    x = rng.uniform(0.5, 1.5, nv)
    x0 = x.copy()
    sens = np.stack([A[r].T @ mrow[r] for r in rows])
    for it in range(2):
        for m in range(3):
            r = rows[m]
            ratio = mrow[r] * y.ravel()[r] / (mrow[r] * (A[r] @ x) + contam.ravel()[r])
            bp = A[r].T @ ratio
            x = np.where(sens[m] > 0, x * bp / np.where(sens[m] > 0, sens[m], 1.0), 0.0)
    sens_o = oracle.sino_sens_tof(xs, xe, off, mult, geom.n, geom.origin, geom.voxsize, *TARGS)
    assert np.abs(sens_o.reshape(3, nv) - sens).max() <= 1e-12 * sens.max()
    xo = oracle.sino_osem_tof(xs, xe, off, y, mult, contam, sens_o, x0.reshape(geom.n), geom.origin, geom.voxsize,
                              *TARGS, n_iter=2)
    assert np.abs(xo.ravel() - x).max() <= 1e-11 * x.max()


def test_H_histogrammed_listmode_equals_listmode_osem():
    """y[j,k] = number of events on LOR j in bin k, mult = 1, contam = 0, ONE subset: sinogram ML-EM and
    listmode ML-EM (orc_lm_osem on the expanded event list, sens = A^T 1 over all LOR-bins) are the same update."""
    c = inputs.config0(n_lors=400)
    g = c["geom"]
    xs, xe = c["xstart"], c["xend"]
    rng = np.random.default_rng(11)
    nb = TOF["n_tofbins"]
    y = rng.poisson(0.4, (400, nb)).astype(np.float64)
    off = np.array([0, 400])
    mult = np.ones(400)
    sens = oracle.sino_sens_tof(xs, xe, off, mult, g.n, g.origin, g.voxsize, *TARGS)
    xs_s = oracle.sino_osem_tof(xs, xe, off, y, mult, np.zeros_like(y), sens, np.ones(g.n), g.origin, g.voxsize,
                                *TARGS, n_iter=3)
    jj, kk = np.nonzero(y)
    rep = y[jj, kk].astype(np.int64)
    ev = np.repeat(jj, rep)
    tb = np.repeat(kk - (nb - 1) // 2, rep).astype(np.int16)      # reading A9: it = k - (n_tofbins - 1) / 2
    xl = oracle.lm_osem(xs[:, ev], xe[:, ev], tb, sens[0], np.ones(g.n), g.origin, g.voxsize, *TARGS[:3],
                        n_subsets=1, n_iter=3)
    assert np.abs(xs_s - xl).max() <= 1e-11 * xl.max()
