"""float64 CPU oracle for the Joseph projector -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It does not import the CUDA package
``paper_2212_12519_b200`` and that package does not import it.

The arithmetic lives in ``joseph_oracle.c`` (plain C, IEEE double, OpenMP over LORs), written from
PAPER.md section 2.1 with the readings A1..A14 of SURVEY.md section 8(c); the image-based resolution model
(readings R1-R3) is in the same file, the TOF sinogram OSEM with multiplicative factors and contamination (readings
S1-S3) is written with numpy in this module on top of the C projector calls.  Otherwise this module only marshals
numpy arrays.  ``build()`` compiles the C file with gcc.

Pins: tests/test_oracle_pins.py (projectors, listmode OSEM), tests/test_oracle_resolution.py (R1-R3),
tests/test_oracle_sino_osem.py (S1-S3).  "parity unpinned" (pure conventions the paper does not fix): A3 tie
direction, A9 TOF index origin / sign, A14 and S1 / S3 subset rules and the 1e-9 guards.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "joseph_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile joseph_oracle.c -> liboracle.so (in-tree).  No fused multiply-add contraction."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-std=c11",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Geom(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("o", C.c_double * 3), ("v", C.c_double * 3)]


class _Tof(C.Structure):
    _fields_ = [("delta", C.c_double), ("sigma", C.c_double), ("nsig", C.c_double),
                ("nbins", C.c_int32), ("coff", C.c_double)]


class _Lors(C.Structure):
    _fields_ = [("c", C.c_void_p * 6), ("is_f64", C.c_int)]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        for name in ("orc_classify", "orc_fwd", "orc_back", "orc_fwd_tof_sino", "orc_back_tof_sino",
                     "orc_fwd_tof_lm", "orc_back_tof_lm", "orc_lm_osem", "orc_num_threads", "orc_gauss3d",
                     "orc_lm_osem_res"):
            getattr(_lib, name).restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _geom(n, origin, voxsize) -> _Geom:
    g = _Geom()
    for a in range(3):
        g.n[a] = int(n[a])
        g.o[a] = float(origin[a])
        g.v[a] = float(voxsize[a])
    return g


def _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset=0.0) -> _Tof:
    return _Tof(float(tofbin_width), float(sigma_tof), float(n_sigmas), int(n_tofbins),
                float(center_offset))


def _lors(xstart, xend):
    """xstart, xend: (3, n) SoA or (n, 3) arrays, float32 (promoted exactly) or float64."""
    xs = np.asarray(xstart)
    xe = np.asarray(xend)
    if xs.ndim == 2 and xs.shape[0] != 3 and xs.shape[1] == 3:
        xs, xe = xs.T, xe.T
    assert xs.shape == xe.shape and xs.shape[0] == 3, "endpoints must be (3, n)"
    dt = np.float64 if (xs.dtype == np.float64 or xe.dtype == np.float64) else np.float32
    keep = [np.ascontiguousarray(xs[a], dtype=dt) for a in range(3)] + \
           [np.ascontiguousarray(xe[a], dtype=dt) for a in range(3)]
    l = _Lors()
    for k in range(6):
        l.c[k] = keep[k].ctypes.data
    l.is_f64 = 1 if dt == np.float64 else 0
    return l, keep, int(xs.shape[1])


def _dptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def classify(xstart, xend, n, origin, voxsize):
    l, keep, nl = _lors(xstart, xend)
    out = np.zeros(nl, dtype=np.uint8)
    g = _geom(n, origin, voxsize)
    _check(_load().orc_classify(C.byref(l), C.c_int64(nl), C.byref(g), _dptr(out)), "classify")
    return out


def fwd(xstart, xend, img, origin, voxsize):
    img = _f64(img)
    l, keep, nl = _lors(xstart, xend)
    g = _geom(img.shape, origin, voxsize)
    p = np.zeros(nl, dtype=np.float64)
    _check(_load().orc_fwd(C.byref(l), C.c_int64(0), C.c_int64(1), C.c_int64(nl), C.byref(g),
                           _dptr(img), _dptr(p)), "fwd")
    return p


def back(xstart, xend, y, n, origin, voxsize, img=None):
    """Accumulates into img (a float64 C-order array of shape n) and returns it."""
    l, keep, nl = _lors(xstart, xend)
    y = _f64(y)
    assert y.shape == (nl,)
    if img is None:
        img = np.zeros(tuple(int(x) for x in n), dtype=np.float64)
    assert img.dtype == np.float64 and img.flags.c_contiguous
    g = _geom(n, origin, voxsize)
    _check(_load().orc_back(C.byref(l), C.c_int64(0), C.c_int64(1), C.c_int64(nl), C.byref(g),
                            _dptr(y), _dptr(img)), "back")
    return img


def fwd_tof_sino(xstart, xend, img, origin, voxsize, tofbin_width, sigma_tof, n_sigmas, n_tofbins,
                 center_offset=0.0):
    img = _f64(img)
    l, keep, nl = _lors(xstart, xend)
    g = _geom(img.shape, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    p = np.zeros((nl, int(n_tofbins)), dtype=np.float64)
    _check(_load().orc_fwd_tof_sino(C.byref(l), C.c_int64(0), C.c_int64(1), C.c_int64(nl),
                                    C.byref(g), C.byref(tf), _dptr(img), _dptr(p)), "fwd_tof_sino")
    return p


def back_tof_sino(xstart, xend, y, n, origin, voxsize, tofbin_width, sigma_tof, n_sigmas, n_tofbins,
                  center_offset=0.0, img=None):
    l, keep, nl = _lors(xstart, xend)
    y = _f64(y)
    assert y.shape == (nl, int(n_tofbins))
    if img is None:
        img = np.zeros(tuple(int(x) for x in n), dtype=np.float64)
    assert img.dtype == np.float64 and img.flags.c_contiguous
    g = _geom(n, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    _check(_load().orc_back_tof_sino(C.byref(l), C.c_int64(0), C.c_int64(1), C.c_int64(nl),
                                     C.byref(g), C.byref(tf), _dptr(y), _dptr(img)), "back_tof_sino")
    return img


def _bins(tofbin, nl):
    tb = np.ascontiguousarray(tofbin, dtype=np.int16)
    assert tb.shape == (nl,)
    return tb


def fwd_tof_lm(xstart, xend, tofbin, img, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
               n_tofbins=1, center_offset=0.0):
    img = _f64(img)
    l, keep, nl = _lors(xstart, xend)
    tb = _bins(tofbin, nl)
    g = _geom(img.shape, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    p = np.zeros(nl, dtype=np.float64)
    _check(_load().orc_fwd_tof_lm(C.byref(l), _dptr(tb), C.c_int64(0), C.c_int64(1), C.c_int64(nl),
                                  C.byref(g), C.byref(tf), _dptr(img), _dptr(p)), "fwd_tof_lm")
    return p


def back_tof_lm(xstart, xend, tofbin, y, n, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
                n_tofbins=1, center_offset=0.0, img=None):
    l, keep, nl = _lors(xstart, xend)
    tb = _bins(tofbin, nl)
    y = _f64(y)
    assert y.shape == (nl,)
    if img is None:
        img = np.zeros(tuple(int(x) for x in n), dtype=np.float64)
    assert img.dtype == np.float64 and img.flags.c_contiguous
    g = _geom(n, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    _check(_load().orc_back_tof_lm(C.byref(l), _dptr(tb), C.c_int64(0), C.c_int64(1), C.c_int64(nl),
                                   C.byref(g), C.byref(tf), _dptr(y), _dptr(img)), "back_tof_lm")
    return img


def lm_osem(xstart, xend, tofbin, sens, img0, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
            n_subsets, n_iter, n_tofbins=1, center_offset=0.0, return_ybar=False):
    """Listmode OSEM (reading A14).  Returns the final float64 image (and the last ybar)."""
    l, keep, nl = _lors(xstart, xend)
    tb = _bins(tofbin, nl)
    img = np.array(img0, dtype=np.float64, order="C", copy=True)
    sens = _f64(sens)
    assert sens.shape == img.shape
    g = _geom(img.shape, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    ybar = np.zeros(nl, dtype=np.float64) if return_ybar else None
    _check(_load().orc_lm_osem(C.byref(l), _dptr(tb), C.c_int64(nl), C.byref(g), C.byref(tf),
                               _dptr(sens), _dptr(img), C.c_int(int(n_subsets)), C.c_int(int(n_iter)),
                               _dptr(ybar) if return_ybar else None), "lm_osem")
    return (img, ybar) if return_ybar else img


def fwhm_to_sigma(fwhm: float) -> float:
    """sigma of a Gaussian of the given full width at half maximum: FWHM = 2 sqrt(2 ln 2) sigma"""
    return float(fwhm) / (2.0 * np.sqrt(2.0 * np.log(2.0)))


def gauss3d(img, voxsize, sigma_mm, n_sigmas=3.0):
    """Image-based resolution model (readings R1, R2): truncated, per-axis normalised 3-D Gaussian, zero boundary."""
    img = _f64(img)
    g = _geom(img.shape, (0.0, 0.0, 0.0), voxsize)
    out = np.zeros_like(img)
    _check(_load().orc_gauss3d(_dptr(img), _dptr(out), C.byref(g), C.c_double(float(sigma_mm)),
                               C.c_double(float(n_sigmas))), "gauss3d")
    return out


def lm_osem_res(xstart, xend, tofbin, sens, img0, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
                n_subsets, n_iter, res_sigma_mm, res_n_sigmas=3.0, n_tofbins=1, center_offset=0.0):
    """Listmode OSEM with the image-based resolution model (reading R3).  Returns the final float64 image."""
    l, keep, nl = _lors(xstart, xend)
    tb = _bins(tofbin, nl)
    img = np.array(img0, dtype=np.float64, order="C", copy=True)
    sens = _f64(sens)
    assert sens.shape == img.shape
    g = _geom(img.shape, origin, voxsize)
    tf = _tof(tofbin_width, sigma_tof, n_sigmas, n_tofbins, center_offset)
    _check(_load().orc_lm_osem_res(C.byref(l), _dptr(tb), C.c_int64(nl), C.byref(g), C.byref(tf),
                                   _dptr(sens), _dptr(img), C.c_int(int(n_subsets)), C.c_int(int(n_iter)),
                                   C.c_double(float(res_sigma_mm)), C.c_double(float(res_n_sigmas))), "lm_osem_res")
    return img


# ---- TOF sinogram OSEM with multiplicative factors and additive contamination ----------
# "the projection work required for an OSEM subset update [37]-[39]"; sinogram OSEM
# keeps "the complete image volume, the emission sinogram, the forward projection and the contamination
# sinogram" on the GPU.  The paper gives no formula; this is OSEM (Hudson & Larkin, PAPER.md:193 ref. 39) for the
# usual PET model  ybar = mult * (A x) + contam  (mult: attenuation x normalisation per LOR, the same for every
# TOF bin; contam: randoms + scatter per LOR and bin).  Readings (S1-S3):
#   S1  subset m = LORs [subset_offsets[m], subset_offsets[m+1]) of the caller's list (the caller arranges the
#       list subset-major; for a ring scanner a subset is every n_subsets-th view), in order;
#   S2  r[j,k] = mult[j] y[j,k] / ybar[j,k] if ybar[j,k] > 1e-9 else 0   (the guard of A14);
#   S3  x <- x * (A_m^T r) / sens_m  where sens_m > 0, else 0;  sens_m = A_m^T (mult (x) 1_bins).
# Written with numpy on top of the pinned projector calls, in that order, nothing fused.
def sino_sens_tof(xstart, xend, subset_offsets, mult, n, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
                  n_tofbins, center_offset=0.0):
    """sens[m] = A_m^T (mult broadcast over the TOF bins): float64 [n_subsets, n0, n1, n2]"""
    off = [int(o) for o in subset_offsets]
    xs, xe = np.asarray(xstart), np.asarray(xend)
    out = np.zeros((len(off) - 1,) + tuple(int(a) for a in n), dtype=np.float64)
    for m in range(len(off) - 1):
        a, b = off[m], off[m + 1]
        if b > a:
            ones = np.repeat(np.asarray(mult, dtype=np.float64)[a:b, None], int(n_tofbins), axis=1)
            out[m] = back_tof_sino(xs[:, a:b], xe[:, a:b], ones, n, origin, voxsize, tofbin_width, sigma_tof,
                                   n_sigmas, n_tofbins, center_offset)
    return out


def sino_osem_tof(xstart, xend, subset_offsets, y, mult, contam, sens, img0, origin, voxsize, tofbin_width,
                  sigma_tof, n_sigmas, n_tofbins, n_iter, center_offset=0.0):
    """TOF sinogram OSEM (readings S1-S3).  y, contam: [n, n_tofbins]; mult: [n]; sens: [n_subsets, n0, n1, n2].
    Returns the final float64 image."""
    off = [int(o) for o in subset_offsets]
    xs, xe = np.asarray(xstart), np.asarray(xend)
    x = np.array(img0, dtype=np.float64, order="C", copy=True)
    y = np.asarray(y, dtype=np.float64)
    mult = np.asarray(mult, dtype=np.float64)
    contam = np.asarray(contam, dtype=np.float64)
    sens = np.asarray(sens, dtype=np.float64)
    for _ in range(int(n_iter)):
        for m in range(len(off) - 1):
            a, b = off[m], off[m + 1]
            if b > a:
                p = fwd_tof_sino(xs[:, a:b], xe[:, a:b], x, origin, voxsize, tofbin_width, sigma_tof, n_sigmas,
                                 n_tofbins, center_offset)
                ybar = mult[a:b, None] * p + contam[a:b]
                r = np.zeros_like(ybar)
                ok = ybar > 1e-9
                r[ok] = (mult[a:b, None] * y[a:b])[ok] / ybar[ok]
                bp = back_tof_sino(xs[:, a:b], xe[:, a:b], r, x.shape, origin, voxsize, tofbin_width, sigma_tof,
                                   n_sigmas, n_tofbins, center_offset)
            else:
                bp = np.zeros_like(x)
            pos = sens[m] > 0.0
            x = np.where(pos, x * bp / np.where(pos, sens[m], 1.0), 0.0)
    return x
