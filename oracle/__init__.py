"""float64 CPU oracle for the Joseph projector -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It does not import the CUDA package
``paper_2212_12519_b200`` and that package does not import it.

The arithmetic lives in ``joseph_oracle.c`` (plain C, IEEE double, OpenMP over LORs), written from
PAPER.md section 2.1 with the readings A1..A14 of SURVEY.md section 8(c).  This module only
marshals numpy arrays into it.  ``build()`` compiles it with gcc.
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
