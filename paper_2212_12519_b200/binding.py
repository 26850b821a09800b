"""Thin ctypes binding over libjoseph_b200.so -- same names as include/joseph_b200.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of the library.  PyTorch
is used for device memory and streams.  There is NO CPU fallback: if the library is missing or a
tensor is not on a CUDA device the call raises.

LOR end points are passed as two float32 CUDA tensors of shape (3, n) (row a = coordinate a of all
LORs: the SoA layout of the C ABI) or as any tensors whose rows are contiguous.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjoseph_b200.so")
_lib = None

JP_MAX_TOFBINS = 64


class JosephError(RuntimeError):
    pass


class jp_geom(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("origin", C.c_float * 3), ("voxsize", C.c_float * 3)]


class jp_tof(C.Structure):
    _fields_ = [("tofbin_width_mm", C.c_float), ("sigma_tof_mm", C.c_float), ("n_sigmas", C.c_float),
                ("n_tofbins", C.c_int32), ("center_offset_mm", C.c_float)]


class jp_lors(C.Structure):
    _fields_ = [("xs", C.c_void_p), ("ys", C.c_void_p), ("zs", C.c_void_p),
                ("xe", C.c_void_p), ("ye", C.c_void_p), ("ze", C.c_void_p), ("n", C.c_int64)]


# every symbol include/joseph_b200.h declares (tests/test_abi.py checks header <-> library <-> this list)
EXPORTS = {
    "jp_fwd": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.c_void_p, C.c_void_p]),
    "jp_back": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.c_void_p, C.c_void_p]),
    "jp_fwd_tof_sino": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof),
                                  C.c_void_p, C.c_void_p]),
    "jp_back_tof_sino": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof),
                                   C.c_void_p, C.c_void_p]),
    "jp_fwd_tof_lm": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_void_p, C.POINTER(jp_geom),
                                C.POINTER(jp_tof), C.c_void_p, C.c_void_p]),
    "jp_back_tof_lm": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_void_p, C.POINTER(jp_geom),
                                 C.POINTER(jp_tof), C.c_void_p, C.c_void_p]),
    "jp_classify": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_void_p]),
    "jp_plane_steps": (C.c_int, [C.POINTER(jp_lors), C.POINTER(jp_geom), C.c_void_p, C.c_void_p]),
    "jp_plane_steps_tof_lm": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof),
                                        C.c_void_p, C.c_void_p]),
    "jp_lm_osem_workspace_bytes": (C.c_size_t, [C.c_int64, C.POINTER(jp_geom), C.c_int]),
    "jp_lm_osem": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p,
                             C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]),
    "jp_lm_plan_create": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_int,
                                    C.c_void_p, C.POINTER(C.c_void_p)]),
    "jp_lm_plan_destroy": (C.c_int, [C.c_void_p]),
    "jp_lm_plan_subset_count": (C.c_int64, [C.c_void_p, C.c_int]),
    "jp_lm_plan_set_path": (C.c_int, [C.c_void_p, C.c_int]),
    "jp_fwd_tof_lm_planned": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_back_tof_lm_planned": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_fwd_tof_lm_planned_sorted": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_back_tof_lm_planned_sorted": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_lm_plan_permute": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "jp_fwd_lm_planned": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_back_lm_planned": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_lm_osem_planned_workspace_bytes": (C.c_size_t, [C.c_void_p]),
    "jp_lm_osem_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_size_t,
                                     C.c_void_p]),
    "jp_lm_osem_planned_res": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_float, C.c_float, C.c_void_p,
                                         C.c_size_t, C.c_void_p]),
    "jp_lm_osem_planned_backratio": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t,
                                               C.c_void_p]),
    "jp_osem_update": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.POINTER(jp_geom), C.c_void_p]),
    "jp_gauss3d": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_float, C.c_float, C.c_void_p]),
    "jp_gauss3d_static": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_float, C.c_float, C.c_void_p]),
    "jp_sino_osem_tof_workspace_bytes": (C.c_size_t, [C.c_void_p, C.c_int, C.c_int64, C.POINTER(jp_tof)]),
    "jp_sino_sens_tof": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_int, C.c_void_p, C.POINTER(jp_geom),
                                   C.POINTER(jp_tof), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "jp_sino_osem_tof": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p, C.c_int, C.c_void_p,
                                   C.c_size_t, C.c_void_p]),
    "jp_sino_plan_create": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(C.c_void_p)]),
    "jp_sino_plan_info": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int32)]),
    "jp_plan_destroy": (C.c_int, [C.c_void_p]),
    "jp_fwd_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_void_p, C.c_void_p]),
    "jp_back_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_void_p, C.c_void_p]),
    "jp_fwd_tof_sino_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p,
                                          C.c_void_p]),
    "jp_back_tof_sino_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p,
                                           C.c_void_p]),
    "jp_sino_sens_tof_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.POINTER(jp_geom),
                                           C.POINTER(jp_tof), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "jp_sino_osem_tof_planned": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p, C.c_int,
                                           C.c_void_p, C.c_size_t, C.c_void_p]),
    "jp_hybrid_create": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_void_p)]),
    "jp_hybrid_destroy": (C.c_int, [C.c_void_p]),
    "jp_hybrid_worker_count": (C.c_int, [C.c_void_p]),
    "jp_hybrid_set_lors": (C.c_int, [C.c_void_p, C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof)]),
    "jp_hybrid_fwd": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_void_p]),
    "jp_hybrid_back": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.c_void_p]),
    "jp_hybrid_fwd_tof_sino": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p]),
    "jp_hybrid_back_tof_sino": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p]),
    "jp_hybrid_fwd_tof_lm": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_hybrid_back_tof_lm": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "jp_fwd_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.c_void_p]),
    "jp_back_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.c_void_p]),
    "jp_fwd_tof_sino_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p]),
    "jp_back_tof_sino_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof), C.c_void_p]),
    "jp_fwd_tof_lm_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof),
                                     C.c_void_p]),
    "jp_back_tof_lm_host": (C.c_int, [C.POINTER(jp_lors), C.c_void_p, C.c_void_p, C.POINTER(jp_geom), C.POINTER(jp_tof),
                                      C.c_void_p]),
    "jp_last_error": (C.c_char_p, []),
    "jp_version": (C.c_int, []),
}


def load():
    """dlopen the library (works without a GPU; compute calls need one).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise JosephError(f"{LIB_PATH} not found: build it with `python -m paper_2212_12519_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load().jp_last_error().decode()
        raise JosephError(f"{what} failed with code {rc}: {msg}")


def _stream(stream) -> C.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dev(t: torch.Tensor, dtype, what: str) -> torch.Tensor:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise JosephError(f"{what} must be a CUDA tensor (no CPU fallback)")
    if t.dtype != dtype:
        raise JosephError(f"{what} must be {dtype}, got {t.dtype}")
    if t.device.index != torch.cuda.current_device():
        raise JosephError(f"{what} is on cuda:{t.device.index} but the current device is cuda:{torch.cuda.current_device()} "
                          "(the library launches on the current device)")
    return t


def make_geom(n, origin, voxsize) -> jp_geom:
    g = jp_geom()
    for a in range(3):
        g.n[a] = int(n[a])
        g.origin[a] = float(origin[a])
        g.voxsize[a] = float(voxsize[a])
    return g


def make_tof(tofbin_width, sigma_tof, n_sigmas=3.0, n_tofbins=1, center_offset=0.0) -> jp_tof:
    return jp_tof(float(tofbin_width), float(sigma_tof), float(n_sigmas), int(n_tofbins), float(center_offset))


def make_lors(xstart: torch.Tensor, xend: torch.Tensor):
    """(3, n) float32 CUDA tensors -> jp_lors (plus the tensors to keep alive)."""
    _dev(xstart, torch.float32, "xstart")
    _dev(xend, torch.float32, "xend")
    if xstart.ndim != 2 or xstart.shape[0] != 3 or xend.shape != xstart.shape:
        raise JosephError("xstart / xend must both have shape (3, n)")
    rows = []
    for t in (xstart, xend):
        for a in range(3):
            row = t[a]
            if not row.is_contiguous():    # no hidden copies: a temporary would have to outlive the asynchronous call
                raise JosephError("every row of xstart / xend must be contiguous (use t.contiguous())")
            rows.append(row)
    l = jp_lors(*[r.data_ptr() for r in rows], int(xstart.shape[1]))
    return l, rows


def _img(img: torch.Tensor) -> torch.Tensor:
    _dev(img, torch.float32, "img")
    if img.ndim != 3 or not img.is_contiguous():
        raise JosephError("img must be a contiguous 3-D tensor (C order, axis 2 fastest)")
    return img


def jp_version() -> int:
    return int(load().jp_version())


def jp_classify(xstart, xend, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    out = torch.empty(l.n, dtype=torch.uint8, device=xstart.device)
    _check(load().jp_classify(C.byref(l), out.data_ptr(), _stream(stream)), "jp_classify")
    return out


def jp_plane_steps(xstart, xend, n, origin, voxsize, stream=None) -> int:
    """number of (LOR, plane) pairs the projectors visit (synchronises to return a Python int)"""
    l, keep = make_lors(xstart, xend)
    g = make_geom(n, origin, voxsize)
    total = torch.zeros(1, dtype=torch.int64, device=xstart.device)
    _check(load().jp_plane_steps(C.byref(l), C.byref(g), total.data_ptr(), _stream(stream)), "jp_plane_steps")
    return int(total.item())


def jp_plane_steps_tof_lm(xstart, xend, tofbin, n, origin, voxsize, tof: jp_tof, stream=None) -> int:
    """number of (event, plane) pairs the TOF listmode projectors visit (synchronises)"""
    l, keep = make_lors(xstart, xend)
    tofbin = _bins(tofbin, l.n)
    g = make_geom(n, origin, voxsize)
    total = torch.zeros(1, dtype=torch.int64, device=xstart.device)
    _check(load().jp_plane_steps_tof_lm(C.byref(l), tofbin.data_ptr(), C.byref(g), C.byref(tof), total.data_ptr(),
                                        _stream(stream)), "jp_plane_steps_tof_lm")
    return int(total.item())


def jp_fwd(xstart, xend, img, origin, voxsize, out=None, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty(l.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == l.n and out.is_contiguous()
    _check(load().jp_fwd(C.byref(l), img.data_ptr(), C.byref(g), out.data_ptr(), _stream(stream)), "jp_fwd")
    return out


def jp_back(xstart, xend, y, n, origin, voxsize, img=None, stream=None) -> torch.Tensor:
    """img += A^T y (a zero image is made when img is None)."""
    l, keep = make_lors(xstart, xend)
    _dev(y, torch.float32, "y")
    assert y.numel() == l.n and y.is_contiguous()
    if img is None:
        img = torch.zeros(tuple(int(x) for x in n), dtype=torch.float32, device=y.device)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back(C.byref(l), y.data_ptr(), C.byref(g), img.data_ptr(), _stream(stream)), "jp_back")
    return img


def jp_fwd_tof_sino(xstart, xend, img, origin, voxsize, tof: jp_tof, out=None, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty((l.n, tof.n_tofbins), dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == l.n * tof.n_tofbins and out.is_contiguous()
    _check(load().jp_fwd_tof_sino(C.byref(l), img.data_ptr(), C.byref(g), C.byref(tof), out.data_ptr(),
                                  _stream(stream)), "jp_fwd_tof_sino")
    return out


def jp_back_tof_sino(xstart, xend, y, n, origin, voxsize, tof: jp_tof, img=None, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    _dev(y, torch.float32, "y")
    assert y.numel() == l.n * tof.n_tofbins and y.is_contiguous()
    if img is None:
        img = torch.zeros(tuple(int(x) for x in n), dtype=torch.float32, device=y.device)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_tof_sino(C.byref(l), y.data_ptr(), C.byref(g), C.byref(tof), img.data_ptr(),
                                   _stream(stream)), "jp_back_tof_sino")
    return img


def _bins(tofbin, n):
    _dev(tofbin, torch.int16, "tofbin")
    assert tofbin.numel() == n and tofbin.is_contiguous()
    return tofbin


def jp_fwd_tof_lm(xstart, xend, tofbin, img, origin, voxsize, tof: jp_tof, out=None, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    tofbin = _bins(tofbin, l.n)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty(l.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == l.n and out.is_contiguous()
    _check(load().jp_fwd_tof_lm(C.byref(l), tofbin.data_ptr(), img.data_ptr(), C.byref(g), C.byref(tof),
                                out.data_ptr(), _stream(stream)), "jp_fwd_tof_lm")
    return out


def jp_back_tof_lm(xstart, xend, tofbin, y, n, origin, voxsize, tof: jp_tof, img=None, stream=None) -> torch.Tensor:
    l, keep = make_lors(xstart, xend)
    tofbin = _bins(tofbin, l.n)
    _dev(y, torch.float32, "y")
    assert y.numel() == l.n and y.is_contiguous()
    if img is None:
        img = torch.zeros(tuple(int(x) for x in n), dtype=torch.float32, device=y.device)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_tof_lm(C.byref(l), tofbin.data_ptr(), y.data_ptr(), C.byref(g), C.byref(tof),
                                 img.data_ptr(), _stream(stream)), "jp_back_tof_lm")
    return img


def jp_lm_osem_workspace_bytes(n_events: int, n, n_subsets: int) -> int:
    g = make_geom(n, (0, 0, 0), (1, 1, 1))
    return int(load().jp_lm_osem_workspace_bytes(int(n_events), C.byref(g), int(n_subsets)))


def jp_lm_osem(xstart, xend, tofbin, sens, img, origin, voxsize, tof: jp_tof, n_subsets: int, n_iter: int,
               workspace=None, stream=None) -> torch.Tensor:
    """Listmode OSEM in place on ``img`` (start image in, result out); returns img."""
    l, keep = make_lors(xstart, xend)
    tofbin = _bins(tofbin, l.n)
    img = _img(img)
    sens = _img(sens)
    assert sens.shape == img.shape
    g = make_geom(img.shape, origin, voxsize)
    need = jp_lm_osem_workspace_bytes(l.n, img.shape, n_subsets)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=img.device)
    assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= need
    _check(load().jp_lm_osem(C.byref(l), tofbin.data_ptr(), C.byref(g), C.byref(tof), sens.data_ptr(),
                             img.data_ptr(), int(n_subsets), int(n_iter), workspace.data_ptr(),
                             workspace.numel() * workspace.element_size(), _stream(stream)), "jp_lm_osem")
    return img


# ---- listmode plan (sorted events) ----------------------------------------------------------------------------
class LmPlan:
    """Owner of a jp_plan handle (the sort is done by jp_lm_plan_create; this class only holds the handle)."""

    def __init__(self, xstart, xend, tofbin, n, origin, voxsize, tof: jp_tof, n_subsets: int = 1, stream=None):
        l, keep = make_lors(xstart, xend)
        tofbin = _bins(tofbin, l.n)
        self.n = int(l.n)
        self.shape = tuple(int(x) for x in n)
        self.n_subsets = int(n_subsets)
        self.device = xstart.device
        g = make_geom(self.shape, origin, voxsize)
        h = C.c_void_p()
        _check(load().jp_lm_plan_create(C.byref(l), tofbin.data_ptr(), C.byref(g), C.byref(tof), int(n_subsets),
                                        _stream(stream), C.byref(h)), "jp_lm_plan_create")
        self.handle = h

    def subset_count(self, subset: int = -1) -> int:
        return int(load().jp_lm_plan_subset_count(self.handle, int(subset)))

    def set_path(self, path: int):
        """0: automatic, 1: line tiles, 2: quad image, 3: image bricks forward + float adjoint (jp_lm_plan_set_path)"""
        _check(load().jp_lm_plan_set_path(self.handle, int(path)), "jp_lm_plan_set_path")
        return self

    def destroy(self):
        if self.handle is not None and self.handle.value:
            _check(load().jp_lm_plan_destroy(self.handle), "jp_lm_plan_destroy")
        self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def jp_fwd_tof_lm_planned(plan: LmPlan, img, subset: int = -1, out=None, stream=None) -> torch.Tensor:
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    if out is None:
        out = torch.zeros(plan.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == plan.n and out.is_contiguous()
    _check(load().jp_fwd_tof_lm_planned(plan.handle, int(subset), img.data_ptr(), out.data_ptr(), _stream(stream)),
           "jp_fwd_tof_lm_planned")
    return out


def jp_back_tof_lm_planned(plan: LmPlan, y, subset: int = -1, img=None, stream=None) -> torch.Tensor:
    _dev(y, torch.float32, "y")
    assert y.numel() == plan.n and y.is_contiguous()
    if img is None:
        img = torch.zeros(plan.shape, dtype=torch.float32, device=y.device)
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    _check(load().jp_back_tof_lm_planned(plan.handle, int(subset), y.data_ptr(), img.data_ptr(), _stream(stream)),
           "jp_back_tof_lm_planned")
    return img


def jp_fwd_tof_lm_planned_sorted(plan: LmPlan, img, subset: int = -1, out=None, stream=None) -> torch.Tensor:
    """forward projection with the per-event results in PLAN order (see jp_lm_plan_permute)"""
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    if out is None:
        out = torch.zeros(plan.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == plan.n and out.is_contiguous()
    _check(load().jp_fwd_tof_lm_planned_sorted(plan.handle, int(subset), img.data_ptr(), out.data_ptr(), _stream(stream)),
           "jp_fwd_tof_lm_planned_sorted")
    return out


def jp_back_tof_lm_planned_sorted(plan: LmPlan, y_sorted, subset: int = -1, img=None, stream=None) -> torch.Tensor:
    _dev(y_sorted, torch.float32, "y_sorted")
    assert y_sorted.numel() == plan.n and y_sorted.is_contiguous()
    if img is None:
        img = torch.zeros(plan.shape, dtype=torch.float32, device=y_sorted.device)
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    _check(load().jp_back_tof_lm_planned_sorted(plan.handle, int(subset), y_sorted.data_ptr(), img.data_ptr(),
                                                _stream(stream)), "jp_back_tof_lm_planned_sorted")
    return img


def jp_lm_plan_permute(plan: LmPlan, values, to_plan_order: bool, out=None, stream=None) -> torch.Tensor:
    """per-event float32 values between caller order and plan order"""
    _dev(values, torch.float32, "values")
    assert values.numel() == plan.n and values.is_contiguous()
    if out is None:
        out = torch.empty_like(values)
    _check(load().jp_lm_plan_permute(plan.handle, values.data_ptr(), out.data_ptr(), 1 if to_plan_order else 0,
                                     _stream(stream)), "jp_lm_plan_permute")
    return out


def jp_fwd_lm_planned(plan: LmPlan, img, subset: int = -1, out=None, stream=None) -> torch.Tensor:
    """NON-TOF forward projection of the plan's events, results in caller order"""
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    if out is None:
        out = torch.zeros(plan.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == plan.n and out.is_contiguous()
    _check(load().jp_fwd_lm_planned(plan.handle, int(subset), img.data_ptr(), out.data_ptr(), _stream(stream)),
           "jp_fwd_lm_planned")
    return out


def jp_back_lm_planned(plan: LmPlan, y, subset: int = -1, img=None, stream=None) -> torch.Tensor:
    """NON-TOF back projection of per-event values over the plan's events; ACCUMULATES into img"""
    _dev(y, torch.float32, "y")
    assert y.numel() == plan.n and y.is_contiguous()
    if img is None:
        img = torch.zeros(plan.shape, dtype=torch.float32, device=y.device)
    img = _img(img)
    assert tuple(img.shape) == plan.shape
    _check(load().jp_back_lm_planned(plan.handle, int(subset), y.data_ptr(), img.data_ptr(), _stream(stream)),
           "jp_back_lm_planned")
    return img


def jp_lm_osem_planned(plan: LmPlan, sens, img, n_iter: int, workspace=None, stream=None) -> torch.Tensor:
    img = _img(img)
    sens = _img(sens)
    assert tuple(img.shape) == plan.shape and sens.shape == img.shape
    need = int(load().jp_lm_osem_planned_workspace_bytes(plan.handle))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=img.device)
    assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= need
    _check(load().jp_lm_osem_planned(plan.handle, sens.data_ptr(), img.data_ptr(), int(n_iter), workspace.data_ptr(),
                                     workspace.numel() * workspace.element_size(), _stream(stream)),
           "jp_lm_osem_planned")
    return img


def jp_lm_osem_planned_res(plan: LmPlan, sens, img, n_iter: int, res_sigma_mm: float, res_n_sigmas: float = 3.0,
                           workspace=None, stream=None) -> torch.Tensor:
    """listmode OSEM with the image-based resolution model in every subset"""
    img = _img(img)
    sens = _img(sens)
    assert tuple(img.shape) == plan.shape and sens.shape == img.shape
    need = int(load().jp_lm_osem_planned_workspace_bytes(plan.handle))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=img.device)
    assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= need
    _check(load().jp_lm_osem_planned_res(plan.handle, sens.data_ptr(), img.data_ptr(), int(n_iter), float(res_sigma_mm),
                                         float(res_n_sigmas), workspace.data_ptr(),
                                         workspace.numel() * workspace.element_size(), _stream(stream)),
           "jp_lm_osem_planned_res")
    return img


def jp_lm_osem_planned_backratio(plan: LmPlan, subset: int, x, out=None, workspace=None, stream=None) -> torch.Tensor:
    """b = A_m^T (1 / (A_m x)) over the plan's events of one subset (overwrites ``out``): the projection half of an
    OSEM subset update; sum b over the GPUs, then jp_osem_update."""
    x = _img(x)
    if out is None:
        out = torch.empty_like(x)
    out = _img(out)
    need = int(load().jp_lm_osem_planned_workspace_bytes(plan.handle))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=x.device)
    _check(load().jp_lm_osem_planned_backratio(plan.handle, int(subset), x.data_ptr(), out.data_ptr(),
                                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                               _stream(stream)), "jp_lm_osem_planned_backratio")
    return out


def jp_osem_update(x, b, sens, scale: float, voxsize=(1.0, 1.0, 1.0), stream=None) -> torch.Tensor:
    """x <- x b scale / sens where sens > 0, else 0; b <- 0.  In place; returns x."""
    x, b, sens = _img(x), _img(b), _img(sens)
    assert x.shape == b.shape == sens.shape
    g = make_geom(x.shape, (0.0, 0.0, 0.0), voxsize)
    _check(load().jp_osem_update(x.data_ptr(), b.data_ptr(), sens.data_ptr(), float(scale), C.byref(g),
                                 _stream(stream)), "jp_osem_update")
    return x


def jp_gauss3d(img, voxsize, sigma_mm: float, n_sigmas: float = 3.0, out=None, stream=None) -> torch.Tensor:
    """out = G img: the image-based resolution model (3-D Gaussian, zero boundary); out may be img"""
    img = _img(img)
    g = make_geom(img.shape, (0.0, 0.0, 0.0), voxsize)
    if out is None:
        out = torch.empty_like(img)
    _dev(out, torch.float32, "out")
    assert out.shape == img.shape and out.is_contiguous()
    _check(load().jp_gauss3d(img.data_ptr(), out.data_ptr(), C.byref(g), float(sigma_mm), float(n_sigmas),
                             _stream(stream)), "jp_gauss3d")
    return out


GAUSS3D_STATIC_MAX_VOXELS = 4194304   # JP_GAUSS3D_STATIC_MAX_VOXELS of joseph_b200.h


def jp_gauss3d_static(img, voxsize, sigma_mm: float, n_sigmas: float, out, stream=None) -> torch.Tensor:
    """out = G img like jp_gauss3d, for callers that cannot allocate device memory (all of it already handed out,
    an acquisition loop that may not stall on the allocator, no stream-ordered pool): the library's built-in
    16 MiB scratch serves as the intermediate image, so nothing is allocated -- which is also why `out` must be
    given here (it may be img).  Images above GAUSS3D_STATIC_MAX_VOXELS voxels raise JosephError.  All calls on a
    device share the scratch: keep them on one stream, or order them; overlapping calls race."""
    img = _img(img)
    g = make_geom(img.shape, (0.0, 0.0, 0.0), voxsize)
    _dev(out, torch.float32, "out")
    assert out.shape == img.shape and out.is_contiguous()
    _check(load().jp_gauss3d_static(img.data_ptr(), out.data_ptr(), C.byref(g), float(sigma_mm), float(n_sigmas),
                                    _stream(stream)), "jp_gauss3d_static")
    return out


# ---- hybrid mode: host tensors in and out -------------------------------------------------------
# ---- TOF sinogram OSEM (multiplicative factors + additive contamination) -----------------------------------------
def _offsets(subset_offsets):
    off = (C.c_int64 * len(subset_offsets))(*[int(o) for o in subset_offsets])
    return off, len(subset_offsets) - 1


def _opt(t, numel, what):
    if t is None:
        return None
    _dev(t, torch.float32, what)
    assert t.numel() == numel and t.is_contiguous(), what
    return t.data_ptr()


def jp_sino_osem_tof_workspace_bytes(subset_offsets, n: int, tof: jp_tof) -> int:
    off, ns = _offsets(subset_offsets)
    return int(load().jp_sino_osem_tof_workspace_bytes(off, ns, int(n), C.byref(tof)))


def jp_sino_sens_tof(xstart, xend, subset_offsets, mult, n, origin, voxsize, tof: jp_tof, out=None, workspace=None,
                     stream=None) -> torch.Tensor:
    """sens[m] = A_m^T (mult x 1_bins) for every subset: float32 [n_subsets, n0, n1, n2] (overwritten)"""
    l, keep = make_lors(xstart, xend)
    off, ns = _offsets(subset_offsets)
    shape = tuple(int(x) for x in n)
    if out is None:
        out = torch.empty((ns,) + shape, dtype=torch.float32, device=xstart.device)
    _dev(out, torch.float32, "sens")
    assert out.shape == (ns,) + shape and out.is_contiguous()
    g = make_geom(shape, origin, voxsize)
    wp, wb = (workspace.data_ptr(), workspace.numel() * workspace.element_size()) if workspace is not None else (None, 0)
    _check(load().jp_sino_sens_tof(C.byref(l), off, ns, _opt(mult, l.n, "mult"), C.byref(g), C.byref(tof),
                                   out.data_ptr(), wp, wb, _stream(stream)), "jp_sino_sens_tof")
    return out


def jp_sino_osem_tof(xstart, xend, subset_offsets, y, mult, contam, sens, img, origin, voxsize, tof: jp_tof,
                     n_iter: int, workspace=None, stream=None) -> torch.Tensor:
    """TOF sinogram OSEM in place on ``img`` (start image in, result out); returns img."""
    l, keep = make_lors(xstart, xend)
    off, ns = _offsets(subset_offsets)
    img = _img(img)
    _dev(sens, torch.float32, "sens")
    assert sens.shape == (ns,) + tuple(img.shape) and sens.is_contiguous()
    g = make_geom(img.shape, origin, voxsize)
    nb = int(tof.n_tofbins)
    need = int(load().jp_sino_osem_tof_workspace_bytes(off, ns, int(l.n), C.byref(tof)))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=img.device)
    assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= need
    _check(load().jp_sino_osem_tof(C.byref(l), off, ns, _opt(y, l.n * nb, "y"), _opt(mult, l.n, "mult"),
                                   _opt(contam, l.n * nb, "contam"), sens.data_ptr(), C.byref(g), C.byref(tof),
                                   img.data_ptr(), int(n_iter), workspace.data_ptr(),
                                   workspace.numel() * workspace.element_size(), _stream(stream)), "jp_sino_osem_tof")
    return img


# ---- sinogram plan (regular LOR lists: tracks with a common axial pattern) ---------------------------------------
class SinoPlan:
    """Owner of a jp_plan handle made by jp_sino_plan_create (the analysis runs in the library)."""

    def __init__(self, xstart, xend, stream=None):
        l, keep = make_lors(xstart, xend)
        self.device = xstart.device
        h = C.c_void_p()
        _check(load().jp_sino_plan_create(C.byref(l), _stream(stream), C.byref(h)), "jp_sino_plan_create")
        self.handle = h
        n, k, t = C.c_int64(), C.c_int64(), C.c_int32()
        _check(load().jp_sino_plan_info(h, C.byref(n), C.byref(k), C.byref(t)), "jp_sino_plan_info")
        self.n, self.n_tracks, self.track_length = int(n.value), int(k.value), int(t.value)

    @property
    def regular(self) -> bool:
        return self.track_length > 0

    def destroy(self):
        if self.handle is not None and self.handle.value:
            _check(load().jp_plan_destroy(self.handle), "jp_plan_destroy")
        self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def jp_fwd_planned(plan: SinoPlan, img, origin, voxsize, out=None, stream=None) -> torch.Tensor:
    """non-TOF forward projection of the plan's LORs (results in list order)"""
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty(plan.n, dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == plan.n and out.is_contiguous()
    _check(load().jp_fwd_planned(plan.handle, img.data_ptr(), C.byref(g), out.data_ptr(), _stream(stream)),
           "jp_fwd_planned")
    return out


def jp_back_planned(plan: SinoPlan, y, n, origin, voxsize, img=None, stream=None) -> torch.Tensor:
    """img += A^T y over the plan's LORs (a zero image is made when img is None)"""
    _dev(y, torch.float32, "y")
    assert y.numel() == plan.n and y.is_contiguous()
    if img is None:
        img = torch.zeros(tuple(int(x) for x in n), dtype=torch.float32, device=y.device)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_planned(plan.handle, y.data_ptr(), C.byref(g), img.data_ptr(), _stream(stream)),
           "jp_back_planned")
    return img


def jp_fwd_tof_sino_planned(plan: SinoPlan, img, origin, voxsize, tof: jp_tof, out=None, stream=None) -> torch.Tensor:
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty((plan.n, tof.n_tofbins), dtype=torch.float32, device=img.device)
    _dev(out, torch.float32, "out")
    assert out.numel() == plan.n * tof.n_tofbins and out.is_contiguous()
    _check(load().jp_fwd_tof_sino_planned(plan.handle, img.data_ptr(), C.byref(g), C.byref(tof), out.data_ptr(),
                                          _stream(stream)), "jp_fwd_tof_sino_planned")
    return out


def jp_back_tof_sino_planned(plan: SinoPlan, y, n, origin, voxsize, tof: jp_tof, img=None, stream=None) -> torch.Tensor:
    _dev(y, torch.float32, "y")
    assert y.numel() == plan.n * tof.n_tofbins and y.is_contiguous()
    if img is None:
        img = torch.zeros(tuple(int(x) for x in n), dtype=torch.float32, device=y.device)
    img = _img(img)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_tof_sino_planned(plan.handle, y.data_ptr(), C.byref(g), C.byref(tof), img.data_ptr(),
                                           _stream(stream)), "jp_back_tof_sino_planned")
    return img


def jp_sino_sens_tof_planned(plan: SinoPlan, subset_offsets, mult, n, origin, voxsize, tof: jp_tof, out=None,
                             workspace=None, stream=None) -> torch.Tensor:
    off, ns = _offsets(subset_offsets)
    shape = tuple(int(x) for x in n)
    if out is None:
        out = torch.empty((ns,) + shape, dtype=torch.float32, device=plan.device)
    _dev(out, torch.float32, "sens")
    assert out.shape == (ns,) + shape and out.is_contiguous()
    g = make_geom(shape, origin, voxsize)
    wp, wb = (workspace.data_ptr(), workspace.numel() * workspace.element_size()) if workspace is not None else (None, 0)
    _check(load().jp_sino_sens_tof_planned(plan.handle, off, ns, _opt(mult, plan.n, "mult"), C.byref(g), C.byref(tof),
                                           out.data_ptr(), wp, wb, _stream(stream)), "jp_sino_sens_tof_planned")
    return out


def jp_sino_osem_tof_planned(plan: SinoPlan, subset_offsets, y, mult, contam, sens, img, origin, voxsize, tof: jp_tof,
                             n_iter: int, workspace=None, stream=None) -> torch.Tensor:
    off, ns = _offsets(subset_offsets)
    img = _img(img)
    _dev(sens, torch.float32, "sens")
    assert sens.shape == (ns,) + tuple(img.shape) and sens.is_contiguous()
    g = make_geom(img.shape, origin, voxsize)
    nb = int(tof.n_tofbins)
    need = int(load().jp_sino_osem_tof_workspace_bytes(off, ns, int(plan.n), C.byref(tof)))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=img.device)
    assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= need
    _check(load().jp_sino_osem_tof_planned(plan.handle, off, ns, _opt(y, plan.n * nb, "y"), _opt(mult, plan.n, "mult"),
                                           _opt(contam, plan.n * nb, "contam"), sens.data_ptr(), C.byref(g),
                                           C.byref(tof), img.data_ptr(), int(n_iter), workspace.data_ptr(),
                                           workspace.numel() * workspace.element_size(), _stream(stream)),
           "jp_sino_osem_tof_planned")
    return img


def _host_lors(xstart: torch.Tensor, xend: torch.Tensor):
    for t in (xstart, xend):
        if t.is_cuda or t.dtype != torch.float32 or t.ndim != 2 or t.shape[0] != 3:
            raise JosephError("host end points must be CPU float32 tensors of shape (3, n)")
    rows = [t[a] if t[a].is_contiguous() else t[a].contiguous() for t in (xstart, xend) for a in range(3)]
    return jp_lors(*[r.data_ptr() for r in rows], int(xstart.shape[1])), rows


class Hybrid:
    """Owner of a jp_hybrid handle: host tensors in and out, the work split over the handle's devices.
    ``devices``: list of CUDA ordinals (None: all visible; an ordinal may repeat: several workers on one GPU)."""

    def __init__(self, devices=None):
        h = C.c_void_p()
        if devices is None:
            rc = load().jp_hybrid_create(None, 0, C.byref(h))
        else:
            arr = (C.c_int * len(devices))(*[int(d) for d in devices])
            rc = load().jp_hybrid_create(arr, len(devices), C.byref(h))
        _check(rc, "jp_hybrid_create")
        self.handle = h
        self.n = 0
        self.shape = None

    @property
    def workers(self) -> int:
        return int(load().jp_hybrid_worker_count(self.handle))

    def set_lors(self, xstart, xend, tofbin=None, n=None, origin=None, voxsize=None, tof: jp_tof = None):
        l, keep = _host_lors(xstart, xend)
        self.n = int(l.n)
        if tofbin is None:
            _check(load().jp_hybrid_set_lors(self.handle, C.byref(l), None, None, None), "jp_hybrid_set_lors")
        else:
            _host_bins(tofbin, l.n)
            self.shape = tuple(int(x) for x in n)
            g = make_geom(self.shape, origin, voxsize)
            _check(load().jp_hybrid_set_lors(self.handle, C.byref(l), tofbin.data_ptr(), C.byref(g), C.byref(tof)),
                   "jp_hybrid_set_lors")
        return self

    def fwd(self, img, origin, voxsize, out=None):
        img = _host_f32(img, "img")
        if out is None:
            out = torch.empty(self.n, dtype=torch.float32)
        _host_f32(out, "out", self.n)
        g = make_geom(img.shape, origin, voxsize)
        _check(load().jp_hybrid_fwd(self.handle, img.data_ptr(), C.byref(g), out.data_ptr()), "jp_hybrid_fwd")
        return out

    def back(self, y, img, origin, voxsize):
        _host_f32(y, "y", self.n)
        img = _host_f32(img, "img")
        g = make_geom(img.shape, origin, voxsize)
        _check(load().jp_hybrid_back(self.handle, y.data_ptr(), C.byref(g), img.data_ptr()), "jp_hybrid_back")
        return img

    def fwd_tof_sino(self, img, origin, voxsize, tof: jp_tof, out=None):
        img = _host_f32(img, "img")
        if out is None:
            out = torch.empty((self.n, int(tof.n_tofbins)), dtype=torch.float32)
        _host_f32(out, "out", self.n * int(tof.n_tofbins))
        g = make_geom(img.shape, origin, voxsize)
        _check(load().jp_hybrid_fwd_tof_sino(self.handle, img.data_ptr(), C.byref(g), C.byref(tof), out.data_ptr()),
               "jp_hybrid_fwd_tof_sino")
        return out

    def back_tof_sino(self, y, img, origin, voxsize, tof: jp_tof):
        _host_f32(y, "y", self.n * int(tof.n_tofbins))
        img = _host_f32(img, "img")
        g = make_geom(img.shape, origin, voxsize)
        _check(load().jp_hybrid_back_tof_sino(self.handle, y.data_ptr(), C.byref(g), C.byref(tof), img.data_ptr()),
               "jp_hybrid_back_tof_sino")
        return img

    def fwd_tof_lm(self, img, out=None):
        img = _host_f32(img, "img")
        assert tuple(img.shape) == self.shape
        if out is None:
            out = torch.empty(self.n, dtype=torch.float32)
        _host_f32(out, "out", self.n)
        _check(load().jp_hybrid_fwd_tof_lm(self.handle, img.data_ptr(), out.data_ptr()), "jp_hybrid_fwd_tof_lm")
        return out

    def back_tof_lm(self, y, img):
        _host_f32(y, "y", self.n)
        img = _host_f32(img, "img")
        assert tuple(img.shape) == self.shape
        _check(load().jp_hybrid_back_tof_lm(self.handle, y.data_ptr(), img.data_ptr()), "jp_hybrid_back_tof_lm")
        return img

    def destroy(self):
        if self.handle is not None and self.handle.value:
            _check(load().jp_hybrid_destroy(self.handle), "jp_hybrid_destroy")
        self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def jp_fwd_host(xstart, xend, img, origin, voxsize, out=None) -> torch.Tensor:
    """CPU tensors in, CPU tensor out; the projection itself runs on the current CUDA device."""
    l, keep = _host_lors(xstart, xend)
    if img.is_cuda or img.dtype != torch.float32 or not img.is_contiguous():
        raise JosephError("img must be a contiguous CPU float32 tensor")
    g = make_geom(img.shape, origin, voxsize)
    if out is None:
        out = torch.empty(l.n, dtype=torch.float32)
    assert not out.is_cuda and out.numel() == l.n and out.is_contiguous()
    _check(load().jp_fwd_host(C.byref(l), img.data_ptr(), C.byref(g), out.data_ptr()), "jp_fwd_host")
    return out


def jp_back_host(xstart, xend, y, img, origin, voxsize) -> torch.Tensor:
    """img (CPU, float32) += A^T y, computed on the current CUDA device."""
    l, keep = _host_lors(xstart, xend)
    if img.is_cuda or img.dtype != torch.float32 or not img.is_contiguous():
        raise JosephError("img must be a contiguous CPU float32 tensor")
    assert not y.is_cuda and y.dtype == torch.float32 and y.numel() == l.n and y.is_contiguous()
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_host(C.byref(l), y.data_ptr(), C.byref(g), img.data_ptr()), "jp_back_host")
    return img


def _host_f32(t, what, numel=None):
    if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise JosephError(f"{what} must be a contiguous CPU float32 tensor")
    if numel is not None and t.numel() != numel:
        raise JosephError(f"{what} has {t.numel()} elements, expected {numel}")
    return t


def _host_bins(tofbin, n):
    if tofbin.is_cuda or tofbin.dtype != torch.int16 or not tofbin.is_contiguous() or tofbin.numel() != n:
        raise JosephError("tofbin must be a contiguous CPU int16 tensor with one entry per event")
    return tofbin


def jp_fwd_tof_sino_host(xstart, xend, img, origin, voxsize, tof: jp_tof, out=None) -> torch.Tensor:
    l, keep = _host_lors(xstart, xend)
    img = _host_f32(img, "img")
    if out is None:
        out = torch.empty((l.n, int(tof.n_tofbins)), dtype=torch.float32)
    _host_f32(out, "out", l.n * int(tof.n_tofbins))
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_fwd_tof_sino_host(C.byref(l), img.data_ptr(), C.byref(g), C.byref(tof), out.data_ptr()),
           "jp_fwd_tof_sino_host")
    return out


def jp_back_tof_sino_host(xstart, xend, y, img, origin, voxsize, tof: jp_tof) -> torch.Tensor:
    l, keep = _host_lors(xstart, xend)
    _host_f32(y, "y", l.n * int(tof.n_tofbins))
    img = _host_f32(img, "img")
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_tof_sino_host(C.byref(l), y.data_ptr(), C.byref(g), C.byref(tof), img.data_ptr()),
           "jp_back_tof_sino_host")
    return img


def jp_fwd_tof_lm_host(xstart, xend, tofbin, img, origin, voxsize, tof: jp_tof, out=None) -> torch.Tensor:
    l, keep = _host_lors(xstart, xend)
    _host_bins(tofbin, l.n)
    img = _host_f32(img, "img")
    if out is None:
        out = torch.empty(l.n, dtype=torch.float32)
    _host_f32(out, "out", l.n)
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_fwd_tof_lm_host(C.byref(l), tofbin.data_ptr(), img.data_ptr(), C.byref(g), C.byref(tof),
                                     out.data_ptr()), "jp_fwd_tof_lm_host")
    return out


def jp_back_tof_lm_host(xstart, xend, tofbin, y, img, origin, voxsize, tof: jp_tof) -> torch.Tensor:
    l, keep = _host_lors(xstart, xend)
    _host_bins(tofbin, l.n)
    _host_f32(y, "y", l.n)
    img = _host_f32(img, "img")
    g = make_geom(img.shape, origin, voxsize)
    _check(load().jp_back_tof_lm_host(C.byref(l), tofbin.data_ptr(), y.data_ptr(), C.byref(g), C.byref(tof),
                                      img.data_ptr()), "jp_back_tof_lm_host")
    return img
