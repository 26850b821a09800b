"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path (bench.py, tests -m gpu) and the oracle-side tests.  It holds
none of the projector's arithmetic: only the scanner / phantom / event models that make the inputs.
It stands in for the paper's GE Discovery MI sinograms and its NEMA listmode
acquisition, which are not available here.

Small tables (crystal positions, phantom spheres, config 0) are made with numpy ``default_rng`` in
float64 and cast to float32 at the end; the big index expansions (151.6 M sinogram LORs, 40 M events)
are plain torch tensor ops that run on the CPU or on ``cuda`` alike.  Event sampling uses a seeded
``torch.Generator`` of the target device, so an event list is reproducible per device type; parity
tests always hand the *same* arrays to both sides.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

BASE_SEED = 221212519

# ---- scanner of configs 1-4 (BASELINE.json configs[1]) -------------------------------------------
SCANNER_RADIUS = 400.0
N_RINGS = 48
RING_PITCH = 4.0
N_CRYSTALS = 512
N_RADIAL = 257          # r in [-128, 128]
N_VIEWS = 256
# ---- TOF (configs[2]) -----------------------------------------------------------------------------
TOF_BIN_WIDTH = 17.0
TOF_SIGMA = 13.6
TOF_NSIGMAS = 3.0
TOF_NBINS = 29


@dataclass
class Geometry:
    n: tuple
    voxsize: tuple
    origin: tuple = field(default=None)

    def __post_init__(self):
        if self.origin is None:  # "centred at the origin": o_a = -(n_a-1)/2 v_a
            self.origin = tuple(-(n - 1) / 2.0 * v for n, v in zip(self.n, self.voxsize))
        # the values both sides actually see are float32
        self.voxsize = tuple(float(np.float32(v)) for v in self.voxsize)
        self.origin = tuple(float(np.float32(o)) for o in self.origin)


@dataclass
class TofParams:
    tofbin_width: float = TOF_BIN_WIDTH
    sigma_tof: float = TOF_SIGMA
    n_sigmas: float = TOF_NSIGMAS
    n_tofbins: int = TOF_NBINS
    center_offset: float = 0.0

    def __post_init__(self):
        self.tofbin_width = float(np.float32(self.tofbin_width))
        self.sigma_tof = float(np.float32(self.sigma_tof))
        self.n_sigmas = float(np.float32(self.n_sigmas))
        self.center_offset = float(np.float32(self.center_offset))


GEOM_SMALL = Geometry((32, 32, 16), (4.0, 4.0, 4.0))
GEOM_SCANNER = Geometry((200, 200, 96), (2.0, 2.0, 2.0))


# ---- config 0 -------------------------------------------------------------------------------------
def config0(n_lors: int = 50_000, seed: int = BASE_SEED):
    """Random chords of a cylinder (r = 150 mm, |z| < 40 mm) through a 32x32x16 image of 4 mm voxels.

    Returns dict: xstart (3,n) f32, xend (3,n) f32, img (32,32,16) f32, y (n,) f32, geom."""
    rng = np.random.default_rng(seed)
    phi_s = rng.uniform(0.0, 2 * np.pi, n_lors)
    z_s = rng.uniform(-40.0, 40.0, n_lors)
    phi_e = rng.uniform(0.0, 2 * np.pi, n_lors)
    z_e = rng.uniform(-40.0, 40.0, n_lors)
    xs = np.stack([150.0 * np.cos(phi_s), 150.0 * np.sin(phi_s), z_s]).astype(np.float32)
    xe = np.stack([150.0 * np.cos(phi_e), 150.0 * np.sin(phi_e), z_e]).astype(np.float32)
    img = rng.uniform(0.0, 1.0, GEOM_SMALL.n).astype(np.float32)
    y = rng.uniform(0.0, 1.0, n_lors).astype(np.float32)
    return dict(xstart=xs, xend=xe, img=img, y=y, geom=GEOM_SMALL)


# ---- scanner tables -------------------------------------------------------------------------------
def crystal_table() -> np.ndarray:
    """(512, 48, 3) float32: crystal k of ring z at (400 cos(2 pi k/512), 400 sin(..), (z-23.5)*4)."""
    k = np.arange(N_CRYSTALS, dtype=np.float64)
    ang = 2.0 * np.pi * k / N_CRYSTALS
    z = (np.arange(N_RINGS, dtype=np.float64) - (N_RINGS - 1) / 2.0) * RING_PITCH
    tab = np.empty((N_CRYSTALS, N_RINGS, 3), dtype=np.float64)
    tab[:, :, 0] = (SCANNER_RADIUS * np.cos(ang))[:, None]
    tab[:, :, 1] = (SCANNER_RADIUS * np.sin(ang))[:, None]
    tab[:, :, 2] = z[None, :]
    return tab.astype(np.float32)


def phantom(seed: int = BASE_SEED + 1, geom: Geometry = GEOM_SCANNER) -> np.ndarray:
    """Uniform cylinder (r = 150 mm, value 1) plus 10 hot spheres (r = 10 mm, value 4), float32."""
    rng = np.random.default_rng(seed)
    centres = []
    while len(centres) < 10:
        c = rng.uniform([-140.0, -140.0, -86.0], [140.0, 140.0, 86.0])
        if c[0] ** 2 + c[1] ** 2 <= 140.0 ** 2:
            centres.append(c)
    ax = [geom.origin[a] + np.arange(geom.n[a], dtype=np.float64) * geom.voxsize[a] for a in range(3)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    img = np.zeros(geom.n, dtype=np.float32)
    img[X ** 2 + Y ** 2 <= 150.0 ** 2] = 1.0
    for c in centres:
        img[(X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2 <= 10.0 ** 2] = 4.0
    return img


# ---- sinogram LORs (configs 1, 2) -----------------------------------------------------------------
def sinogram_lors(views=None, radial=None, device="cpu"):
    """LOR endpoints of the sinogram in the order j = ((v*257 + (r+128))*48 + ring_a)*48 + ring_b.

    views: iterable of view indices (default all 256), radial: iterable of r in [-128,128]
    (default all 257).  start = crystal (v-r) mod 512 of ring_a, end = crystal (v+r+256) mod 512 of
    ring_b.  Returns xstart (3, n), xend (3, n) float32 torch tensors on ``device``."""
    views = torch.arange(N_VIEWS) if views is None else torch.as_tensor(list(views))
    radial = torch.arange(-128, 129) if radial is None else torch.as_tensor(list(radial))
    tab = torch.from_numpy(crystal_table()).to(device)          # (512, 48, 3)
    v = views.to(device).view(-1, 1)
    r = radial.to(device).view(1, -1)
    ca = torch.remainder(v - r, N_CRYSTALS).reshape(-1)          # (nv*nr,)
    cb = torch.remainder(v + r + N_CRYSTALS // 2, N_CRYSTALS).reshape(-1)
    nvr = ca.numel()
    n = nvr * N_RINGS * N_RINGS
    xs = torch.empty((3, n), dtype=torch.float32, device=device)
    xe = torch.empty((3, n), dtype=torch.float32, device=device)
    xs4 = xs.view(3, nvr, N_RINGS, N_RINGS)
    xe4 = xe.view(3, nvr, N_RINGS, N_RINGS)
    for a in range(3):
        xs4[a] = tab[ca, :, a].view(nvr, N_RINGS, 1)              # ring_a slow
        xe4[a] = tab[cb, :, a].view(nvr, 1, N_RINGS)              # ring_b fast
    return xs, xe


SUBSET_VIEWS = tuple(range(0, N_VIEWS, 16))   # config 2: every 16th view


# ---- listmode events (configs 3, 4) ---------------------------------------------------------------
def listmode_events(n_events: int = 40_000_000, seed: int = BASE_SEED + 3, device="cpu",
                    img: np.ndarray | None = None, geom: Geometry = GEOM_SCANNER,
                    chunk: int = 8_000_000):
    """Sample emission points from the phantom, isotropic directions, intersect with the cylinder,
    snap to crystal centres, derive an int16 TOF bin from the true position plus Gaussian noise.

    Returns xstart (3, n) f32, xend (3, n) f32, tofbin (n,) int16 -- generation (unsorted) order."""
    if img is None:
        img = phantom(geom=geom)
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    tab = torch.from_numpy(crystal_table()).to(dev)
    cdf = torch.cumsum(torch.from_numpy(img.astype(np.float64).ravel()).to(dev), 0)
    total = float(cdf[-1])
    n0, n1, n2 = geom.n
    o = torch.tensor(geom.origin, dtype=torch.float64, device=dev)
    vs = torch.tensor(geom.voxsize, dtype=torch.float64, device=dev)
    cos_max = 0.26  # larger axial tilts can never hit two rings of a 188 mm long, 800 mm wide scanner
    outs, outs_e, outs_b, have = [], [], [], 0
    while have < n_events:
        m = chunk
        u = torch.rand((8, m), dtype=torch.float64, device=dev, generator=gen)
        noise = torch.randn(m, dtype=torch.float64, device=dev, generator=gen)
        vox = torch.searchsorted(cdf, u[0] * total, right=True).clamp_(max=cdf.numel() - 1)
        i2 = vox % n2
        i1 = (vox // n2) % n1
        i0 = vox // (n1 * n2)
        idx = torch.stack([i0, i1, i2]).to(torch.float64)
        pos = o.view(3, 1) + (idx + u[1:4] - 0.5) * vs.view(3, 1)            # uniform in the voxel
        ct = (2.0 * u[4] - 1.0) * cos_max
        st = torch.sqrt(1.0 - ct * ct)
        az = 2.0 * math.pi * u[5]
        dirv = torch.stack([st * torch.cos(az), st * torch.sin(az), ct])
        # intersections with x^2 + y^2 = R^2: pos + lam*dir
        a = dirv[0] ** 2 + dirv[1] ** 2
        b = pos[0] * dirv[0] + pos[1] * dirv[1]
        c = pos[0] ** 2 + pos[1] ** 2 - SCANNER_RADIUS ** 2
        disc = torch.sqrt(b * b - a * c)
        lam_s = (-b - disc) / a
        lam_e = (-b + disc) / a
        ps = pos + lam_s * dirv
        pe = pos + lam_e * dirv
        ring_s = torch.floor(ps[2] / RING_PITCH + N_RINGS / 2.0).to(torch.int64)
        ring_e = torch.floor(pe[2] / RING_PITCH + N_RINGS / 2.0).to(torch.int64)
        ok = (ring_s >= 0) & (ring_s < N_RINGS) & (ring_e >= 0) & (ring_e < N_RINGS)
        sc = N_CRYSTALS / (2.0 * math.pi)
        cs = torch.remainder(torch.round(torch.atan2(ps[1], ps[0]) * sc).to(torch.int64), N_CRYSTALS)
        ce = torch.remainder(torch.round(torch.atan2(pe[1], pe[0]) * sc).to(torch.int64), N_CRYSTALS)
        ok &= ~((cs == ce) & (ring_s == ring_e))
        sel = torch.nonzero(ok).squeeze(1)
        xs = tab[cs[sel], ring_s[sel]]                                         # (k, 3) f32
        xe = tab[ce[sel], ring_e[sel]]
        xs64, xe64 = xs.to(torch.float64), xe.to(torch.float64)
        d = xe64 - xs64
        uhat = d / torch.linalg.norm(d, dim=1, keepdim=True)
        mid = 0.5 * (xs64 + xe64)
        tau = ((pos[:, sel].T - mid) * uhat).sum(1) + TOF_SIGMA * noise[sel]
        it = torch.floor(tau / TOF_BIN_WIDTH + 0.5).to(torch.int16)
        outs.append(xs.T.contiguous())
        outs_e.append(xe.T.contiguous())
        outs_b.append(it)
        have += int(sel.numel())
    xs = torch.cat(outs, 1)[:, :n_events].contiguous()
    xe = torch.cat(outs_e, 1)[:, :n_events].contiguous()
    tb = torch.cat(outs_b)[:n_events].contiguous()
    return xs, xe, tb


def uniform_values(n, lo: float, hi: float, seed: int, device="cpu") -> torch.Tensor:
    """Seeded U[lo, hi) float32 vector (back-projection inputs)."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    shape = (n,) if isinstance(n, int) else tuple(n)
    return torch.rand(shape, dtype=torch.float32, device=dev, generator=gen) * (hi - lo) + lo


# ---- multi-GPU sharding helper (LORs are independent units) ----------------
def shard_range(n: int, rank: int, world: int, align: int = 32):
    """Contiguous [lo, hi) slice of n LORs for ``rank`` of ``world``; boundaries aligned to ``align``."""
    per = -(-n // world)
    per = -(-per // align) * align
    lo = min(n, rank * per)
    hi = min(n, lo + per)
    return lo, hi
