"""Seeded synthetic inputs (volumes and cone-beam geometries) for tests and bench.

This module is the ONLY code shared by the fp64 CPU oracle (``oracle/``) and the
CUDA path (``paper_1609_00958_b200.fp``).  It holds none of the projector's
arithmetic: it only draws ellipsoid phantoms and detector/source poses.

The five presets C1..C5 are the BASELINE.json configs.  They stand in for the
paper's benchmark workload (a cylinder inside a 512^3 fp32 box, 512^2 detector,
10 degree cone, 360 angles on a circular orbit whose rotation axis is parallel to
the fastest memory index -- PAPER.md:312-314 section 3.2, :326 Fig. 9), whose
actual data is not available.  Recipe: SURVEY.md section 8(d), restated in DESIGN.md.

Conventions:
  * volume array is C-order ``[nx][ny][nz]`` fp32, z fastest;
  * ``origin`` is the world position of the CENTRE of voxel (0,0,0);
    "centred at origin" means origin_a = -(N_a - 1)/2 * voxel_size;
  * a geometry row is 12 float64: source xyz, det_origin xyz (centre of pixel
    (0,0)), u-pitch vector xyz, v-pitch vector xyz, world units; pixel (iu, iv)
    centre is det_origin + iu*u + iv*v.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

SEED_BASE = 160900958  # arXiv id 1609.00958 as an integer


@dataclass(frozen=True)
class Config:
    name: str
    number: int
    n: Tuple[int, int, int]          # nx, ny, nz
    voxel_size: float
    n_ellipsoids: int
    semi_axes: Tuple[float, float]   # world units
    noise: str                       # "gauss" | "uniform"
    noise_amp: float                 # sigma, or half-width
    orbit: str                       # "circular" | "random"
    n_proj: int
    sid: float                       # source-to-isocentre
    sdd: float                       # source-to-detector
    nu: int
    nv: int
    pitch: float
    batch: Optional[int] = None      # projections per fp_project call (None = all)
    cylinder: bool = False           # zero the volume outside the inscribed cylinder about z

    @property
    def seed(self) -> int:
        return SEED_BASE + self.number

    @property
    def origin(self) -> Tuple[float, float, float]:
        return tuple(-(k - 1) / 2.0 * self.voxel_size for k in self.n)

    @property
    def half_extent(self) -> float:
        return max(self.n) * self.voxel_size / 2.0


CONFIGS = {
    "C1": Config("C1", 1, (32, 32, 32), 1.0, 8, (2.0, 10.0), "gauss", 0.01,
                 "circular", 16, 64.0, 128.0, 48, 48, 1.5),
    "C2": Config("C2", 2, (128, 128, 128), 1.0, 20, (4.0, 40.0), "uniform", 0.02,
                 "circular", 180, 256.0, 512.0, 192, 192, 1.5),
    "C3": Config("C3", 3, (512, 512, 512), 1.0, 40, (10.0, 160.0), "gauss", 0.01,
                 "circular", 360, 1000.0, 1500.0, 768, 768, 1.0),
    "C4": Config("C4", 4, (512, 512, 512), 1.0, 40, (10.0, 160.0), "gauss", 0.01,
                 "random", 256, 600.0, 900.0, 1024, 1024, 1.25),
    "C5": Config("C5", 5, (1024, 1024, 1024), 0.5, 60, (10.0, 150.0), "gauss", 0.01,
                 "circular", 720, 800.0, 1200.0, 1536, 1536, 0.6, batch=64),
    # Paper-shaped workload (SURVEY.md 8(f) #4; PAPER.md:312 sec. 3.2, :283 Eq. 17): 512^3 box, 512^2 detector,
    # 10 degree full cone, 360 angles, grid matched by Eq. 17 (voxel pitch 1): S = 256 / sin 5deg, D = S / 2,
    # detector pitch (S + D) tan 5deg / 256.  Not a BASELINE.json config; the volume is the C3 phantom (the
    # paper's data is not available) set to zero outside the inscribed cylinder about z, the paper's object shape.
    "P1": Config("P1", 6, (512, 512, 512), 1.0, 40, (10.0, 160.0), "gauss", 0.01,
                 "circular", 360, 2937.2705908915, 4405.9058863372, 512, 512, 1.5057297563, cylinder=True),
}


def scaled_config(cfg: Config, **kw) -> Config:
    """A copy of a preset with some fields replaced (ragged / edge-case tests)."""
    d = {f: getattr(cfg, f) for f in cfg.__dataclass_fields__}
    d.update(kw)
    return Config(**d)


# --------------------------------------------------------------------------- volumes

def ellipsoid_params(cfg: Config, rng: np.random.Generator):
    """Centres, semi-axes, rotations and values of the phantom's ellipsoids."""
    h = cfg.half_extent
    out = []
    for _ in range(cfg.n_ellipsoids):
        c = rng.uniform(-0.625 * h, 0.625 * h, size=3)
        a = rng.uniform(cfg.semi_axes[0], cfg.semi_axes[1], size=3)
        q, r = np.linalg.qr(rng.standard_normal((3, 3)))
        q = q * np.sign(np.diag(r))          # sign-fixed rotation/reflection
        val = rng.uniform(0.0, 1.0)
        out.append((c, a, q, val))
    return out


def make_volume(cfg: Config, device: str = "cpu"):
    """fp32 torch tensor (nx, ny, nz), contiguous, on ``device``.

    Ellipsoid parameters come from numpy's ``default_rng(cfg.seed)`` (identical on
    every machine); the indicator functions are rasterised with torch on
    ``device`` slab by slab; the noise comes from numpy on CPU (identical
    everywhere) or from a seeded torch generator on CUDA (fast; the same array is
    always handed to both the oracle and the CUDA path, so cross-device RNG
    equality is never relied on).
    """
    import torch

    rng = np.random.default_rng(cfg.seed)
    ells = ellipsoid_params(cfg, rng)
    nx, ny, nz = cfg.n
    dev = torch.device(device)
    dt = torch.float32
    ox, oy, oz = cfg.origin
    ys = (torch.arange(ny, device=dev, dtype=dt) * cfg.voxel_size + oy).view(1, ny, 1)
    zs = (torch.arange(nz, device=dev, dtype=dt) * cfg.voxel_size + oz).view(1, 1, nz)
    vol = torch.empty((nx, ny, nz), device=dev, dtype=dt)
    slab = max(1, min(nx, (1 << 24) // max(1, ny * nz)))
    for x0 in range(0, nx, slab):
        x1 = min(nx, x0 + slab)
        xs = (torch.arange(x0, x1, device=dev, dtype=dt) * cfg.voxel_size + ox).view(-1, 1, 1)
        acc = torch.zeros((x1 - x0, ny, nz), device=dev, dtype=dt)
        for (c, a, q, val) in ells:
            # local coordinates y = diag(1/a) * q^T (x - c)
            m = (q / a[None, :]).T            # rows: local axes scaled by 1/a
            dx, dy, dz = xs - float(c[0]), ys - float(c[1]), zs - float(c[2])
            r2 = torch.zeros_like(acc)
            for k in range(3):
                r2 += (float(m[k, 0]) * dx + float(m[k, 1]) * dy + float(m[k, 2]) * dz) ** 2
            acc += float(val) * (r2 <= 1.0).to(dt)
        vol[x0:x1] = acc
    if dev.type == "cpu":
        if cfg.noise == "gauss":
            noise = rng.standard_normal(size=cfg.n, dtype=np.float32) * np.float32(cfg.noise_amp)
        else:
            noise = rng.uniform(-cfg.noise_amp, cfg.noise_amp, size=cfg.n).astype(np.float32)
        vol += torch.from_numpy(noise)
    else:
        g = torch.Generator(device=dev)
        g.manual_seed(cfg.seed)
        for x0 in range(0, nx, slab):
            x1 = min(nx, x0 + slab)
            shape = (x1 - x0, ny, nz)
            if cfg.noise == "gauss":
                vol[x0:x1] += torch.randn(shape, generator=g, device=dev, dtype=dt) * cfg.noise_amp
            else:
                vol[x0:x1] += (torch.rand(shape, generator=g, device=dev, dtype=dt) * 2 - 1) * cfg.noise_amp
    if cfg.cylinder:
        ix = torch.arange(nx, device=dev, dtype=dt).view(nx, 1, 1) - 0.5 * (nx - 1)
        iy = torch.arange(ny, device=dev, dtype=dt).view(1, ny, 1) - 0.5 * (ny - 1)
        vol *= ((ix * ix + iy * iy) <= (0.5 * min(nx, ny)) ** 2).to(dt)
    return vol.contiguous()


# ------------------------------------------------------------------------ geometries

def circular_orbit(n_proj: int, sid: float, sdd: float, nu: int, nv: int, pitch: float,
                   angle_offset: float = 0.0) -> np.ndarray:
    """Circular cone-beam orbit about z (the fastest memory index).

    theta_k = 2 pi k / n_proj (+ offset); source S = sid (cos, sin, 0); flat detector
    perpendicular to the source-isocentre line at distance sdd from the source;
    u = pitch (-sin, cos, 0), v = pitch (0, 0, 1).
    """
    g = np.zeros((n_proj, 12), dtype=np.float64)
    for k in range(n_proj):
        th = 2.0 * math.pi * k / n_proj + angle_offset
        c, s = math.cos(th), math.sin(th)
        S = np.array([sid * c, sid * s, 0.0])
        C = S - sdd * np.array([c, s, 0.0])
        U = pitch * np.array([-s, c, 0.0])
        V = pitch * np.array([0.0, 0.0, 1.0])
        O = C - (nu - 1) / 2.0 * U - (nv - 1) / 2.0 * V
        g[k, 0:3], g[k, 3:6], g[k, 6:9], g[k, 9:12] = S, O, U, V
    return g


def random_poses(n_proj: int, sid: float, sdd: float, nu: int, nv: int, pitch: float,
                 rng: np.random.Generator) -> np.ndarray:
    """Source directions uniform on the sphere, detector perpendicular to the
    source-isocentre line with a random in-plane roll (BASELINE.json config 4)."""
    g = np.zeros((n_proj, 12), dtype=np.float64)
    for k in range(n_proj):
        nrm = rng.standard_normal(3)
        nrm /= np.linalg.norm(nrm)
        S = sid * nrm
        C = S - sdd * nrm
        ax = np.zeros(3)
        ax[int(np.argmin(np.abs(nrm)))] = 1.0
        e1 = np.cross(nrm, ax)
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(nrm, e1)
        phi = rng.uniform(0.0, 2.0 * math.pi)
        U = pitch * (math.cos(phi) * e1 + math.sin(phi) * e2)
        V = pitch * (-math.sin(phi) * e1 + math.cos(phi) * e2)
        O = C - (nu - 1) / 2.0 * U - (nv - 1) / 2.0 * V
        g[k, 0:3], g[k, 3:6], g[k, 6:9], g[k, 9:12] = S, O, U, V
    return g


def make_geometry(cfg: Config) -> np.ndarray:
    """float64 [n_proj][12] geometry rows of a preset."""
    if cfg.orbit == "circular":
        return circular_orbit(cfg.n_proj, cfg.sid, cfg.sdd, cfg.nu, cfg.nv, cfg.pitch)
    rng = np.random.default_rng(cfg.seed + 1000)
    return random_poses(cfg.n_proj, cfg.sid, cfg.sdd, cfg.nu, cfg.nv, cfg.pitch, rng)


def sample_rays(cfg: Config, n_rays: int, seed_offset: int = 2000) -> np.ndarray:
    """int32 [n_rays][3] = (projection, iv, iu) drawn uniformly (parity subsets)."""
    rng = np.random.default_rng(cfg.seed + seed_offset)
    ids = np.empty((n_rays, 3), dtype=np.int32)
    ids[:, 0] = rng.integers(0, cfg.n_proj, size=n_rays)
    ids[:, 1] = rng.integers(0, cfg.nv, size=n_rays)
    ids[:, 2] = rng.integers(0, cfg.nu, size=n_rays)
    return ids
