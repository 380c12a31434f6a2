"""Seeded synthetic inputs for the CBCT hot path (shared by tests, bench and smoke).

This module holds NO arithmetic of the method (no projector discretisation, no
CGLS, no tight frame, no multigrid).  It only builds the *inputs* that both the
fp64 oracle (`oracle/`) and the CUDA path are fed:

* the five workload geometries of BASELINE.json:configs,
* seeded additive-ellipsoid phantoms,
* the data model of a scanner: closed-form line integrals through those
  ellipsoids (textbook ray/quadric intersection; Eq. 1 evaluated
  analytically for a piecewise-constant object) and the Poisson noise recipe
  of SURVEY.md §8(c) item 27,
* seeded uniform test vectors.

These stand in for the NCAT phantom, the Catphan OBI scans and the patient
scan of PAPER.md:256, none of which exist in this container.

Geometry convention (Fig. 1 of the paper is missing):
world frame in mm, origin at the isocentre, z the rotation axis,
source x_S = (SAD cos th, SAD sin th, 0), detector centre
c_D = -(SDD-SAD)(cos th, sin th, 0), e_u = (-sin th, cos th, 0), e_v = (0,0,1).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 1008_2042  # seed = 1008_2042 + config index


@dataclass(frozen=True)
class Geometry:
    """Plain description of volume, detector and orbit (lengths mm, angles rad)."""

    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    nu: int
    nv: int
    du: float
    dv: float
    sad: float
    sdd: float
    angles: Tuple[float, ...]
    ox: float = 0.0
    oy: float = 0.0
    oz: float = 0.0
    u0: float = 0.0
    v0: float = 0.0
    step_mm: float = 0.0  # <= 0 -> 0.5 * min(dx, dy, dz)

    @property
    def n_views(self) -> int:
        return len(self.angles)

    @property
    def vol_shape(self) -> Tuple[int, int, int]:
        return (self.nz, self.ny, self.nx)  # f[z][y][x], x fastest

    @property
    def proj_shape(self) -> Tuple[int, int, int]:
        return (self.n_views, self.nv, self.nu)  # g[view][v][u], u fastest

    @property
    def step(self) -> float:
        return self.step_mm if self.step_mm > 0 else 0.5 * min(self.dx, self.dy, self.dz)

    def with_views(self, angles) -> "Geometry":
        return replace(self, angles=tuple(float(a) for a in angles))

    def coarsen_xy(self, factor: int = 2) -> "Geometry":
        """Same extent, voxel pitch x`factor` in x and y."""
        assert self.nx % factor == 0 and self.ny % factor == 0
        return replace(self, nx=self.nx // factor, ny=self.ny // factor,
                       dx=self.dx * factor, dy=self.dy * factor)


    def bin_detector(self, factor: int = 2) -> "Geometry":
        """Same detector extent and centre, pixel pitch x`factor` (detector binning at the
        coarse multigrid levels; block (i, j) of factor x factor pixels becomes one pixel at the block's centre)."""
        assert self.nu % factor == 0 and self.nv % factor == 0
        return replace(self, nu=self.nu // factor, nv=self.nv // factor, du=self.du * factor, dv=self.dv * factor)


def short_scan(n_views: int, arc_deg: float = 200.0, start_deg: float = -10.0) -> Tuple[float, ...]:
    """n views evenly over an arc, BOTH endpoints included (the scanner's "200 deg ... arcs"; SURVEY.md
    §8(f) NEXT-4).  The default arc, -10 deg .. 190 deg, is 180 deg + a 20 deg fan margin."""
    a0, arc = math.radians(start_deg), math.radians(arc_deg)
    return tuple(a0 + arc * k / (n_views - 1) for k in range(n_views))


def full_circle(n_views: int) -> Tuple[float, ...]:
    """theta_k = 2 pi k / n, endpoint excluded."""
    return tuple(2.0 * math.pi * k / n_views for k in range(n_views))


@dataclass(frozen=True)
class Ellipsoid:
    """Axis-aligned ellipsoid: centre (mm), semi-axes (mm), additive density (1/mm)."""

    cx: float
    cy: float
    cz: float
    ax: float
    ay: float
    az: float
    rho: float


@dataclass(frozen=True)
class Workload:
    name: str
    index: int            # 1-based config number of SURVEY.md §8
    geometry: Geometry
    n_ellipsoids: int
    kind: str             # "random" | "random+rods" | "torso"
    photons: Optional[float]  # N0 of the Poisson model, None = noiseless
    seed: int = field(default=0)


def workload(index: int) -> Workload:
    """The five configurations of BASELINE.json:configs (1-based)."""
    sad, sdd = 1000.0, 1500.0
    if index == 1:
        g = Geometry(64, 64, 16, 4.0, 4.0, 4.0, 96, 32, 3.2, 3.2, sad, sdd, full_circle(32))
        return Workload("tiny", 1, g, 6, "random", None, SEED_BASE + 1)
    if index == 2:
        g = Geometry(128, 128, 32, 2.0, 2.0, 5.0, 256, 96, 1.55, 1.55, sad, sdd, full_circle(40))
        return Workload("small", 2, g, 10, "random", 1e5, SEED_BASE + 2)
    if index == 3:
        g = Geometry(256, 256, 70, 1.0, 1.0, 2.5, 512, 384, 0.78, 0.78, sad, sdd, full_circle(40))
        return Workload("sweep", 3, g, 20, "random+rods", None, SEED_BASE + 3)
    if index == 4:
        g = Geometry(512, 512, 70, 0.5, 0.5, 2.5, 512, 384, 0.78, 0.78, sad, sdd, full_circle(40))
        return Workload("paper", 4, g, 0, "torso", 5e4, SEED_BASE + 4)
    if index == 5:
        g = Geometry(512, 512, 70, 0.5, 0.5, 2.5, 1024, 768, 0.39, 0.39, sad, sdd, full_circle(360))
        return Workload("stress", 5, g, 0, "torso", 1e4, SEED_BASE + 5)
    raise ValueError(f"no workload {index}")


# ----------------------------------------------------------------------------
# phantoms
# ----------------------------------------------------------------------------
def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def random_ellipsoids(geom: Geometry, n: int, seed: int, rho_lo: float, rho_hi: float) -> List[Ellipsoid]:
    """n ellipsoids: semi-axes U[8 %, 30 %] of the extent per axis, centres uniform
    such that the ellipsoid stays inside the volume, density U[rho_lo, rho_hi]."""
    rng = _rng(seed)
    ext = np.array([geom.nx * geom.dx, geom.ny * geom.dy, geom.nz * geom.dz])
    org = np.array([geom.ox, geom.oy, geom.oz])
    out = []
    for _ in range(n):
        semi = rng.uniform(0.08, 0.30, 3) * ext
        room = 0.5 * ext - semi
        c = org + rng.uniform(-1.0, 1.0, 3) * room
        rho = rng.uniform(rho_lo, rho_hi)
        out.append(Ellipsoid(*c.tolist(), *semi.tolist(), float(rho)))
    return out


def rod_ellipsoids(geom: Geometry, n: int, seed: int, rho: float) -> List[Ellipsoid]:
    """z-aligned high-contrast rods of 1 mm radius, modelled as prolate ellipsoids
    (semi-axes 1, 1, 0.45 * z-extent) so that their line integrals stay closed-form."""
    rng = _rng(seed + 7919)
    ext = np.array([geom.nx * geom.dx, geom.ny * geom.dy, geom.nz * geom.dz])
    out = []
    for _ in range(n):
        r = rng.uniform(0.1, 0.4) * min(ext[0], ext[1])
        phi = rng.uniform(0.0, 2.0 * math.pi)
        out.append(Ellipsoid(geom.ox + r * math.cos(phi), geom.oy + r * math.sin(phi), geom.oz,
                             1.0, 1.0, 0.45 * ext[2], rho))
    return out


def torso_ellipsoids(geom: Geometry) -> List[Ellipsoid]:
    """Torso-like nested ellipsoids (SURVEY.md §8(d) cfg 4): body 0.02/mm, two lung
    cavities at 0.005/mm (additive -0.015), spine and rib-like inserts at 0.05/mm
    (additive +0.03).  Sizes are fractions of the volume extent."""
    ex, ey, ez = geom.nx * geom.dx, geom.ny * geom.dy, geom.nz * geom.dz
    ox, oy, oz = geom.ox, geom.oy, geom.oz
    e = [Ellipsoid(ox, oy, oz, 0.46 * ex, 0.36 * ey, 0.60 * ez, 0.020)]
    for sgn in (-1.0, 1.0):
        e.append(Ellipsoid(ox + sgn * 0.20 * ex, oy + 0.02 * ey, oz, 0.14 * ex, 0.22 * ey, 0.42 * ez, -0.015))
    e.append(Ellipsoid(ox, oy - 0.24 * ey, oz, 0.045 * ex, 0.045 * ey, 0.55 * ez, 0.030))  # spine
    for k in range(6):  # rib-like inserts on an arc
        phi = math.pi * (0.15 + 0.14 * k)
        e.append(Ellipsoid(ox + 0.40 * ex * math.cos(phi), oy + 0.30 * ey * math.sin(phi), oz + (k - 2.5) * 0.05 * ez,
                           0.020 * ex, 0.020 * ey, 0.10 * ez, 0.030))
    e.append(Ellipsoid(ox + 0.05 * ex, oy + 0.08 * ey, oz, 0.08 * ex, 0.07 * ey, 0.25 * ez, 0.004))  # heart-like
    return e


def ellipsoids_for(w: Workload) -> List[Ellipsoid]:
    g = w.geometry
    if w.kind == "torso":
        return torso_ellipsoids(g)
    if w.index == 1:
        lo, hi = 0.01, 0.10        # 0.1 - 1.0 per cm (x0.1 -> per mm)
    else:
        lo, hi = 0.002, 0.020      # keeps max line integral ~ 5 so Poisson noise is meaningful
    ells = random_ellipsoids(g, w.n_ellipsoids, w.seed, lo, hi)
    if w.kind == "random+rods":
        ells += rod_ellipsoids(g, 8, w.seed, 2.0 * hi)
    return ells


def voxelise(geom: Geometry, ells: List[Ellipsoid], sub: int = 2, dtype=np.float32) -> np.ndarray:
    """Additive ellipsoids; voxel value = rho * (fraction of sub^3 sub-samples inside)
    (SURVEY.md §8(c) item 28).  Returns f[z][y][x]."""
    f = np.zeros(geom.vol_shape, dtype=np.float64)
    xs = geom.ox + (np.arange(geom.nx) - 0.5 * (geom.nx - 1)) * geom.dx
    ys = geom.oy + (np.arange(geom.ny) - 0.5 * (geom.ny - 1)) * geom.dy
    zs = geom.oz + (np.arange(geom.nz) - 0.5 * (geom.nz - 1)) * geom.dz
    offs = (np.arange(sub) + 0.5) / sub - 0.5
    for e in ells:
        ix = np.nonzero(np.abs(xs - e.cx) <= e.ax + geom.dx)[0]
        iy = np.nonzero(np.abs(ys - e.cy) <= e.ay + geom.dy)[0]
        iz = np.nonzero(np.abs(zs - e.cz) <= e.az + geom.dz)[0]
        if len(ix) == 0 or len(iy) == 0 or len(iz) == 0:
            continue
        frac = np.zeros((len(iz), len(iy), len(ix)))
        for oz_ in offs:
            qz = ((zs[iz] + oz_ * geom.dz - e.cz) / e.az) ** 2
            for oy_ in offs:
                qy = ((ys[iy] + oy_ * geom.dy - e.cy) / e.ay) ** 2
                for ox_ in offs:
                    qx = ((xs[ix] + ox_ * geom.dx - e.cx) / e.ax) ** 2
                    frac += (qz[:, None, None] + qy[None, :, None] + qx[None, None, :]) <= 1.0
        f[np.ix_(iz, iy, ix)] += e.rho * frac / sub ** 3
    return np.ascontiguousarray(f.astype(dtype))


# ----------------------------------------------------------------------------
# scanner data model: closed-form line integrals + Poisson noise
# ----------------------------------------------------------------------------
def ray_endpoints(geom: Geometry, view: int) -> Tuple[np.ndarray, np.ndarray]:
    """Source position (3,) and pixel centres (nv, nu, 3) of one view, convention c.1."""
    th = geom.angles[view]
    c, s = math.cos(th), math.sin(th)
    src = np.array([geom.sad * c, geom.sad * s, 0.0])
    u = geom.u0 + (np.arange(geom.nu) - 0.5 * (geom.nu - 1)) * geom.du
    v = geom.v0 + (np.arange(geom.nv) - 0.5 * (geom.nv - 1)) * geom.dv
    cd = -(geom.sdd - geom.sad) * np.array([c, s, 0.0])
    pix = (cd[None, None, :] + u[None, :, None] * np.array([-s, c, 0.0])[None, None, :]
           + v[:, None, None] * np.array([0.0, 0.0, 1.0])[None, None, :])
    return src, pix


def analytic_projections(geom: Geometry, ells: List[Ellipsoid], dtype=np.float32) -> np.ndarray:
    """Exact line integrals of the piecewise-constant ellipsoid object along every
    source->pixel-centre ray: sum_e rho_e * chord_e.  g[view][v][u]."""
    g = np.zeros(geom.proj_shape, dtype=np.float64)
    for view in range(geom.n_views):
        src, pix = ray_endpoints(geom, view)
        d = pix - src[None, None, :]
        d /= np.linalg.norm(d, axis=-1, keepdims=True)
        for e in ells:
            inv = 1.0 / np.array([e.ax, e.ay, e.az])
            o = (src - np.array([e.cx, e.cy, e.cz])) * inv
            n = d * inv[None, None, :]
            A = np.sum(n * n, axis=-1)
            B = n @ o
            C = float(o @ o) - 1.0
            disc = B * B - A * C
            g[view] += e.rho * 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A
    return np.ascontiguousarray(g.astype(dtype))


def add_poisson_noise(g: np.ndarray, photons: float, seed: int) -> np.ndarray:
    """I = Poisson(N0 exp(-g)); g_noisy = ln(N0 / max(I, 1))."""
    rng = _rng(seed + 104729)
    lam = photons * np.exp(-g.astype(np.float64))
    counts = rng.poisson(lam)
    return np.log(photons / np.maximum(counts, 1)).astype(g.dtype)


def uniform_volume(geom: Geometry, seed: int, dtype=np.float32) -> np.ndarray:
    return _rng(seed).random(geom.vol_shape).astype(dtype)


def uniform_projections(geom: Geometry, seed: int, dtype=np.float32) -> np.ndarray:
    return _rng(seed + 1).random(geom.proj_shape).astype(dtype)


def make_inputs(index: int, noisy: bool = True):
    """(workload, ellipsoids, phantom f0 fp32, projections g fp32) for config `index`.
    g is the scanner data model (analytic line integrals, plus Poisson noise when the
    config asks for it) -- it is never produced by either implementation under test."""
    w = workload(index)
    ells = ellipsoids_for(w)
    f0 = voxelise(w.geometry, ells)
    g = analytic_projections(w.geometry, ells)
    if noisy and w.photons is not None:
        g = add_poisson_noise(g, w.photons, w.seed)
    return w, ells, f0, g
