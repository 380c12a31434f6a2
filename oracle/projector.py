"""ctypes front end of oracle/cbct_oracle.c (fp64 P, P^T, Eq. 3) and oracle/siddon_oracle.c (the paper's Siddon
projector and its transpose).  TEST INFRASTRUCTURE ONLY.

`geom` is any object with the attributes nx, ny, nz, dx, dy, dz, ox, oy, oz, nu, nv,
du, dv, u0, v0, sad, sdd, angles (iterable of radians) and step (mm, > 0).
Arrays: volumes f[z][y][x], projections g[view][v][u], float64, C-contiguous.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build


class _Geom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("ox", C.c_double), ("oy", C.c_double), ("oz", C.c_double),
                ("nu", C.c_int32), ("nv", C.c_int32),
                ("du", C.c_double), ("dv", C.c_double), ("u0", C.c_double), ("v0", C.c_double),
                ("sad", C.c_double), ("sdd", C.c_double),
                ("n_views", C.c_int32), ("angles", C.POINTER(C.c_double)),
                ("step", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(os.path.abspath(path))
        dp, gp = C.POINTER(C.c_double), C.POINTER(_Geom)
        ip = C.POINTER(C.c_int64)
        L.orc_grid.argtypes = [gp, dp, dp, C.POINTER(C.c_int32)]
        L.orc_forward.argtypes = [gp, dp, dp]
        L.orc_forward_rays.argtypes = [gp, dp, C.c_long, ip, dp]
        L.orc_back_scatter.argtypes = [gp, dp, dp]
        L.orc_back_gather.argtypes = [gp, dp, dp]
        L.orc_back_gather_voxels.argtypes = [gp, dp, C.c_long, ip, dp]
        L.orc_back_eq3.argtypes = [gp, dp, dp]
        L.orc_sample_count.argtypes = [gp]
        L.orc_sample_count.restype = C.c_double
        L.orc_siddon_forward.argtypes = [gp, dp, dp]
        L.orc_siddon_back.argtypes = [gp, dp, dp]
        L.orc_siddon_nnz.argtypes = [gp, C.c_long, C.c_long]
        L.orc_siddon_nnz.restype = C.c_double
        L.orc_siddon_forward.restype = None
        L.orc_siddon_back.restype = None
        for fn in (L.orc_grid, L.orc_forward, L.orc_forward_rays, L.orc_back_scatter,
                   L.orc_back_gather, L.orc_back_gather_voxels, L.orc_back_eq3):
            fn.restype = None
        _lib = L
    return _lib


def _pack(geom):
    ang = np.ascontiguousarray(np.asarray(list(geom.angles), dtype=np.float64))
    g = _Geom(geom.nx, geom.ny, geom.nz, geom.dx, geom.dy, geom.dz, geom.ox, geom.oy, geom.oz,
              geom.nu, geom.nv, geom.du, geom.dv, geom.u0, geom.v0, geom.sad, geom.sdd,
              len(ang), ang.ctypes.data_as(C.POINTER(C.c_double)), float(geom.step))
    return g, ang  # keep `ang` alive with the struct


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _vol(geom, f):
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert f.shape == (geom.nz, geom.ny, geom.nx), f.shape
    return f


def _proj(geom, g):
    g = np.ascontiguousarray(g, dtype=np.float64)
    assert g.shape == (len(tuple(geom.angles)), geom.nv, geom.nu), g.shape
    return g


def grid(geom):
    """(R, t_min, K) of the global sample grid, SURVEY.md §8(c) c.2."""
    G, keep = _pack(geom)
    R, t0, K = C.c_double(), C.c_double(), C.c_int32()
    lib().orc_grid(C.byref(G), C.byref(R), C.byref(t0), C.byref(K))
    return R.value, t0.value, K.value


def forward(geom, f):
    """g = P f (Eq. 1, fixed-step trilinear reading)."""
    G, keep = _pack(geom)
    f = _vol(geom, f)
    g = np.empty((G.n_views, geom.nv, geom.nu), dtype=np.float64)
    lib().orc_forward(C.byref(G), _d(f), _d(g))
    return g


def forward_rays(geom, f, rays):
    """(P f)[rays] for flat ray indices (view*nv + iv)*nu + iu."""
    G, keep = _pack(geom)
    f = _vol(geom, f)
    rays = np.ascontiguousarray(rays, dtype=np.int64)
    out = np.empty(len(rays), dtype=np.float64)
    lib().orc_forward_rays(C.byref(G), _d(f), len(rays), rays.ctypes.data_as(C.POINTER(C.c_int64)), _d(out))
    return out


def back_scatter(geom, g):
    """f = P^T g, literal scatter transpose."""
    G, keep = _pack(geom)
    g = _proj(geom, g)
    f = np.empty((geom.nz, geom.ny, geom.nx), dtype=np.float64)
    lib().orc_back_scatter(C.byref(G), _d(g), _d(f))
    return f


def back_gather(geom, g):
    """f = P^T g, voxel-driven gather form."""
    G, keep = _pack(geom)
    g = _proj(geom, g)
    f = np.empty((geom.nz, geom.ny, geom.nx), dtype=np.float64)
    lib().orc_back_gather(C.byref(G), _d(g), _d(f))
    return f


def back_gather_voxels(geom, g, voxels):
    """(P^T g)[voxels] for flat voxel indices (iz*ny + iy)*nx + ix."""
    G, keep = _pack(geom)
    g = _proj(geom, g)
    voxels = np.ascontiguousarray(voxels, dtype=np.int64)
    out = np.empty(len(voxels), dtype=np.float64)
    lib().orc_back_gather_voxels(C.byref(G), _d(g), len(voxels),
                                 voxels.ctypes.data_as(C.POINTER(C.c_int64)), _d(out))
    return out


def back_eq3(geom, g):
    """The paper's approximate adjoint, Eq. 3 (pin only)."""
    G, keep = _pack(geom)
    g = _proj(geom, g)
    f = np.empty((geom.nz, geom.ny, geom.nx), dtype=np.float64)
    lib().orc_back_eq3(C.byref(G), _d(g), _d(f))
    return f


def sample_count(geom):
    """Algorithmic sample count: sum over rays of chord(padded box)/step."""
    G, keep = _pack(geom)
    return float(lib().orc_sample_count(C.byref(G)))


def siddon_forward(geom, f):
    """g = P_siddon f: exact radiological path through piecewise-constant voxels (Siddon 1985)."""
    G, keep = _pack(geom)
    f = _vol(geom, f)
    g = np.empty((G.n_views, geom.nv, geom.nu), dtype=np.float64)
    lib().orc_siddon_forward(C.byref(G), _d(f), _d(g))
    return g


def siddon_back(geom, g):
    """f = P_siddon^T g, literal ray-by-ray transpose."""
    G, keep = _pack(geom)
    g = _proj(geom, g)
    f = np.empty((geom.nz, geom.ny, geom.nx), dtype=np.float64)
    lib().orc_siddon_back(C.byref(G), _d(g), _d(f))
    return f


def siddon_nnz(geom, first=0, stride=1):
    """Number of (ray, voxel) pairs with positive intersection length over rays first, first+stride, ..."""
    G, keep = _pack(geom)
    return float(lib().orc_siddon_nnz(C.byref(G), int(first), int(stride)))
