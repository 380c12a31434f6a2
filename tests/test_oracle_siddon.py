"""Pins for the Siddon oracle (oracle/siddon_oracle.c: the paper's own forward projector, and its
transpose) against what the paper and the mathematics fix.  None of these call the CUDA path.

SURVEY.md §8(f) NEXT-2; pins follow SURVEY.md §8(c) "P (5)": analytic chords and the non-zero count of PAPER.md:211.
"""
import math
import os

import numpy as np

from oracle import projector as op
from paper_1008_2042_b200 import synthetic as syn

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def ray_ends(G):
    """Source and pixel-centre positions of every ray, own arithmetic: S[view], D[view][iv][iu]."""
    S, D = [], []
    for th in G.angles:
        c, s = math.cos(th), math.sin(th)
        S.append(np.array([G.sad * c, G.sad * s, 0.0]))
        u = G.u0 + (np.arange(G.nu) - (G.nu - 1) / 2) * G.du
        v = G.v0 + (np.arange(G.nv) - (G.nv - 1) / 2) * G.dv
        uu, vv = np.meshgrid(u, v)
        D.append(np.stack([-(G.sdd - G.sad) * c - uu * s, -(G.sdd - G.sad) * s + uu * c, vv], axis=-1))
    return np.array(S), np.array(D)


def box_chords(G):
    """Length of every ray inside the volume box by the textbook slab method (no grid planes involved)."""
    S, D = ray_ends(G)
    lo = np.array([G.ox - G.nx * G.dx / 2, G.oy - G.ny * G.dy / 2, G.oz - G.nz * G.dz / 2])
    hi = np.array([G.ox + G.nx * G.dx / 2, G.oy + G.ny * G.dy / 2, G.oz + G.nz * G.dz / 2])
    d = D - S[:, None, None, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        t0 = (lo - S[:, None, None, :]) / d
        t1 = (hi - S[:, None, None, :]) / d
    tin = np.nanmax(np.minimum(t0, t1), axis=-1)
    tout = np.nanmin(np.maximum(t0, t1), axis=-1)
    tin, tout = np.maximum(tin, 0.0), np.minimum(tout, 1.0)
    return np.maximum(tout - tin, 0.0) * np.linalg.norm(d, axis=-1)


ODD = syn.Geometry(9, 7, 5, 3.0, 4.0, 6.0, 14, 9, 3.5, 4.5, 1000.0, 1500.0, (0.0, 0.7, math.pi / 2, 2.2, math.pi, 4.4, 5.9),
                   ox=2.0, oy=-3.0, oz=1.5, u0=1.2, v0=-2.1)


def test_uniform_volume_gives_the_box_chord_exactly():
    """f = 1: the voxel crossings of a ray tile its chord through the box, so g = chord to rounding; the central ray
    of a centred geometry at angle 0 runs along -x and must give nx*dx."""
    for G in (ODD, syn.workload(1).geometry):
        g = op.siddon_forward(G, np.ones(G.vol_shape))
        ref = box_chords(G)
        assert np.max(np.abs(g - ref)) <= 1e-10 * np.max(ref)
    Gc = syn.Geometry(8, 8, 4, 4.0, 4.0, 4.0, 13, 7, 6.0, 6.0, 1000.0, 1500.0, (0.0, math.pi / 2))
    g = op.siddon_forward(Gc, np.ones(Gc.vol_shape))
    assert abs(g[0, 3, 6] - 8 * 4.0) < 1e-10 and abs(g[1, 3, 6] - 8 * 4.0) < 1e-10


def test_path_lengths_against_dense_nearest_neighbour_sampling():
    """Independent route to the same integral: sample the ray every 2e-3 mm and look up the voxel that contains the
    sample (piecewise-constant model).  Converges to the exact path with error <= step * crossings."""
    G = ODD
    f = syn.uniform_volume(G, 3, np.float64)
    g = op.siddon_forward(G, f)
    S, D = ray_ends(G)
    lo = np.array([G.ox - G.nx * G.dx / 2, G.oy - G.ny * G.dy / 2, G.oz - G.nz * G.dz / 2])
    h = np.array([G.dx, G.dy, G.dz])
    n = np.array([G.nx, G.ny, G.nz])
    rng = np.random.default_rng(0)
    for _ in range(25):
        vi, iv, iu = rng.integers(G.n_views), rng.integers(G.nv), rng.integers(G.nu)
        d = D[vi, iv, iu] - S[vi]
        L = np.linalg.norm(d)
        m = int(L / 2e-3)
        a = (np.arange(m) + 0.5) / m
        p = S[vi][None, :] + a[:, None] * d[None, :]
        idx = np.floor((p - lo) / h).astype(int)
        ok = np.all((idx >= 0) & (idx < n), axis=1)
        est = f[idx[ok, 2], idx[ok, 1], idx[ok, 0]].sum() * (L / m)
        assert abs(est - g[vi, iv, iu]) <= 2e-3 * (G.nx + G.ny + G.nz) + 1e-9, (vi, iv, iu, est, g[vi, iv, iu])


def test_adjoint_identity_and_explicit_matrix():
    G = ODD
    x = syn.uniform_volume(G, 11, np.float64)
    y = syn.uniform_projections(G, 11, np.float64)
    lhs, rhs = np.sum(op.siddon_forward(G, x) * y), np.sum(x * op.siddon_back(G, y))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    # columns P e_j against rows P^T e_i on a tiny system
    Gt = syn.Geometry(4, 3, 2, 5.0, 5.0, 7.0, 5, 3, 6.0, 7.0, 1000.0, 1500.0, (0.3, 2.0))
    nvox, nray = 4 * 3 * 2, 2 * 3 * 5
    A = np.zeros((nray, nvox))
    for j in range(nvox):
        e = np.zeros(nvox)
        e[j] = 1.0
        A[:, j] = op.siddon_forward(Gt, e.reshape(Gt.vol_shape)).ravel()
    for i in range(nray):
        e = np.zeros(nray)
        e[i] = 1.0
        assert np.max(np.abs(op.siddon_back(Gt, e.reshape(Gt.proj_shape)).ravel() - A[i])) <= 1e-13
    assert np.all(A >= 0) and np.all(A.sum(axis=1) <= np.sqrt(20.0 ** 2 + 15.0 ** 2 + 14.0 ** 2) + 1e-9)


def test_sphere_chords_first_order_convergence():
    """A voxelised sphere converges to the analytic chords at first order in the voxel size (as the trilinear
    projector does); both discretisations agree with each other within that error."""
    centre, rad, rho = np.array([6.0, -4.0, 3.0]), 25.0, 0.05
    errs = []
    for vox in (4.0, 2.0, 1.0):
        n = int(round(96 / vox))
        G = syn.Geometry(n, n, n, vox, vox, vox, 48, 40, 2.4, 2.4, 1000.0, 1500.0, (0.3, 1.9, 4.0))
        ell = [syn.Ellipsoid(*centre, rad, rad, rad, rho)]
        f = syn.voxelise(G, ell, sub=4, dtype=np.float64)
        g = op.siddon_forward(G, f)
        ref = syn.analytic_projections(G, ell, dtype=np.float64)
        errs.append(np.linalg.norm(g - ref) / np.linalg.norm(ref))
        assert abs(g.sum() - ref.sum()) / ref.sum() < 0.01
    assert errs[0] / errs[1] >= 1.7 and errs[1] / errs[2] >= 1.7, errs
    assert errs[2] < 0.03, errs


def test_nonzeros_at_the_papers_geometry():
    """P "contains approximately 4 x 10^9 non-zero elements" for 512x512x70 voxels of 0.88x0.88x2.0 mm,
    a 512x384 imager over 40x30 cm and 40 views.  Counted on every 257th ray and scaled."""
    kv = {}
    for l in open(os.path.join(GOLD, "paper_constants.txt")):
        l = l.split("#")[0].split()
        if len(l) == 2:
            kv[l[0]] = float(l[1])
    G = syn.Geometry(512, 512, 70, 0.88, 0.88, 2.0, 512, 384, 400.0 / 512, 300.0 / 384, 1000.0, 1500.0, syn.full_circle(40))
    stride = 257
    nnz = op.siddon_nnz(G, 0, stride) * stride
    assert 0.75 * kv["siddon_nonzeros"] <= nnz <= 1.25 * kv["siddon_nonzeros"], nnz
