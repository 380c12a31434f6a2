"""Pins for the fp64 projector oracle (oracle/cbct_oracle.c) against what the paper and the
mathematics fix -- none of these call the CUDA path and none re-use oracle code.

PAPER.md:73 Eq. 1 (line integral), PAPER.md:211 (P^T is the transpose of P), Eq. 3 and
PAPER.md:506 ("numerical error less than 1%"); SURVEY.md §8(c) "What pins each part".
"""
import math

import numpy as np
import pytest

from oracle import projector as op
from paper_1008_2042_b200 import synthetic as syn


def small_geom(nx=8, ny=8, nz=4, d=4.0, nu=12, nv=6, du=6.0, n_views=6, **kw):
    return syn.Geometry(nx, ny, nz, d, d, kw.pop("dz", d), nu, nv, du, kw.pop("dv", du), 1000.0, 1500.0,
                        kw.pop("angles", syn.full_circle(n_views)), **kw)


# ---------------------------------------------------------------- grid
def test_global_grid_matches_survey_table():
    for idx, K in ((1, 187), (2, 401), (3, 809), (4, 1616), (5, 1616)):
        G = syn.workload(idx).geometry
        R, t_min, k = op.grid(G)
        assert k == K
        assert abs(t_min - (G.sad - R)) < 1e-12
        hx, hy, hz = (G.nx + 1) * G.dx / 2, (G.ny + 1) * G.dy / 2, (G.nz + 1) * G.dz / 2
        assert abs(R - math.sqrt(hx * hx + hy * hy + hz * hz)) < 1e-12


# ---------------------------------------------------------------- brute force on a tiny input
def dense_matrix_by_hats(G):
    """Independent construction of the system matrix: A[ray, voxel] = step * sum_k prod_axis
    max(0, 1 - |X_axis(t_k) - c_axis|), i.e. the hat-function form of trilinear interpolation,
    in vectorised numpy with its own geometry arithmetic."""
    R = math.sqrt(sum(((n + 1) * d / 2) ** 2 for n, d in ((G.nx, G.dx), (G.ny, G.dy), (G.nz, G.dz)))) \
        + math.sqrt(G.ox ** 2 + G.oy ** 2 + G.oz ** 2)
    step = G.step
    K = math.ceil(2 * R / step)
    t = (G.sad - R) + (np.arange(K) + 0.5) * step
    A = np.zeros((G.n_views * G.nv * G.nu, G.nz * G.ny * G.nx))
    cz, cy, cx = np.meshgrid(np.arange(G.nz), np.arange(G.ny), np.arange(G.nx), indexing="ij")
    cx, cy, cz = cx.ravel(), cy.ravel(), cz.ravel()
    row = 0
    for th in G.angles:
        c, s = math.cos(th), math.sin(th)
        src = np.array([G.sad * c, G.sad * s, 0.0])
        for iv in range(G.nv):
            for iu in range(G.nu):
                u = G.u0 + (iu - (G.nu - 1) / 2) * G.du
                v = G.v0 + (iv - (G.nv - 1) / 2) * G.dv
                det = np.array([-(G.sdd - G.sad) * c - u * s, -(G.sdd - G.sad) * s + u * c, v])
                n = (det - src) / np.linalg.norm(det - src)
                pts = src[None, :] + t[:, None] * n[None, :]
                X = (pts[:, 0] - G.ox) / G.dx + (G.nx - 1) / 2
                Y = (pts[:, 1] - G.oy) / G.dy + (G.ny - 1) / 2
                Z = (pts[:, 2] - G.oz) / G.dz + (G.nz - 1) / 2
                wx = np.maximum(0.0, 1.0 - np.abs(X[:, None] - cx[None, :]))
                wy = np.maximum(0.0, 1.0 - np.abs(Y[:, None] - cy[None, :]))
                wz = np.maximum(0.0, 1.0 - np.abs(Z[:, None] - cz[None, :]))
                A[row] = step * np.sum(wx * wy * wz, axis=0)
                row += 1
    return A


@pytest.fixture(scope="module")
def tiny():
    G = small_geom(8, 8, 4, 4.0, nu=10, nv=5, du=7.0, n_views=5, ox=1.5, oy=-2.0, oz=0.7, u0=0.9, v0=-1.1)
    return G, dense_matrix_by_hats(G)


def test_forward_equals_bruteforce_matrix(tiny):
    G, A = tiny
    rng = np.random.default_rng(1)
    f = rng.random(G.vol_shape)
    g = op.forward(G, f)
    ref = (A @ f.ravel()).reshape(G.proj_shape)
    assert np.max(np.abs(g - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_explicit_system_matrix_columns_vs_rows(tiny):
    """Columns P e_j against rows P^T e_i on 8x8x4 (north_star check 3)."""
    G, A = tiny
    n_vox, n_ray = A.shape[1], A.shape[0]
    cols = np.zeros_like(A)
    for j in range(0, n_vox, 7):  # every 7th unit volume (37 columns) through the C forward
        e = np.zeros(n_vox)
        e[j] = 1.0
        cols[:, j] = op.forward(G, e.reshape(G.vol_shape)).ravel()
        assert np.max(np.abs(cols[:, j] - A[:, j])) <= 1e-13
    for back in (op.back_scatter, op.back_gather):
        for i in range(0, n_ray, 11):  # every 11th unit projection through both transposes
            e = np.zeros(n_ray)
            e[i] = 1.0
            rowi = back(G, e.reshape(G.proj_shape)).ravel()
            assert np.max(np.abs(rowi - A[i, :])) <= 1e-13


def test_backprojectors_equal_matrix_transpose(tiny):
    G, A = tiny
    rng = np.random.default_rng(2)
    g = rng.random(G.proj_shape) - 0.25
    ref = (A.T @ g.ravel()).reshape(G.vol_shape)
    for back in (op.back_scatter, op.back_gather):
        out = back(G, g)
        assert np.max(np.abs(out - ref)) <= 1e-12 * np.max(np.abs(ref))
    vox = np.array([0, 5, 17, 100, G.nx * G.ny * G.nz - 1])
    assert np.allclose(op.back_gather_voxels(G, g, vox), ref.ravel()[vox], rtol=1e-12, atol=0)
    rays = np.array([0, 3, 49, 101, A.shape[0] - 1])
    f = rng.random(G.vol_shape)
    assert np.allclose(op.forward_rays(G, f, rays), (A @ f.ravel())[rays], rtol=1e-12, atol=0)


# ---------------------------------------------------------------- adjoint identity (north_star check 2)
@pytest.mark.parametrize("cfg", [1])
def test_adjoint_identity_1e12(cfg):
    G = syn.workload(cfg).geometry
    x = syn.uniform_volume(G, 11, np.float64)
    y = syn.uniform_projections(G, 11, np.float64)
    lhs = float(np.sum(op.forward(G, x) * y))
    for back in (op.back_scatter, op.back_gather):
        rhs = float(np.sum(x * back(G, y)))
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_scatter_equals_gather_anisotropic_offset():
    G = small_geom(12, 10, 6, 2.0, dz=5.0, nu=20, nv=9, du=2.2, dv=2.9, n_views=7, ox=3.0, oz=-2.0, v0=4.0,
                   step_mm=0.7)
    g = syn.uniform_projections(G, 5, np.float64)
    a, b = op.back_scatter(G, g), op.back_gather(G, g)
    assert np.max(np.abs(a - b)) <= 1e-13 * np.max(np.abs(a))


# ---------------------------------------------------------------- analytic chords (north_star check 1)
def analytic_chords(G, centre, semi):
    """Textbook ray/ellipsoid intersection, retyped here: o'=(o-c)/a, n'=n/a, A=n'.n', B=o'.n',
    C=o'.o'-1, chord = 2 sqrt(B^2 - A C)/A."""
    out = np.zeros(G.proj_shape)
    for vi, th in enumerate(G.angles):
        c, s = math.cos(th), math.sin(th)
        o = np.array([G.sad * c, G.sad * s, 0.0])
        for iv in range(G.nv):
            for iu in range(G.nu):
                u = G.u0 + (iu - (G.nu - 1) / 2) * G.du
                v = G.v0 + (iv - (G.nv - 1) / 2) * G.dv
                d = np.array([-(G.sdd - G.sad) * c - u * s, -(G.sdd - G.sad) * s + u * c, v]) - o
                n = d / np.linalg.norm(d)
                op_, np_ = (o - centre) / semi, n / semi
                A, B, Cc = np_ @ np_, op_ @ np_, op_ @ op_ - 1.0
                disc = B * B - A * Cc
                out[vi, iv, iu] = 2.0 * math.sqrt(disc) / A if disc > 0 else 0.0
    return out


def test_sphere_chords_first_order_convergence():
    """25 mm sphere at 4 -> 2 -> 1 mm voxels: rel-L2 falls >= 1.7x per halving; interior rays
    (chord > 80 % of the diameter) are within 2.5 % / 1.2 % / 0.6 % (SURVEY.md §8(c) pins, P (1))."""
    centre, rad, rho = np.array([6.0, -4.0, 3.0]), 25.0, 0.05
    errs = []
    for vox, interior_tol in ((4.0, 0.025), (2.0, 0.012), (1.0, 0.006)):
        n = int(round(96 / vox))
        G = syn.Geometry(n, n, n, vox, vox, vox, 48, 40, 2.4, 2.4, 1000.0, 1500.0, (0.3, 1.9, 4.0))
        ell = [syn.Ellipsoid(*centre, rad, rad, rad, rho)]
        f = syn.voxelise(G, ell, sub=4, dtype=np.float64)
        g = op.forward(G, f)
        ref = rho * analytic_chords(G, centre, np.array([rad, rad, rad]))
        errs.append(np.linalg.norm(g - ref) / np.linalg.norm(ref))
        inner = ref > 0.8 * 2 * rad * rho
        assert inner.sum() > 100
        assert np.max(np.abs(g[inner] - ref[inner]) / ref[inner]) < interior_tol
        assert abs(g.sum() - ref.sum()) / ref.sum() < 0.01          # summed mass
    assert errs[0] / errs[1] >= 1.7 and errs[1] / errs[2] >= 1.7, errs
    assert errs[2] < 0.03, errs


def test_ellipsoid_chords_and_generator_agree():
    """Anisotropic ellipsoid, anisotropic voxels; also checks synthetic.analytic_projections."""
    G = syn.Geometry(96, 96, 40, 1.0, 1.0, 2.5, 64, 48, 1.9, 1.9, 1000.0, 1500.0, (0.0, 0.8, 2.5, 4.4))
    e = syn.Ellipsoid(5.0, -7.0, 4.0, 30.0, 18.0, 25.0, 0.03)
    f = syn.voxelise(G, [e], sub=4, dtype=np.float64)
    g = op.forward(G, f)
    ref = e.rho * analytic_chords(G, np.array([e.cx, e.cy, e.cz]), np.array([e.ax, e.ay, e.az]))
    assert np.allclose(syn.analytic_projections(G, [e], np.float64), ref, rtol=1e-10, atol=1e-9)
    assert np.linalg.norm(g - ref) / np.linalg.norm(ref) < 0.05  # first order in the 2.5 mm voxel edge
    inner = ref > 0.8 * ref.max()
    assert np.max(np.abs(g[inner] - ref[inner]) / ref[inner]) < 0.01


def test_uniform_volume_central_ray_closed_form():
    """Uniform f=1, ray along -x through voxel-centre height: the zero-padded trilinear profile is a
    trapezoid of area nx*dx; the midpoint rule is exact on it up to the four kinks, O(step^2/dx)."""
    nx, dx = 20, 3.0
    G = syn.Geometry(nx, 9, 7, dx, 2.0, 2.5, 5, 3, 2.0, 2.0, 1000.0, 1500.0, (0.0, math.pi / 2), step_mm=0.25)
    g = op.forward(G, np.ones(G.vol_shape))
    assert abs(g[0, 1, 2] - nx * dx) < 4 * 0.25 ** 2 / dx
    # view at 90 deg travels along y: ny*dy
    assert abs(g[1, 1, 2] - 9 * 2.0) < 4 * 0.25 ** 2 / 2.0


def test_rotation_and_mirror_symmetry():
    """nx=ny, dx=dy, phantom invariant under 90 deg rotation => view th == view th+90 deg;
    z-mirror-symmetric phantom => g(u,v) == g(u,-v)."""
    G = syn.Geometry(16, 16, 6, 3.0, 3.0, 4.0, 24, 10, 3.1, 3.3, 1000.0, 1500.0,
                     (0.2, 0.2 + math.pi / 2, 0.2 + math.pi, 0.2 + 1.5 * math.pi))
    rng = np.random.default_rng(3)
    q = rng.random((6, 16, 16))
    q = q + q[::-1]                                   # z-mirror symmetric
    f = q + np.rot90(q, 1, (1, 2)) + np.rot90(q, 2, (1, 2)) + np.rot90(q, 3, (1, 2))  # C4 about z
    g = op.forward(G, f)
    for k in range(1, 4):
        assert np.max(np.abs(g[k] - g[0])) <= 1e-12 * np.max(np.abs(g[0]))
    assert np.max(np.abs(g - g[:, ::-1, :])) <= 1e-12 * np.max(np.abs(g))


def test_linearity_and_nonnegativity():
    G = small_geom(10, 9, 5, 3.0, nu=14, nv=7, du=4.0, n_views=4)
    rng = np.random.default_rng(4)
    a, b = rng.random(G.vol_shape), rng.random(G.vol_shape)
    ga, gb, gab = op.forward(G, a), op.forward(G, b), op.forward(G, 2.0 * a - 3.0 * b)
    assert np.max(np.abs(gab - (2.0 * ga - 3.0 * gb))) <= 1e-12 * np.max(np.abs(ga))
    assert ga.min() >= 0.0
    assert op.back_gather(G, np.abs(ga)).min() >= 0.0


# ---------------------------------------------------------------- the paper's Eq. 3
def test_eq3_agrees_with_exact_transpose_within_paper_bound():
    """On a smooth g the paper's analytic backprojector must agree with the exact transpose in the
    interior to about 1 % (PAPER.md:506 'numerical error less than 1%'; tolerance 2 %).  This pins the
    absolute scaling (step, voxel/pixel measures, magnification) and the geometry of P^T independently
    of the P code."""
    G = syn.workload(1).geometry
    vi, iv, iu = np.meshgrid(np.arange(G.n_views), np.arange(G.nv), np.arange(G.nu), indexing="ij")
    g = 1.0 + 0.3 * np.cos(2 * np.pi * iu / G.nu) * np.cos(2 * np.pi * iv / G.nv) + 0.1 * np.sin(2 * np.pi * vi / G.n_views)
    exact = op.back_gather(G, g)
    eq3 = op.back_eq3(G, g)
    inner = (slice(4, -4), slice(12, -12), slice(12, -12))
    rel = np.linalg.norm(exact[inner] - eq3[inner]) / np.linalg.norm(exact[inner])
    assert rel < 0.02, rel
    assert abs(np.mean(eq3[inner] / exact[inner]) - 1.0) < 0.005


# ---------------------------------------------------------------- sample count
def test_sample_count_closed_form_and_survey_value():
    # a single ray along -x through the box centre: chord of the padded box = (nx+1)*dx
    G = syn.Geometry(20, 9, 7, 3.0, 2.0, 2.5, 1, 1, 2.0, 2.0, 1000.0, 1500.0, (0.0,), step_mm=0.25)
    assert abs(op.sample_count(G) - 21 * 3.0 / 0.25) < 1e-9
    # 1.26e7 algorithmic samples at config 1
    assert abs(op.sample_count(syn.workload(1).geometry) / 1.26e7 - 1.0) < 0.01
