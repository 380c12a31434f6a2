"""GPU parity of P and P^T against the fp64 oracle, through the C ABI (python -m pytest -m gpu).

Tolerances (BASELINE.json north_star): relative L2 <= 1e-5 per projection view and per backprojected
volume; adjoint identity <= 1e-5 in fp32.  SURVEY.md §8(c) item 29 defines the norm.
"""
import math
from dataclasses import replace

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import projector as op                      # noqa: E402
from paper_1008_2042_b200 import binding as cb          # noqa: E402
from paper_1008_2042_b200 import synthetic as syn       # noqa: E402

TOL = 1e-5


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def rel_l2_per_view(g, ref):
    num = np.sqrt(np.sum((g.astype(np.float64) - ref) ** 2, axis=(1, 2)))
    den = np.sqrt(np.sum(ref ** 2, axis=(1, 2)))
    scale = np.max(np.abs(ref))
    return np.max(np.where(den > 0, num / np.where(den > 0, den, 1.0), num / (scale if scale > 0 else 1.0)))


def rel_l2(a, ref):
    return float(np.linalg.norm(a.astype(np.float64).ravel() - ref.ravel()) / np.linalg.norm(ref.ravel()))


def gpu_forward(G, f):
    h = cb.Geometry(G)
    out = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
    h.forward(dev(f), out)
    torch.cuda.synchronize()
    return out.cpu().numpy(), h


def gpu_back(G, g):
    h = cb.Geometry(G)
    out = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
    h.backproject(dev(g), out)
    torch.cuda.synchronize()
    return out.cpu().numpy(), h


def require_fast_variants():
    """The packed instruction streams / skewed lane layout are product paths only on a device whose create-time self-check
    accepted them (geometry.cu: fast_variants_ok; cbct_geometry_describe reports a rejection).  Where it rejected them the
    library serves every handle with the plain variants, and the tests that FORCE the fast ones are skipped, loudly."""
    d = cb.Geometry(syn.workload(1).geometry).describe()
    if "rejected" in d:
        pytest.skip("fast kernel variants rejected by the create-time self-check on this device: " + d)


def test_default_kernels_are_reported():
    """which kernels serve the paper-size config on this device (cbct_geometry_describe); printed for the record"""
    h = cb.Geometry(syn.workload(4).geometry)
    d = h.describe()
    print("cfg 4:", d)
    assert "forward_tma_kernel<40,30," in d and "backproject_scatter_kernel<40," in d
    assert ("rejected" in d) == (",scalar>" in d.split(";")[0])


ODD = syn.Geometry(37, 29, 11, 2.0, 3.0, 5.0, 45, 19, 2.3, 3.1, 1000.0, 1500.0,
                   (0.0, 0.4, math.pi / 4, math.pi / 2, 2.0, math.pi, 4.0, 5.5), ox=3.0, oy=-4.0, oz=2.0, u0=1.7, v0=-2.9,
                   step_mm=0.7)


def test_geometry_info_matches_oracle_grid():
    for idx in (1, 2):
        G = syn.workload(idx).geometry
        h = cb.Geometry(G)
        R, t_min, K = op.grid(G)
        assert h.K == K and abs(h.t_min - t_min) < 1e-9 and abs(h.step_mm - G.step) < 1e-12
        assert h.n_vox == G.nx * G.ny * G.nz and h.n_rays == G.n_views * G.nv * G.nu
        assert abs(h.n_samples - op.sample_count(G)) <= 1e-9 * h.n_samples + 1
        assert h.workspace_bytes > 0


@pytest.mark.parametrize("cfg", [1, 2])
def test_forward_matches_oracle_full(cfg):
    w, ells, f0, _ = syn.make_inputs(cfg, noisy=False)
    g, h = gpu_forward(w.geometry, f0)
    ref = op.forward(w.geometry, f0.astype(np.float64))
    assert rel_l2_per_view(g, ref) <= TOL


def test_forward_packed_and_scalar_instruction_streams_agree(monkeypatch):
    """forward_tma_kernel has a packed-pair (FFMA2 / FADD2, default) and a scalar (CBCT_FW_PACKED=0) instruction stream;
    both perform the same IEEE operations in the same order: bit-identical projections, both within the bar."""
    require_fast_variants()
    w, _, f0, _ = syn.make_inputs(2, noisy=False)
    ref = op.forward(w.geometry, f0.astype(np.float64))
    out = {}
    for pk in ("1", "0"):
        monkeypatch.setenv("CBCT_FW_PACKED", pk)
        out[pk], _ = gpu_forward(w.geometry, f0)
        assert rel_l2_per_view(out[pk], ref) <= TOL, pk
    assert np.array_equal(out["0"], out["1"])


def test_forward_ragged_offset_geometry():
    f = syn.uniform_volume(ODD, 21)
    g, _ = gpu_forward(ODD, f)
    ref = op.forward(ODD, f.astype(np.float64))
    assert rel_l2_per_view(g, ref) <= TOL


def test_forward_global_kernel_and_oversized_tiles(monkeypatch):
    """The untiled kernel (CBCT_FORWARD_IMPL=global) and geometries whose pixel tiles do not fit the
    shared-memory box (fine voxels under coarse pixels) go through the same parity bar."""
    f = syn.uniform_volume(ODD, 23)
    ref = op.forward(ODD, f.astype(np.float64))
    for impl in ("global", "tiled"):
        monkeypatch.setenv("CBCT_FORWARD_IMPL", impl)
        g, _ = gpu_forward(ODD, f)
        assert rel_l2_per_view(g, ref) <= TOL, impl
        w1, _, f1, _ = syn.make_inputs(1, noisy=False)           # 4-divisible sizes: the same data the TMA path sees
        g1, _ = gpu_forward(w1.geometry, f1)
        assert rel_l2_per_view(g1, op.forward(w1.geometry, f1.astype(np.float64))) <= TOL, impl
    monkeypatch.delenv("CBCT_FORWARD_IMPL")
    for vox, pix in ((0.25, 3.0), (0.6, 2.0), (1.0, 1.2)):
        G = syn.Geometry(96, 80, 24, vox, vox, 2 * vox, 40, 12, pix, pix, 1000.0, 1500.0, (0.1, 0.9, 2.4, 3.9),
                         step_mm=0.8 * vox)
        f = syn.uniform_volume(G, 24)
        g, _ = gpu_forward(G, f)
        assert rel_l2_per_view(g, op.forward(G, f.astype(np.float64))) <= TOL, (vox, pix)


@pytest.mark.parametrize("cfg", [1, 2])
def test_backproject_matches_oracle_full(cfg):
    G = syn.workload(cfg).geometry
    y = syn.uniform_projections(G, 31)
    f, _ = gpu_back(G, y)
    ref = op.back_scatter(G, y.astype(np.float64))
    assert rel_l2(f, ref) <= TOL


def test_backproject_ragged_offset_geometry():
    y = syn.uniform_projections(ODD, 22) - 0.3
    f, _ = gpu_back(ODD, y)
    ref = op.back_scatter(ODD, y.astype(np.float64))
    assert rel_l2(f, ref) <= TOL


@pytest.mark.parametrize("cfg", [1, 2])
def test_adjoint_identity_fp32(cfg):
    """<P x, y> = <x, P^T y> to 1e-5 with U[0,1) vectors, inner products accumulated in fp64."""
    G = syn.workload(cfg).geometry
    x, y = syn.uniform_volume(G, 41), syn.uniform_projections(G, 41)
    Px, _ = gpu_forward(G, x)
    PTy, _ = gpu_back(G, y)
    lhs = float(np.sum(Px.astype(np.float64) * y))
    rhs = float(np.sum(x.astype(np.float64) * PTy))
    assert abs(lhs - rhs) <= TOL * abs(lhs)


def test_degenerate_inputs():
    G = syn.workload(1).geometry
    g, _ = gpu_forward(G, np.zeros(G.vol_shape, np.float32))
    assert np.all(g == 0.0)
    f, _ = gpu_back(G, np.zeros(G.proj_shape, np.float32))
    assert np.all(f == 0.0)
    # detector entirely beside the volume: every ray misses -> exact zeros, and P^T of anything is zero
    Gm = replace(G, u0=5000.0)
    g, _ = gpu_forward(Gm, syn.uniform_volume(Gm, 1))
    assert np.all(g == 0.0)
    f, _ = gpu_back(Gm, syn.uniform_projections(Gm, 1))
    assert np.all(f == 0.0)
    # single voxel, single pixel, single view
    G1 = syn.Geometry(1, 1, 1, 4.0, 4.0, 4.0, 1, 1, 1.0, 1.0, 1000.0, 1500.0, (0.3,))
    g, _ = gpu_forward(G1, np.ones((1, 1, 1), np.float32))
    ref = op.forward(G1, np.ones((1, 1, 1)))
    assert abs(g[0, 0, 0] - ref[0, 0, 0]) <= TOL * ref[0, 0, 0]
    f, _ = gpu_back(G1, np.ones((1, 1, 1), np.float32))
    assert abs(f[0, 0, 0] - op.back_scatter(G1, np.ones((1, 1, 1)))[0, 0, 0]) <= TOL * f[0, 0, 0]


def test_host_buffer_entry_points_match_device_ones():
    G = syn.workload(1).geometry
    h = cb.Geometry(G)
    x, y = syn.uniform_volume(G, 51), syn.uniform_projections(G, 51)
    hx, hy = torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()
    out_g = torch.empty(h.proj_shape, dtype=torch.float32).pin_memory()
    out_f = torch.empty(h.vol_shape, dtype=torch.float32).pin_memory()
    h.forward_host(hx, out_g)
    h.backproject_host(hy, out_f)
    torch.cuda.synchronize()
    g, _ = gpu_forward(G, x)
    f, _ = gpu_back(G, y)
    assert np.array_equal(out_g.numpy(), g) and np.array_equal(out_f.numpy(), f)


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_sampled_outputs(cfg):
    """BASELINE sizes in the launch configuration bench.py times (cfg 4) and the 360-view stress configuration (cfg 5,
    1024x768 detector: 2.4e11 samples per projector call, several int32 accumulation groups in P^T): oracle on sampled
    rays / voxels."""
    w = syn.workload(cfg)
    G = w.geometry
    f0 = syn.voxelise(G, syn.ellipsoids_for(w))
    g, h = gpu_forward(G, f0)
    rng = np.random.default_rng(cfg)
    rays = np.sort(rng.choice(h.n_rays, 4000, replace=False))
    ref = op.forward_rays(G, f0.astype(np.float64), rays)
    got = g.ravel()[rays].astype(np.float64)
    assert np.linalg.norm(got - ref) <= TOL * np.linalg.norm(ref)
    assert np.max(np.abs(got - ref)) <= 2e-5 * np.max(np.abs(ref))
    y = syn.uniform_projections(G, cfg)
    f, hb = gpu_back(G, y)
    vox = np.sort(rng.choice(h.n_vox, 300, replace=False))
    vox[:4] = [0, G.nx - 1, h.n_vox - G.nx, h.n_vox - 1]                 # the four extreme corners too
    refv = op.back_gather_voxels(G, y.astype(np.float64), vox)
    gotv = f.ravel()[vox].astype(np.float64)
    assert np.linalg.norm(gotv - refv) <= TOL * np.linalg.norm(refv)
    assert np.max(np.abs(gotv - refv)) <= 2e-5 * np.max(np.abs(refv))                 # per voxel, as for the rays above
    # no guard of the TMA kernels was triggered (bounded waits, box range checks, fixed-point head-room)
    assert h.status() == (True, []) and hb.status() == (True, [])
    # the input that loads the int32 accumulators most: all ones (P^T of it IS the weight sum the head-room plan bounds)
    ones = np.ones(G.proj_shape, np.float32)
    f1, h1 = gpu_back(G, ones)
    assert h1.status() == (True, []), "fixed-point head-room exhausted"
    sub = vox[::6]
    ref1 = op.back_gather_voxels(G, ones.astype(np.float64), sub)
    assert np.linalg.norm(f1.ravel()[sub] - ref1) <= TOL * np.linalg.norm(ref1)
    assert np.all(f1 >= 0.0)
    # property that holds at any size: adjoint identity
    x = syn.uniform_volume(G, cfg)
    Px, _ = gpu_forward(G, x)
    lhs = float(np.sum(Px.astype(np.float64) * y))
    rhs = float(np.sum(x.astype(np.float64) * f))
    assert abs(lhs - rhs) <= TOL * abs(lhs)


@pytest.mark.parametrize("impl,lanes", [
    ("scatter", "0"), ("scatter", "1"), ("cell", None), ("gather", None)])
def test_backproject_every_implementation_matches_oracle(monkeypatch, impl, lanes):
    """cbct_backproject has three kernels behind it: the TMA scatter kernel (default where the geometry allows,
    both lane layouts), the cell-driven kernel (fall-back) and the per-voxel gather kernel (cross-check).
    Each one, forced through CBCT_BACKPROJECT_IMPL, meets the same bar against the oracle; signed input."""
    if lanes == "0":
        require_fast_variants()
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", impl)
    if lanes is not None:
        monkeypatch.setenv("CBCT_BT_LANES", lanes)
        monkeypatch.setenv("CBCT_BT_PACKED", "1" if lanes == "0" else "0")      # the two shipped pairings
    for cfg in (1, 2):
        G = syn.workload(cfg).geometry
        y = syn.uniform_projections(G, 33 + cfg) - 0.4
        f, _ = gpu_back(G, y)
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, (impl, lanes, cfg)


def test_backproject_scatter_packed_and_scalar_streams(monkeypatch):
    """The scatter kernel's packed-pair instruction stream (FFMA2 / FADD2 / FMUL2, default) and the scalar one
    (CBCT_BT_PACKED=0) visit the same samples with the same positions; both meet the bar, and they agree with each other
    to the fixed-point unit (the weight products may round differently)."""
    require_fast_variants()
    G = syn.workload(2).geometry
    y = syn.uniform_projections(G, 36) - 0.4
    ref = op.back_scatter(G, y.astype(np.float64))
    out = {}
    for pk in ("1", "0"):
        monkeypatch.setenv("CBCT_BT_PACKED", pk)
        out[pk], _ = gpu_back(G, y)
        assert rel_l2(out[pk], ref) <= TOL, pk
    assert rel_l2(out["1"], out["0"].astype(np.float64)) <= 1e-6


def test_backproject_scatter_is_deterministic_and_scale_invariant():
    """The scatter kernel accumulates in fixed point relative to max|g|: the result is bit-identical from run
    to run (integer atomics are order-independent) and scales exactly with a power-of-two factor; a single
    hot pixel 100x above the rest keeps the volume within the bar (its error is relative to max|g|)."""
    G = syn.workload(2).geometry
    y = syn.uniform_projections(G, 35)
    f1, _ = gpu_back(G, y)
    f2, _ = gpu_back(G, y)
    assert np.array_equal(f1, f2)
    f4, _ = gpu_back(G, 4.0 * y)
    assert np.array_equal(f4, 4.0 * f1)
    y_hot = y.copy()
    y_hot[3, G.nv // 2, G.nu // 3] = 100.0
    f, _ = gpu_back(G, y_hot)
    assert rel_l2(f, op.back_scatter(G, y_hot.astype(np.float64))) <= TOL


def test_backproject_scatter_heavy_tailed_input_and_non_finite_input():
    """White noise with a heavy tail (40 rays at 20 .. 300 rms, both signs: the shape of a CGLS residual of low-count
    Poisson data).  The fixed-point unit follows T = min(max|g|, 8 rms(g)); rays above T are added by
    backproject_outlier_kernel with their own unit, so the usual bar holds.  Non-finite input gives a NaN volume."""
    for cfg in (1, 2):
        G = syn.workload(cfg).geometry
        rng = np.random.default_rng(37 + cfg)
        y = rng.standard_normal(G.proj_shape).astype(np.float32) * 0.05
        idx = rng.choice(y.size, 40, replace=False)
        y.ravel()[idx] = (rng.choice([-1.0, 1.0], 40) * 0.05 * np.geomspace(20.0, 300.0, 40)).astype(np.float32)
        f, h = gpu_back(G, y)
        assert h.status() == (True, [])
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, cfg
        f2, _ = gpu_back(G, y)
        assert np.array_equal(f, f2)
    G = syn.workload(1).geometry
    y = syn.uniform_projections(G, 39)
    for bad in (np.nan, np.inf):
        y[2, 5, 7] = bad
        f, _ = gpu_back(G, y)
        assert np.all(np.isnan(f))


def test_poisson_residual_backprojection_at_paper_size():
    """The input P^T actually sees inside CGLS at the paper-size config: the residual g - P f of Poisson data (5e4 photons
    per ray, max(I,1) floor) against the noiseless phantom -- noise with a heavy tail where the body is thick.  Oracle on
    sampled voxels (gather form), L2 and per-voxel bounds."""
    w, ells, f0, g = syn.make_inputs(4)
    G = w.geometry
    r = g - syn.analytic_projections(G, ells)
    f, h = gpu_back(G, r)
    assert h.status() == (True, [])
    rng = np.random.default_rng(4)
    vox = np.sort(rng.choice(h.n_vox, 300, replace=False))
    ref = op.back_gather_voxels(G, r.astype(np.float64), vox)
    got = f.ravel()[vox].astype(np.float64)
    assert np.linalg.norm(got - ref) <= TOL * np.linalg.norm(ref)
    assert np.max(np.abs(got - ref)) <= 5e-5 * np.max(np.abs(ref))


def test_backproject_scatter_headroom_bound():
    """The fixed-point plan assumes a bound on the sum of trilinear weights one voxel can receive; P^T of the
    all-ones projections IS that sum (times step), so it must stay below the planned head-room, and
    the all-ones result must still match the oracle (no wrap-around of the int32 accumulators)."""
    for cfg in (1, 2):
        G = syn.workload(cfg).geometry
        ones = np.ones(G.proj_shape, np.float32)
        f, h = gpu_back(G, ones)
        ref = op.back_scatter(G, ones.astype(np.float64))
        assert rel_l2(f, ref) <= TOL
        assert np.all(f >= 0.0)
        assert h.status() == (True, [])                                  # in particular: CBCT_STATUS_FIXED_POINT_RANGE not raised


def test_backproject_gather_kernel_cross_check(monkeypatch):
    """The per-voxel gather kernel (CBCT_BACKPROJECT_IMPL=gather) is kept as an in-library cross-check
    of the cell-driven kernel; both must meet the parity bar and agree with each other."""
    y = syn.uniform_projections(ODD, 25)
    ref = op.back_scatter(ODD, y.astype(np.float64))
    f_cell, _ = gpu_back(ODD, y)
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", "gather")
    f_gather, _ = gpu_back(ODD, y)
    monkeypatch.delenv("CBCT_BACKPROJECT_IMPL")
    assert rel_l2(f_cell, ref) <= TOL and rel_l2(f_gather, ref) <= TOL
    assert rel_l2(f_cell, f_gather.astype(np.float64)) <= TOL


def test_flat_cells_steep_rays():
    """Flat voxels under a tall detector (steep rays): exercises the z-clipped variant of the
    cell-driven backprojector and tall shared-memory boxes in the forward projector."""
    G = syn.Geometry(24, 20, 40, 4.0, 4.0, 0.5, 28, 64, 5.0, 8.0, 1000.0, 1500.0, (0.2, 1.3, 2.9, 4.1, 5.6),
                     oz=3.0, step_mm=0.4)
    y = syn.uniform_projections(G, 28) - 0.2
    f, _ = gpu_back(G, y)
    assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL
    x = syn.uniform_volume(G, 29)
    g, _ = gpu_forward(G, x)
    assert rel_l2_per_view(g, op.forward(G, x.astype(np.float64))) <= TOL


def test_backproject_axis_parallel_rays_and_fine_steps():
    """Rays exactly parallel to a grid axis (central pixel at 0 and 90 degrees, odd detector) and a
    sampling step much finer / coarser than the voxel."""
    for step in (0.05, 0.9, 3.7):
        G = syn.Geometry(20, 18, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi, 1.0),
                         step_mm=step)
        y = syn.uniform_projections(G, 26)
        f, _ = gpu_back(G, y)
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, step
        x = syn.uniform_volume(G, 27)
        g, _ = gpu_forward(G, x)
        assert rel_l2_per_view(g, op.forward(G, x.astype(np.float64))) <= TOL, step


def test_paper_eq3_backprojector_matches_oracle():
    """the paper's own approximate adjoint (Eq. 3) against the oracle's Eq. 3,
    including an offset, ragged geometry whose voxels project beside the imager (zero outside)."""
    for G, seed in ((syn.workload(1).geometry, 61), (syn.workload(2).geometry, 62), (ODD, 63)):
        y = syn.uniform_projections(G, seed)
        h = cb.Geometry(G)
        out = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
        h.backproject_eq3(dev(y), out)
        torch.cuda.synchronize()
        assert rel_l2(out.cpu().numpy(), op.back_eq3(G, y.astype(np.float64))) <= TOL


def _siddon(G, x, y):
    h = cb.Geometry(G)
    g = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
    f = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
    h.siddon_forward(dev(x), g)
    h.siddon_backproject(dev(y), f)
    f2 = torch.empty_like(f)
    h.siddon_backproject(dev(y), f2)
    torch.cuda.synchronize()
    assert torch.equal(f, f2)                                                  # integer accumulation: reproducible
    return g.cpu().numpy(), f.cpu().numpy()


def test_siddon_pair_matches_oracle():
    """the paper's own projector (Siddon's exact radiological path) and its exact
    transpose against the oracle's sort-all-crossings definition; same bar as the trilinear pair.  The axis-parallel case
    uses an odd grid (central rays through voxel centres); rays INSIDE a grid plane are covered by the next test."""
    AXIS = syn.Geometry(21, 19, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi, 1.0))
    for G, seed in ((syn.workload(1).geometry, 91), (syn.workload(2).geometry, 90), (ODD, 92), (AXIS, 94)):
        x, y = syn.uniform_volume(G, seed), syn.uniform_projections(G, seed) - 0.3
        g, f = _siddon(G, x, y)
        assert rel_l2_per_view(g, op.siddon_forward(G, x.astype(np.float64))) <= TOL
        assert rel_l2(f, op.siddon_back(G, y.astype(np.float64))) <= TOL
        lhs, rhs = float(np.sum(g.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * f))
        assert abs(lhs - rhs) <= TOL * abs(lhs)


def test_siddon_ray_inside_a_grid_plane_is_one_of_the_two_valid_answers():
    """Even grid, centred odd detector: the central column of rays of the 0 / 90 / 180 degree views lies IN a grid plane,
    where two answers are equally valid.  Every other ray matches the oracle; the in-plane rays must lie between the
    oracle's answers for the volume shifted by +-1e-6 mm across the plane."""
    G = syn.Geometry(20, 18, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi))
    x = syn.uniform_volume(G, 95)
    g, _ = _siddon(G, x, syn.uniform_projections(G, 95))
    g = g.astype(np.float64)
    ref = op.siddon_forward(G, x.astype(np.float64))
    lim = [op.siddon_forward(replace(G, ox=sx * 1e-6, oy=sy * 1e-6), x.astype(np.float64)) for sx in (-1, 1) for sy in (-1, 1)]
    lo, hi = np.min(lim, axis=0), np.max(lim, axis=0)
    in_plane = np.zeros(G.proj_shape, bool)
    in_plane[:, :, G.nu // 2] = True
    assert np.linalg.norm((g - ref)[~in_plane]) <= TOL * np.linalg.norm(ref[~in_plane])
    tol = 1e-5 * np.max(ref)
    assert np.all(g[in_plane] >= lo[in_plane] - tol) and np.all(g[in_plane] <= hi[in_plane] + tol)


def test_siddon_full_size_sampled_rays_and_adjoint():
    """Paper-size config in the launch configuration bench.py times: oracle on all rays of 2 views (Siddon has no
    per-ray entry point in the oracle; a 2-view geometry built from the same angles is the same rays), adjoint identity
    on the full 40 views."""
    w = syn.workload(4)
    G = w.geometry
    f0 = syn.voxelise(G, syn.ellipsoids_for(w))
    y = syn.uniform_projections(G, 4)
    g, f = _siddon(G, f0, y)
    sub = G.with_views([G.angles[3], G.angles[17]])
    ref = op.siddon_forward(sub, f0.astype(np.float64))
    assert rel_l2_per_view(g[[3, 17]], ref) <= TOL
    x = syn.uniform_volume(G, 4)
    gx, _ = _siddon(G, x, y)
    lhs, rhs = float(np.sum(gx.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * f))
    assert abs(lhs - rhs) <= TOL * abs(lhs)


def test_microbench_runs_and_reports():
    """cbct_microbench (SURVEY.md §8(d) denominators): every kind runs and returns a positive, finite rate; rates outside
    what an SM with 4 schedulers, 128 fp32 lanes and a 128-byte/clk shared-memory pipe can do are reported as warnings
    (they would mean the timed loop is not what it claims), not as failures of the parity suite."""
    import warnings
    r = cb.microbench()
    print("cbct_microbench:", {k: round(v[0], 3) for k, v in r.items()})
    for name, (rate, unit) in r.items():
        assert np.isfinite(rate) and rate > 0.0, (name, rate, unit)
    limits = {"ffma": (2.0, 4.2), "ffma2": (1.0, 4.2), "lds32": (0.5, 1.1), "atoms_add_s32": (0.3, 1.1), "atoms_add_u64": (0.0, 1.1),
              "ldg32_l1_hit": (0.2, 1.1), "l2_read_64MB": (2000.0, 40000.0), "l2_red_add_s32": (1.0, 1e4)}
    for name, (lo, hi) in limits.items():
        if not lo <= r[name][0] <= hi:
            warnings.warn(f"cbct_microbench {name} = {r[name][0]:.3g} {r[name][1]} outside the plausible range [{lo}, {hi}]")
