"""The projector KERNEL SOURCES executed on the host (tests/cpu_shim: one fiber per CUDA thread, guarded memory, TMA and
mbarrier emulation with the hardware's rules enforced) against the fp64 oracle -- `-m "not gpu"`.

This is not a parity claim (the `-m gpu` tests make that, on a B200, through the real library) and not a fallback
(the package never loads the shim).  It checks, without a GPU, what a device would punish with an illegal-address
fault, a hang or a wrong answer: indexing, box planning, alignment, barrier protocol, launch configuration.
The cases mirror tests/test_gpu_projectors.py at the sizes the host can run in seconds; tolerances are the same.
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from cpu_shim import shimlib as sl
from oracle import projector as op
from paper_1008_2042_b200 import synthetic as syn

TOL = 1e-5

ODD = syn.Geometry(37, 29, 11, 2.0, 3.0, 5.0, 45, 19, 2.3, 3.1, 1000.0, 1500.0,
                   (0.0, 0.4, math.pi / 4, math.pi / 2, 2.0, math.pi, 4.0, 5.5), ox=3.0, oy=-4.0, oz=2.0, u0=1.7, v0=-2.9,
                   step_mm=0.7)
# 4-divisible volume (the TMA kernels run), ragged detector (partial pixel tiles), offsets, all four view quadrants
# plus the 45-degree tie of the orientation rule
RAGGED_TMA = syn.Geometry(44, 36, 12, 2.0, 2.5, 4.0, 53, 27, 2.1, 2.9, 1000.0, 1500.0,
                          (0.0, 0.3, math.pi / 4, 1.2, math.pi / 2, 2.2, 3 * math.pi / 4, math.pi, 3.9, 5.0, 5.9),
                          ox=-3.0, oy=5.0, oz=1.5, u0=-2.2, v0=3.3, step_mm=0.9)


def rel_l2_per_view(g, ref):
    num = np.sqrt(np.sum((g.astype(np.float64) - ref) ** 2, axis=(1, 2)))
    den = np.sqrt(np.sum(ref ** 2, axis=(1, 2)))
    scale = np.max(np.abs(ref))
    return np.max(np.where(den > 0, num / np.where(den > 0, den, 1.0), num / (scale if scale > 0 else 1.0)))


def rel_l2(a, ref):
    return float(np.linalg.norm(a.astype(np.float64).ravel() - ref.ravel()) / np.linalg.norm(ref.ravel()))


def forward(G, f):
    return sl.Geometry(G).forward(f)


def back(G, y):
    return sl.Geometry(G).backproject(y)


@pytest.fixture(autouse=True)
def _clean_log():
    sl.kernel_log()
    yield
    sl.check(0, "end of test")


@pytest.mark.parametrize("tma_mode", ["eager", "lazy"])
def test_forward_tma_kernel(monkeypatch, tma_mode):
    """eager: a TMA copy lands the moment it is issued (a missing 'buffer free' barrier corrupts the sums);
    lazy: it lands when the mbarrier is first waited on (a missing wait reads poisoned memory)."""
    monkeypatch.setenv("SHIM_TMA", tma_mode)
    w, _, f0, _ = syn.make_inputs(1, noisy=False)
    g = forward(w.geometry, f0)
    assert any(k.startswith("cbct::forward_tma_kernel<") for k in sl.kernel_log())
    assert rel_l2_per_view(g, op.forward(w.geometry, f0.astype(np.float64))) <= TOL
    f = syn.uniform_volume(RAGGED_TMA, 71)
    g = forward(RAGGED_TMA, f)
    assert any(k.startswith("cbct::forward_tma_kernel<") for k in sl.kernel_log())
    assert rel_l2_per_view(g, op.forward(RAGGED_TMA, f.astype(np.float64))) <= TOL


def test_forward_tma_packed_and_scalar_streams_are_bit_identical(monkeypatch):
    """forward_tma_kernel<.., PK>: the FFMA2 / FADD2 instruction stream (default) and the scalar one (CBCT_FW_PACKED=0)
    perform the same IEEE operations in the same order."""
    out = {}
    for pk in ("1", "0"):
        monkeypatch.setenv("CBCT_FW_PACKED", pk)
        f = syn.uniform_volume(RAGGED_TMA, 73)
        out[pk] = forward(RAGGED_TMA, f)
        assert any(k.startswith("cbct::forward_tma_kernel<") and k.endswith("true>" if pk == "1" else "false>") for k in sl.kernel_log())
    assert np.array_equal(out["0"], out["1"])
    assert rel_l2_per_view(out["1"], op.forward(RAGGED_TMA, f.astype(np.float64))) <= TOL


@pytest.mark.parametrize("order", ["reverse", "random"])
@pytest.mark.parametrize("tma_mode", ["eager", "lazy"])
def test_tma_kernels_with_other_thread_orders(monkeypatch, tma_mode, order):
    """The shim normally resumes thread 0 of a block first, which would hide a consumer running ahead of the thread that
    plans the chunks and issues the TMA operations; here the highest thread index runs first, or the order changes
    (rotation and direction, seeded per block) between every two scheduling points."""
    monkeypatch.setenv("SHIM_ORDER", order)
    monkeypatch.setenv("SHIM_TMA", tma_mode)
    x, y = syn.uniform_volume(RAGGED_TMA, 74), syn.uniform_projections(RAGGED_TMA, 75) - 0.4
    g, f = forward(RAGGED_TMA, x), back(RAGGED_TMA, y)
    log = sl.kernel_log()
    assert any(k.startswith("cbct::forward_tma_kernel<") for k in log) and any(k.startswith("cbct::backproject_scatter_kernel<") for k in log)
    assert rel_l2_per_view(g, op.forward(RAGGED_TMA, x.astype(np.float64))) <= TOL
    assert rel_l2(f, op.back_scatter(RAGGED_TMA, y.astype(np.float64))) <= TOL


def test_forward_fallback_kernels(monkeypatch):
    f = syn.uniform_volume(ODD, 23)
    ref = op.forward(ODD, f.astype(np.float64))
    g = forward(ODD, f)                                   # nx, ny not divisible by 4: no tensor map
    assert "cbct::forward_tiled_kernel" in sl.kernel_log()
    assert rel_l2_per_view(g, ref) <= TOL
    for impl in ("global", "tiled"):
        monkeypatch.setenv("CBCT_FORWARD_IMPL", impl)
        g = forward(ODD, f)
        assert f"cbct::forward_{impl}_kernel" in sl.kernel_log()
        assert rel_l2_per_view(g, ref) <= TOL, impl
    monkeypatch.delenv("CBCT_FORWARD_IMPL")
    for vox, pix in ((0.25, 3.0), (0.6, 2.0), (1.0, 1.2)):    # pixel tiles that do not fit the shared-memory box
        G = syn.Geometry(96, 80, 24, vox, vox, 2 * vox, 40, 12, pix, pix, 1000.0, 1500.0, (0.1, 0.9, 2.4, 3.9),
                         step_mm=0.8 * vox)
        f = syn.uniform_volume(G, 24)
        assert rel_l2_per_view(forward(G, f), op.forward(G, f.astype(np.float64))) <= TOL, (vox, pix)


@pytest.mark.parametrize("packed", ["1", "0"])
@pytest.mark.parametrize("lanes", ["0", "1"])
@pytest.mark.parametrize("tma_mode", ["eager", "lazy"])
def test_backproject_scatter_kernel(monkeypatch, lanes, tma_mode, packed):
    """both lane layouts and both instruction streams (packed pairs / scalar) of the TMA scatter kernel; signed input;
    lazy = tensor reductions read their shared-memory box only at cp.async.bulk.wait_group (clearing the box too early
    loses the contributions)."""
    monkeypatch.setenv("SHIM_TMA", tma_mode)
    monkeypatch.setenv("CBCT_BT_LANES", lanes)
    monkeypatch.setenv("CBCT_BT_PACKED", packed)
    for G, seed in ((syn.workload(1).geometry, 34), (RAGGED_TMA, 72)):
        y = syn.uniform_projections(G, seed) - 0.4
        f = back(G, y)
        want = f", {lanes}, {'true' if packed == '1' else 'false'}>"
        assert any(k.startswith("cbct::backproject_scatter_kernel<") and k.endswith(want) for k in sl.kernel_log())
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, (lanes, tma_mode, packed)


@pytest.mark.parametrize("impl", ["cell", "gather"])
def test_backproject_voxel_driven_kernels(monkeypatch, impl):
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", impl)
    for G, seed in ((syn.workload(1).geometry, 34), (ODD, 25)):
        y = syn.uniform_projections(G, seed) - 0.4
        f = back(G, y)
        assert any(k.startswith(f"cbct::backproject_{impl}_kernel") for k in sl.kernel_log())
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, impl


def test_backproject_default_dispatch_and_adjoint_identity():
    G = syn.workload(1).geometry
    x, y = syn.uniform_volume(G, 41), syn.uniform_projections(G, 41)
    Px, PTy = forward(G, x), back(G, y)
    log = sl.kernel_log()
    assert any(k.startswith("cbct::backproject_scatter_kernel<") for k in log)      # the default where the geometry allows
    lhs, rhs = float(np.sum(Px.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * PTy))
    assert abs(lhs - rhs) <= TOL * abs(lhs)
    y = syn.uniform_projections(ODD, 22) - 0.3                                     # no tensor map: the cell kernel
    f = back(ODD, y)
    assert any(k.startswith("cbct::backproject_cell_kernel<") for k in sl.kernel_log())
    assert rel_l2(f, op.back_scatter(ODD, y.astype(np.float64))) <= TOL


def test_backproject_scatter_fixed_point_properties():
    G = syn.workload(1).geometry
    y = syn.uniform_projections(G, 35)
    f1, f2 = back(G, y), back(G, y)
    assert np.array_equal(f1, f2)                                        # integer accumulation: order independent
    assert np.array_equal(back(G, 4.0 * y), 4.0 * f1)                    # scaled by max|g|: exact for powers of two
    y_hot = y.copy()
    y_hot[3, G.nv // 2, G.nu // 3] = 100.0
    assert rel_l2(back(G, y_hot), op.back_scatter(G, y_hot.astype(np.float64))) <= TOL
    ones = np.ones(G.proj_shape, np.float32)                            # the weight sum the head-room plan bounds
    f = back(G, ones)
    assert rel_l2(f, op.back_scatter(G, ones.astype(np.float64))) <= TOL and np.all(f >= 0.0)


def heavy_tailed_projections(G, seed):
    """white noise (the hardest input for a fixed-point P^T: the result is small by cancellation) with a heavy tail:
    a few dozen rays 20 .. 300 times the rms, both signs -- the shape of a CGLS residual of low-count Poisson data"""
    rng = np.random.default_rng(seed)
    y = rng.standard_normal(G.proj_shape).astype(np.float32) * 0.05
    idx = rng.choice(y.size, 40, replace=False)
    y.ravel()[idx] = (rng.choice([-1.0, 1.0], 40) * 0.05 * np.geomspace(20.0, 300.0, 40)).astype(np.float32)
    return y


@pytest.mark.parametrize("lanes,packed", [("1", "0"), ("0", "1")])
def test_backproject_scatter_heavy_tailed_input(monkeypatch, lanes, packed):
    """The fixed-point unit follows T = min(max|g|, 8 rms(g)), not the single largest value: rays above T are added by
    backproject_outlier_kernel with their own unit.  Against the oracle at the usual bar (a unit tied to max|g|, 300 rms
    here, would be 37 times coarser for every ray)."""
    monkeypatch.setenv("CBCT_BT_LANES", lanes)
    monkeypatch.setenv("CBCT_BT_PACKED", packed)
    for G, seed in ((syn.workload(1).geometry, 37), (RAGGED_TMA, 38)):
        y = heavy_tailed_projections(G, seed)
        f = back(G, y)
        log = sl.kernel_log()
        assert "cbct::backproject_outlier_kernel" in log and any(k.startswith("cbct::backproject_scatter_kernel<") for k in log)
        assert rel_l2(f, op.back_scatter(G, y.astype(np.float64))) <= TOL, (lanes, packed, G.nx)
        assert np.array_equal(f, back(G, y))                                  # still integer sums: reproducible
    # non-finite input is not laundered into finite numbers: the volume is NaN
    G = syn.workload(1).geometry
    y = syn.uniform_projections(G, 39)
    y[2, 5, 7] = np.nan
    assert np.all(np.isnan(back(G, y)))
    y[2, 5, 7] = np.inf
    assert np.all(np.isnan(back(G, y)))


def test_degenerate_inputs():
    G = syn.workload(1).geometry
    assert np.all(forward(G, np.zeros(G.vol_shape, np.float32)) == 0.0)
    assert np.all(back(G, np.zeros(G.proj_shape, np.float32)) == 0.0)
    Gm = replace(G, u0=5000.0)                                           # every ray misses the volume
    assert np.all(forward(Gm, syn.uniform_volume(Gm, 1)) == 0.0)
    assert np.all(back(Gm, syn.uniform_projections(Gm, 1)) == 0.0)
    G1 = syn.Geometry(1, 1, 1, 4.0, 4.0, 4.0, 1, 1, 1.0, 1.0, 1000.0, 1500.0, (0.3,))
    one = np.ones((1, 1, 1), np.float32)
    g, ref = forward(G1, one), op.forward(G1, np.ones((1, 1, 1)))
    assert abs(g[0, 0, 0] - ref[0, 0, 0]) <= TOL * ref[0, 0, 0]
    f = back(G1, one)
    assert abs(f[0, 0, 0] - op.back_scatter(G1, np.ones((1, 1, 1)))[0, 0, 0]) <= TOL * f[0, 0, 0]


def test_steep_rays_axis_parallel_rays_and_odd_steps():
    G = syn.Geometry(24, 20, 40, 4.0, 4.0, 0.5, 28, 64, 5.0, 8.0, 1000.0, 1500.0, (0.2, 1.3, 2.9, 4.1, 5.6),
                     oz=3.0, step_mm=0.4)
    y, x = syn.uniform_projections(G, 28) - 0.2, syn.uniform_volume(G, 29)
    assert rel_l2(back(G, y), op.back_scatter(G, y.astype(np.float64))) <= TOL
    assert rel_l2_per_view(forward(G, x), op.forward(G, x.astype(np.float64))) <= TOL
    for step in (0.05, 0.9, 3.7):
        G = syn.Geometry(20, 18, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi, 1.0),
                         step_mm=step)
        y, x = syn.uniform_projections(G, 26), syn.uniform_volume(G, 27)
        assert rel_l2(back(G, y), op.back_scatter(G, y.astype(np.float64))) <= TOL, step
        assert rel_l2_per_view(forward(G, x), op.forward(G, x.astype(np.float64))) <= TOL, step


def test_paper_eq3_backprojector_kernel():
    for G, seed in ((syn.workload(1).geometry, 61), (ODD, 63)):
        y = syn.uniform_projections(G, seed)
        f = sl.Geometry(G).backproject_eq3(y)
        assert rel_l2(f, op.back_eq3(G, y.astype(np.float64))) <= TOL


def test_siddon_pair_kernels():
    """the paper's own projector (Siddon) and its transpose against the oracle's
    sort-all-crossings definition; 4-divisible and ragged / offset geometries, axis-parallel rays (odd grid: the central
    rays run through voxel centres, parallel to two axes), signed input."""
    AXIS = syn.Geometry(21, 19, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi, 1.0))
    for G, seed in ((syn.workload(1).geometry, 91), (ODD, 92), (RAGGED_TMA, 93), (AXIS, 94)):
        h = sl.Geometry(G)
        x, y = syn.uniform_volume(G, seed), syn.uniform_projections(G, seed) - 0.3
        g, f = h.siddon_forward(x), h.siddon_backproject(y)
        assert {"cbct::siddon_forward_kernel", "cbct::siddon_scatter_kernel"} <= set(sl.kernel_log())
        assert rel_l2_per_view(g, op.siddon_forward(G, x.astype(np.float64))) <= TOL
        assert rel_l2(f, op.siddon_back(G, y.astype(np.float64))) <= TOL
        lhs, rhs = float(np.sum(g.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * f))
        assert abs(lhs - rhs) <= TOL * abs(lhs)
        assert np.array_equal(f, h.siddon_backproject(y))                     # integer accumulation: reproducible
    Gm = replace(syn.workload(1).geometry, u0=5000.0)                         # every ray misses the volume
    hm = sl.Geometry(Gm)
    assert np.all(hm.siddon_forward(syn.uniform_volume(Gm, 1)) == 0.0)
    assert np.all(hm.siddon_backproject(syn.uniform_projections(Gm, 1)) == 0.0)


def test_siddon_ray_inside_a_grid_plane_is_one_of_the_two_valid_answers():
    """Even grid, centred odd detector: the central ray of the 0 / 90 / 180 degree views lies IN the grid plane y = 0
    (x = 0), where 'the voxel the ray is in' has two equally valid answers (and in fp64 the 90-degree ray, whose
    direction is 6e-17 off the plane, even switches sides at an arbitrary point).  What is unique is compared: every
    other ray matches the oracle; the in-plane rays must lie between the oracle's answers for the volume shifted by
    +-1e-6 mm across the plane (the two one-sided limits)."""
    G = syn.Geometry(20, 18, 7, 2.0, 2.0, 3.0, 21, 9, 2.5, 2.5, 1000.0, 1500.0, (0.0, math.pi / 2, math.pi))
    x = syn.uniform_volume(G, 95)
    g = sl.Geometry(G).siddon_forward(x).astype(np.float64)
    ref = op.siddon_forward(G, x.astype(np.float64))
    lim = [op.siddon_forward(replace(G, ox=sx * 1e-6, oy=sy * 1e-6), x.astype(np.float64)) for sx in (-1, 1) for sy in (-1, 1)]
    lo, hi = np.min(lim, axis=0), np.max(lim, axis=0)
    in_plane = np.zeros(G.proj_shape, bool)
    in_plane[:, :, G.nu // 2] = True                                           # u = 0: the column of rays inside the plane
    assert np.linalg.norm((g - ref)[~in_plane]) <= TOL * np.linalg.norm(ref[~in_plane])
    tol = 1e-5 * np.max(ref)
    assert np.all(g[in_plane] >= lo[in_plane] - tol) and np.all(g[in_plane] <= hi[in_plane] + tol)
    assert np.max(hi[in_plane] - lo[in_plane]) > 100 * tol                      # the case is not vacuous


def test_shared_memory_bank_model_reproduces_ncu_and_ranks_the_lane_layouts(monkeypatch):
    """The shim groups the lanes' shared-memory addresses into warp instructions and counts wavefronts (README.md).
    At the paper-size geometry, on a sample of CTAs: the 16x2 lane layout of the scatter kernel must reproduce what
    ncu measured on a B200 (profiles/README.md: 5.03e9 shared wavefronts / 1.63e9 ATOMS = 2.96 per instruction, the
    kernel's bound), which pins the model; the skewed 8x4 layout that is now the default must be clearly below it; the
    forward kernel's loads must be nearly conflict-free (ncu: 1.93e9 wavefronts for 1.67e9 LDS + staging)."""
    G = syn.workload(4).geometry
    y, x = syn.uniform_projections(G, 1), syn.uniform_volume(G, 1)
    stride = 311                                                   # 99 of the 30720 CTAs of a launch, spread over views and tiles
    red = {}
    for name, lanes, packed in (("captured", "1", "0"), ("default", "0", "1")):
        # captured: the 16x2 layout and the scalar stream, i.e. the kernel ncu profiled; default: skewed 8x4 lanes, packed
        # pairs with the second sample of a pair riding on the first one's reductions where both share a cell
        monkeypatch.setenv("CBCT_BT_LANES", lanes)
        monkeypatch.setenv("CBCT_BT_PACKED", packed)
        h = sl.Geometry(G)
        with sl.bank_stats(stride) as st:
            h.backproject(y)
        red[name] = st.red
    assert abs(red["captured"] - 2.96) <= 0.15, red                 # model vs ncu
    assert red["default"] <= 2.15 and red["default"] <= 0.75 * red["captured"], red
    h = sl.Geometry(G)
    with sl.bank_stats(stride) as st:
        h.forward(x)
    assert st.ld <= 1.15, st.ld
