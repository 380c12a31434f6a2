"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/cbct.h declares; argument validation that happens before any CUDA call; the binding fails
loudly without the library."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1008_2042_b200 import binding, build
from paper_1008_2042_b200 import synthetic as syn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    names = []
    for header in ("cbct.h", "cbct_debug.h"):        # the product ABI and the probes
        text = open(os.path.join(ROOT, "include", header)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names += re.findall(r"\b(?:int|long long|size_t|const char \*)\s*\*?\s*((?:cbct|tf|tv|mg)_\w+)\s*\(", text)
    return sorted(set(names))


@pytest.fixture(scope="module")
def cdll():
    path = build.build()
    return ctypes.CDLL(path)


def test_header_symbols_are_exported(cdll):
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(cdll, n), f"{n} declared in include/cbct.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_status_strings_and_version(cdll):
    cdll.cbct_status_string.restype = ctypes.c_char_p
    assert cdll.cbct_status_string(0) == b"ok"
    for code in (-1, -2, -3, -4, 1):
        assert len(cdll.cbct_status_string(code)) > 3
    assert cdll.cbct_version() >= 100
    assert cdll.cbct_last_cuda_error() == 0


def test_invalid_arguments_rejected_before_any_cuda_call():
    L = binding.lib()
    G = syn.workload(1).geometry
    out = ctypes.c_void_p()
    assert L.cbct_geometry_create(None, ctypes.byref(out)) == binding.CBCT_E_INVALID
    bad = [dict(nx=0), dict(dx=-1.0), dict(sdd=900.0), dict(sad=-5.0), dict(nu=0), dict(sad=100.0, sdd=150.0)]
    from dataclasses import replace
    for kw in bad:
        d, keep = binding.make_desc(replace(G, **kw))
        assert L.cbct_geometry_create(ctypes.byref(d), ctypes.byref(out)) == binding.CBCT_E_INVALID, kw
    d, keep = binding.make_desc(G)
    d.angles = None
    assert L.cbct_geometry_create(ctypes.byref(d), ctypes.byref(out)) == binding.CBCT_E_INVALID
    assert L.cbct_forward(None, None, None, None) == binding.CBCT_E_INVALID
    assert L.tf_decompose(None, None, 4, 4, 4, None) == binding.CBCT_E_INVALID
    assert L.mg_restrict(1, 1, 5, 4, 4, 2, 2, 1, None) == binding.CBCT_E_INVALID     # 5 not divisible by 2
    assert L.mg_prolong(1, 1, 4, 4, 4, 3, 1, 1, None) == binding.CBCT_E_INVALID      # factor not in {1,2}
    assert L.cbct_recon_create(ctypes.byref(binding.make_desc(G)[0]), 0, ctypes.byref(out)) == binding.CBCT_E_INVALID


def test_backproject_fixed_point_plan_bounds_the_oracle_weight_sums():
    """Host logic of the scatter backprojector: its int32 accumulators cannot wrap if the planned bound on the
    sum of trilinear weights per voxel and view holds.  P^T of a one-view all-ones projection (oracle) IS that
    sum times step, so the bound is checked against the oracle on ordinary and awkward geometries."""
    from dataclasses import replace
    from oracle import projector as op
    G1 = syn.workload(1).geometry
    cases = [G1, replace(G1, nu=24, nv=8, du=12.8, dv=12.8), replace(G1, step_mm=9.0), replace(G1, ox=30.0, oy=-20.0, oz=10.0),
             syn.Geometry(24, 20, 40, 4.0, 4.0, 0.5, 28, 64, 5.0, 8.0, 1000.0, 1500.0, (0.2, 1.3, 2.9, 4.1, 5.6), oz=3.0,
                          step_mm=0.4)]
    cases += [syn.workload(2).geometry, syn.workload(3).geometry]
    for G in cases:
        qb, group, w_view = binding.backproject_fixed_point_plan(G)
        assert 12 <= qb <= 22 and 1 <= group <= G.n_views
        assert group * w_view * 2.0 ** qb <= 2.0 ** 30          # the plan uses half the int32 range (the other half: detection)
        for v in (0, G.n_views // 3, G.n_views - 1):
            Gv = G.with_views([G.angles[v]])
            measured = op.back_scatter(Gv, np.ones(Gv.proj_shape)).max() / G.step
            assert measured <= w_view / 1.15, (G, v, measured, w_view)       # at least 15 % of margin left
    # paper-size and stress configs: the oracle evaluated voxel by voxel (gather form) on the voxels nearest to the source
    # of a view (where the samples are densest), the volume's corners and a random sample
    rng = np.random.default_rng(7)
    for cfg in (4, 5):
        G = syn.workload(cfg).geometry
        qb, group, w_view = binding.backproject_fixed_point_plan(G)
        xs, ys = (np.arange(G.nx) - (G.nx - 1) / 2) * G.dx, (np.arange(G.ny) - (G.ny - 1) / 2) * G.dy
        for v in (0, 5, G.n_views // 8):
            Gv = G.with_views([G.angles[v]])
            depth = np.add.outer(ys * np.sin(G.angles[v]), xs * np.cos(G.angles[v]))          # towards the source
            near = np.argsort(depth.ravel())[-24:]
            vox = [z * G.nx * G.ny + i for z in (0, G.nz // 2, G.nz - 1) for i in near]
            vox += [0, G.nx - 1, G.nx * G.ny * G.nz - 1] + list(rng.choice(G.nx * G.ny * G.nz, 100, replace=False))
            measured = op.back_gather_voxels(Gv, np.ones(Gv.proj_shape), np.sort(np.array(vox, dtype=np.int64))).max() / G.step
            assert measured <= w_view / 1.15, (cfg, v, measured, w_view)
            assert measured >= 0.4 * w_view, (cfg, v, measured, w_view)              # and the plan is not wasteful
    # paper-size config: 40 views in two groups (21 + 19) at 21 bits
    qb, group, w_view = binding.backproject_fixed_point_plan(syn.workload(4).geometry)
    assert qb == 21 and group == 21
    d, keep = binding.make_desc(replace(G1, sdd=900.0))
    assert binding.lib().cbct_backproject_fixed_point_plan(ctypes.byref(d), None, None, None) == binding.CBCT_E_INVALID


def test_siddon_fixed_point_plan_bounds_the_oracle_path_sums():
    """cbct_siddon_backproject accumulates g * length in int32: the planned bound on the path length one voxel collects
    from one view must hold against the oracle (P_siddon^T of a one-view all-ones projection IS that sum)."""
    from dataclasses import replace
    from oracle import projector as op
    G1 = syn.workload(1).geometry
    cases = [G1, replace(G1, nu=24, nv=8, du=12.8, dv=12.8), replace(G1, ox=30.0, oy=-20.0, oz=10.0), replace(G1, nu=384, du=0.8),
             syn.Geometry(24, 20, 40, 4.0, 4.0, 0.5, 28, 64, 5.0, 8.0, 1000.0, 1500.0, (0.2, 1.3, 2.9, 4.1, 5.6), oz=3.0)]
    for G in cases:
        qb, group, w_view = binding.siddon_fixed_point_plan(G)
        assert 9 <= qb <= 22 and 1 <= group <= G.n_views
        assert group * w_view * 2.0 ** qb < 2.0 ** 31
        for v in (0, G.n_views // 3, G.n_views - 1):
            Gv = G.with_views([G.angles[v]])
            measured = op.siddon_back(Gv, np.ones(Gv.proj_shape)).max()
            assert measured <= w_view, (G, v, measured, w_view)
    qb, group, w_view = binding.siddon_fixed_point_plan(syn.workload(4).geometry)
    assert qb == 19 and group == 40                                      # paper size: all 40 views in one group


def test_no_cpu_fallback_without_a_device():
    """On a box without an sm_100 GPU the product path must refuse, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    d, keep = binding.make_desc(syn.workload(1).geometry)
    out = ctypes.c_void_p()
    assert binding.lib().cbct_geometry_create(ctypes.byref(d), ctypes.byref(out)) == binding.CBCT_E_UNSUPPORTED
    with pytest.raises(binding.CbctError):
        binding.Geometry(syn.workload(1).geometry)


def test_product_path_does_not_import_the_oracle():
    for root, _dirs, files in os.walk(os.path.join(ROOT, "paper_1008_2042_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(root, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "cbct_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1008_2042_b200", text, flags=re.M), f
            assert "csrc/" not in text.replace("paper_1008_2042_b200/csrc)", ""), f


def test_synthetic_workloads_match_baseline_configs():
    shapes = {1: ((16, 64, 64), (32, 32, 96)), 2: ((32, 128, 128), (40, 96, 256)), 3: ((70, 256, 256), (40, 384, 512)),
              4: ((70, 512, 512), (40, 384, 512)), 5: ((70, 512, 512), (360, 768, 1024))}
    for i, (vs, ps) in shapes.items():
        w = syn.workload(i)
        assert w.geometry.vol_shape == vs and w.geometry.proj_shape == ps
        assert w.geometry.sad == 1000.0 and w.geometry.sdd == 1500.0
    w, ells, f0, g = syn.make_inputs(1)
    assert f0.dtype == np.float32 and g.dtype == np.float32 and len(ells) == 6
    assert f0.max() > 0 and g.max() > 0
    w2, _, f2, g2 = syn.make_inputs(1)
    assert np.array_equal(f0, f2) and np.array_equal(g, g2)          # seeded
