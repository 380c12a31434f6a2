"""SLOW, opt-in (CBCT_SLOW=1): the default P / P^T kernels executed on the host (tests/cpu_shim) at BASELINE.json's
full sizes -- cfg 3 (256x256x70) and cfg 4, the paper size (512x512x70, 40 views of 512x384, 6.7e9 samples per projector
call) -- in the launch configuration bench.py times, against the oracle on sampled outputs, plus the adjoint identity.

Each projector call takes minutes on a handful of cores (one fiber per CUDA thread), which is why this is not part of the
default `-m "not gpu"` run; it exists so that the statement "the full-size launch configuration indexes, plans its boxes
and accumulates correctly" is reproducible from the tracked tree without a GPU:

    CBCT_SLOW=1 python -m pytest tests/test_cpu_shim_fullsize.py -q -s          # ~25 min on 8 cores

It is still no parity claim for the device (the `-m gpu` twin is tests/test_gpu_projectors.py::test_full_size_sampled_outputs).
"""
import os

import numpy as np
import pytest

from cpu_shim import shimlib as sl
from oracle import projector as op
from paper_1008_2042_b200 import synthetic as syn

pytestmark = pytest.mark.skipif(os.environ.get("CBCT_SLOW") != "1", reason="slow (minutes per projector call): set CBCT_SLOW=1")

TOL = 1e-5


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_sampled_outputs_under_the_shim(cfg):
    w = syn.workload(cfg)
    G = w.geometry
    f0 = syn.voxelise(G, syn.ellipsoids_for(w))
    h = sl.Geometry(G)
    info = h.info()
    print(f"cfg {cfg}:", h.describe(), flush=True)
    sl.kernel_log()
    g = h.forward(f0)
    assert any(k.startswith("cbct::forward_tma_kernel<") for k in sl.kernel_log())
    rng = np.random.default_rng(cfg)
    rays = np.sort(rng.choice(info["n_rays"], 4000, replace=False))
    ref = op.forward_rays(G, f0.astype(np.float64), rays)
    got = g.ravel()[rays].astype(np.float64)
    print("P  sampled rel-L2", np.linalg.norm(got - ref) / np.linalg.norm(ref), flush=True)
    assert np.linalg.norm(got - ref) <= TOL * np.linalg.norm(ref)
    assert np.max(np.abs(got - ref)) <= 2e-5 * np.max(np.abs(ref))
    y = syn.uniform_projections(G, cfg)
    f = h.backproject(y)
    log = sl.kernel_log()
    assert any(k.startswith("cbct::backproject_scatter_kernel<") for k in log)
    vox = np.sort(rng.choice(info["n_vox"], 300, replace=False))
    vox[:4] = [0, G.nx - 1, info["n_vox"] - G.nx, info["n_vox"] - 1]
    refv = op.back_gather_voxels(G, y.astype(np.float64), vox)
    gotv = f.ravel()[vox].astype(np.float64)
    print("P^T sampled rel-L2", np.linalg.norm(gotv - refv) / np.linalg.norm(refv), flush=True)
    assert np.linalg.norm(gotv - refv) <= TOL * np.linalg.norm(refv)
    assert np.max(np.abs(gotv - refv)) <= 2e-5 * np.max(np.abs(refv))
    assert h.status() == (0, 0)                                  # no guard fired: waits, box ranges, fixed-point head-room
    x = syn.uniform_volume(G, cfg)
    Px = h.forward(x)
    lhs, rhs = float(np.sum(Px.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * f))
    print("adjoint", abs(lhs - rhs) / abs(lhs), flush=True)
    assert abs(lhs - rhs) <= TOL * abs(lhs)
    sl.check(0, "full-size run")
