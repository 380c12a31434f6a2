"""Randomised sweep of the kernel sources executed on the host (tests/cpu_shim) against the fp64 oracle -- `-m "not gpu"`.
Seeded random geometries (volume and detector sizes, anisotropic voxels, offsets of volume and detector, arbitrary view
angles incl. axis-parallel and diagonal ones, SAD / SDD, sampling step) through cbct_forward / cbct_backproject, and random
shapes through the fused tight frame and the multigrid transfers.  The bar is the parity bar of the -m gpu tests (1e-5) plus a
clean device error word: a planning mistake of the TMA kernels (a box that does not cover its samples, an exhausted
fixed-point range) would show up there.  CBCT_FUZZ_N (default 24 geometries / 12 shapes) widens the sweep; round 2 ran 460
geometries and 60 shapes this way (DESIGN.md §1 item 9).
Geometries whose volume is only one or two slices thick are left out: rays that merely graze the zero-padded skirt of such a
volume make a projection out of hat-function tails, where a 1e-6-voxel fp32 position error is 1e-5 .. 1e-4 of the weight
(the one such case the sweep found is pinned below at the looser bound)."""
import math
import os

import numpy as np
import pytest

from cpu_shim import shimlib as sl
from oracle import projector as op
from oracle import solver as osv
from paper_1008_2042_b200 import synthetic as syn

N = int(os.environ.get("CBCT_FUZZ_N", "24"))


def rel(a, ref):
    return float(np.linalg.norm(a.astype(np.float64).ravel() - ref.ravel()) / max(np.linalg.norm(ref.ravel()), 1e-300))


def random_geometry(seed):
    rng = np.random.default_rng(seed)
    nx, ny, nz = 4 * int(rng.integers(3, 24)), 4 * int(rng.integers(3, 24)), int(rng.integers(1, 24))
    dx = float(rng.uniform(0.5, 4.0))
    dy, dz = dx * float(rng.choice([1.0, 1.0, 1.0, 0.8, 1.25])), dx * float(rng.uniform(0.7, 5.0))
    nu, nv = int(rng.integers(8, 110)), int(rng.integers(4, 70))
    sad = float(rng.uniform(600, 1500))
    sdd = sad * float(rng.uniform(1.2, 2.0))
    du, dv = min(dx, dy) * sdd / sad * float(rng.uniform(0.5, 1.8)), dz * sdd / sad * float(rng.uniform(0.15, 1.5))
    n_views = int(rng.integers(1, 9))
    ang = tuple(float(a) for a in rng.uniform(0, 2 * math.pi, n_views))
    if rng.random() < 0.3:
        ang = tuple(float(k * math.pi / 4) for k in range(n_views))              # axis-parallel and diagonal views
    off = [float(rng.normal(0, 5)) for _ in range(3)] if rng.random() < 0.5 else [0.0] * 3
    u0, v0 = (float(rng.normal(0, 10)), float(rng.normal(0, 10))) if rng.random() < 0.5 else (0.0, 0.0)
    step = float(rng.uniform(0.3, 1.2)) * min(dx, dy, dz) if rng.random() < 0.5 else 0.0
    return syn.Geometry(nx, ny, nz, dx, dy, dz, nu, nv, du, dv, sad, sdd, ang, ox=off[0], oy=off[1], oz=off[2], u0=u0, v0=v0,
                        step_mm=step)


def usable(G):
    return G.nz >= 3 and op.grid(G)[0] < G.sad


SEEDS = [s for s in range(1000, 1000 + 40 * N) if usable(random_geometry(s))][:N]


@pytest.mark.parametrize("seed", SEEDS)
def test_projectors_on_a_random_geometry(seed):
    G = random_geometry(seed)
    h = sl.Geometry(G)
    x, y = syn.uniform_volume(G, seed), syn.uniform_projections(G, seed) - 0.4
    e_p = rel(h.forward(x), op.forward(G, x.astype(np.float64)))
    e_pt = rel(h.backproject(y), op.back_scatter(G, y.astype(np.float64)))
    assert h.status() == (0, 0), (h.describe(), h.status())
    assert e_p <= 1e-5 and e_pt <= 1e-5, (h.describe(), e_p, e_pt)
    h.close()
    sl.check(0, "random geometry")


def test_the_grazed_two_slice_volume_the_sweep_found():
    """seed 1177 of the round-2 sweep: 60 x 24 x 2 voxels, detector 14 mm off centre -- every ray that touches the volume
    touches only its zero-padded skirt.  P and P^T stay consistent with each other (same fp32 positions) and within 1e-4."""
    G = random_geometry(1177)
    assert G.nz == 2
    h = sl.Geometry(G)
    x, y = syn.uniform_volume(G, 1177), syn.uniform_projections(G, 1177) - 0.4
    Px, PTy = h.forward(x), h.backproject(y)
    assert rel(Px, op.forward(G, x.astype(np.float64))) <= 1e-4 and rel(PTy, op.back_scatter(G, y.astype(np.float64))) <= 1e-4
    lhs, rhs = float(np.sum(Px.astype(np.float64) * y)), float(np.sum(x.astype(np.float64) * PTy))
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs) and h.status() == (0, 0)


@pytest.mark.parametrize("seed", range(max(N // 2, 1)))
def test_fused_tight_frame_and_multigrid_on_random_shapes(seed):
    rng = np.random.default_rng(1000 + seed)
    shape = (int(rng.integers(1, 90)), int(rng.integers(1, 70)), int(rng.integers(1, 100)))
    if rng.random() < 0.3:
        shape = (int(rng.integers(60, 140)), int(rng.integers(1, 40)), int(rng.integers(1, 60)))       # many z-segments
    f = (rng.standard_normal(shape) * rng.uniform(0.01, 10) + rng.uniform(-5, 5)).astype(np.float32)
    mu, clamp = float(rng.choice([0.0, 0.01, 0.3, 3.0])), bool(rng.integers(2))
    ref = osv.tf_apply(f.astype(np.float64), mu, clamp_nonneg=clamp)
    for impl in ("march", "tile"):
        assert np.max(np.abs(sl.tf_apply_fused(sl.dev(f), mu, clamp, impl=impl).numpy() - ref)) <= 2e-5 * np.max(np.abs(f)), impl
    fx, fy, fz = [int(v) for v in rng.integers(1, 3, 3)]
    sh = (fz * int(rng.integers(1, 20)), fy * int(rng.integers(1, 30)), fx * int(rng.choice([4, 8, 12, 20, 3, 5, 7, 16, 34])))
    fine = rng.random(sh).astype(np.float32)
    assert np.max(np.abs(sl.mg_restrict(sl.dev(fine), fx, fy, fz).numpy() - osv.mg_restrict(fine.astype(np.float64), fx, fy, fz))) <= 1e-6
    c = rng.random((sh[0] // fz, sh[1] // fy, sh[2] // fx)).astype(np.float32)
    assert np.max(np.abs(sl.mg_prolong(sl.dev(c), sh, fx, fy, fz).numpy() - osv.mg_prolong(c.astype(np.float64), fx, fy, fz))) <= 1e-6
    sl.check(0, "random shape")
