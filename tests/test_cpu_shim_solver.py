"""CGLS vector kernels, the tight-frame kernels, multigrid transfers and the A2 driver executed on the host by
tests/cpu_shim against the fp64 oracle -- `-m "not gpu"`.  Same purpose and caveats as test_cpu_shim_projectors.py:
it checks the kernel sources for indexing / synchronisation mistakes without a GPU; parity is claimed by `-m gpu`.
The cases mirror tests/test_gpu_solver.py (same tolerances) at host-sized inputs."""
import numpy as np
import pytest

from cpu_shim import shimlib as sl
from oracle import projector as op
from oracle import solver as osv
from paper_1008_2042_b200 import synthetic as syn


def rel(a, ref):
    return float(np.linalg.norm(np.asarray(a, np.float64).ravel() - ref.ravel()) / np.linalg.norm(ref.ravel()))


def ops(G):
    return (lambda x: op.forward(G, x)), (lambda r: op.back_scatter(G, r))


@pytest.fixture(autouse=True)
def _no_violation():
    yield
    sl.check(0, "end of test")


def test_cgls_teacher_forced_step_scalars_and_breakdown():
    w, _, f0, g = syn.make_inputs(1)
    G = w.geometry
    P, PT = ops(G)
    h = sl.Geometry(G)
    cg = sl.Cgls(h)
    g64 = g.astype(np.float64)
    d_g = sl.dev(g)
    st_free = osv.cgls_init(P, PT, np.zeros(G.vol_shape), g64)
    for step in range(2):
        x32 = np.float32(st_free["x"])
        st = osv.cgls_init(P, PT, x32.astype(np.float64), g64)
        d_x, d_r, d_p = sl.dev(x32), sl.Buf(h.proj_shape), sl.Buf(h.vol_shape)
        cg.init(d_g, d_x, d_r, d_p)
        assert rel(d_r.numpy(), st["r"]) <= 1e-5 and rel(d_p.numpy(), st["p"]) <= 1e-5, step
        sc = cg.scalars(d_r)
        assert abs(sc["gamma"] - st["gamma"]) <= 2e-5 * st["gamma"]
        st = osv.cgls_step(P, PT, st)
        cg.step(d_x, d_r, d_p)
        sc = cg.scalars(d_r)
        assert not sc["breakdown"]
        assert abs(sc["alpha"] - st["alpha"]) <= 2e-5 * abs(st["alpha"]) and abs(sc["beta"] - st["beta"]) <= 5e-5 * abs(st["beta"])
        assert rel(d_x.numpy(), st["x"]) <= 1e-5 and rel(d_r.numpy(), st["r"]) <= 1e-5 and rel(d_p.numpy(), st["p"]) <= 1e-5
        st_free = osv.cgls_step(P, PT, st_free)
    zg, zx = sl.dev(np.zeros(h.proj_shape)), sl.dev(np.zeros(h.vol_shape))
    d_r, d_p = sl.Buf(h.proj_shape), sl.Buf(h.vol_shape)
    cg.init(zg, zx, d_r, d_p)
    cg.step(zx, d_r, d_p)
    sc = cg.scalars(d_r)
    assert sc["breakdown"] and sc["alpha"] == 0.0 and np.all(zx.numpy() == 0) and np.all(np.isfinite(d_p.numpy()))


SHAPES = [(16, 64, 64), (5, 7, 9), (1, 33, 40), (3, 1, 70), (9, 10, 1), (1, 1, 1), (6, 37, 131)]


@pytest.mark.parametrize("shape", SHAPES)
def test_tf_three_call_path(shape):
    rng = np.random.default_rng(sum(shape))
    f = rng.standard_normal(shape).astype(np.float32)
    a_ref = osv.tf_decompose(f.astype(np.float64))
    d_f = sl.dev(f)
    d_a = sl.tf_decompose(d_f)
    a = d_a.numpy().astype(np.float64)
    assert np.max(np.abs(a - a_ref)) <= 1e-5 * np.max(np.abs(a_ref))
    sl.tf_shrink(d_a, 0.4)
    assert np.max(np.abs(d_a.numpy() - osv.tf_shrink(a, 0.4))) <= 1e-5 * np.max(np.abs(a_ref))
    r_ref = osv.tf_reconstruct(d_a.numpy().astype(np.float64))
    assert np.max(np.abs(sl.tf_reconstruct(d_a).numpy() - r_ref)) <= 1e-5 * max(np.max(np.abs(r_ref)), 1e-30)
    assert np.max(np.abs(sl.tf_reconstruct(sl.tf_decompose(d_f)).numpy() - f)) <= 1e-5 * np.max(np.abs(f))     # W^T W = I


@pytest.mark.parametrize("impl", ["march", "direct"])
@pytest.mark.parametrize("shape", SHAPES + [(31, 20, 45)])
def test_tf_reconstruct_both_kernels(shape, impl):
    rng = np.random.default_rng(sum(shape) + 1)
    a = rng.standard_normal((27,) + shape).astype(np.float32)
    sl.kernel_log()
    out = sl.tf_reconstruct(sl.dev(a), direct=(impl == "direct")).numpy()
    assert sl.kernel_log() == ["cbct::tf_reconstruct_march_kernel" if impl == "march" else "cbct::tf_reconstruct_kernel"]
    r_ref = osv.tf_reconstruct(a.astype(np.float64))
    assert np.max(np.abs(out - r_ref)) <= 1e-5 * np.max(np.abs(r_ref))


@pytest.mark.parametrize("impl", ["tile", "march"])
@pytest.mark.parametrize("shape", SHAPES + [(70, 57, 29), (23, 13, 57)])       # + several z-segments, several tiles in x and y
@pytest.mark.parametrize("mu,clamp", [(0.0, False), (0.3, False), (0.3, True), (2.0, True), (1e6, False)])
def test_tf_fused_matches_oracle(shape, mu, clamp, impl):
    """both kernels behind tf_apply_fused (the 3-D tile with 27-tap sums, the separable z-marching one), each on its own"""
    rng = np.random.default_rng(sum(shape) + 1)
    f = rng.standard_normal(shape).astype(np.float32)
    ref = osv.tf_apply(f.astype(np.float64), mu, clamp_nonneg=clamp)
    out = sl.tf_apply_fused(sl.dev(f), mu, clamp, impl=impl).numpy()
    assert sl.kernel_log()[-1].startswith("cbct::tf_fused_march_kernel" if impl == "march" else "cbct::tf_fused_kernel")
    assert np.max(np.abs(out - ref)) <= 2e-5 * np.max(np.abs(f))


@pytest.mark.parametrize("impl", ["tile", "march"])
def test_tf_fused_on_a_large_offset(impl):
    """||alpha_h||^2 must not be formed as a difference of large numbers: a flat region of value 100 with noise 0.01 next
    to an edge (the tile kernel subtracts the centre voxel first, the marching kernel sums squared difference bands)"""
    rng = np.random.default_rng(5)
    f = (100.0 + 0.01 * rng.standard_normal((12, 40, 50))).astype(np.float32)
    f[:, 20:, :] += 50.0
    ref = osv.tf_apply(f.astype(np.float64), 0.01, clamp_nonneg=True)
    assert np.max(np.abs(ref - f)) > 1e-4 * np.max(np.abs(f))                  # the shrinkage does something here
    assert np.max(np.abs(sl.tf_apply_fused(sl.dev(f), 0.01, True, impl=impl).numpy() - ref)) <= 1e-6 * np.max(np.abs(f))


@pytest.mark.parametrize("impl", ["tile", "march"])
def test_tf_fused_on_phantom_with_paper_mu(impl):
    """piecewise-constant phantom, mu = 5e-4: flat regions sit exactly at ||alpha_h|| = 0"""
    w, _, f0, _ = syn.make_inputs(1)
    ref = osv.tf_apply(f0.astype(np.float64), 5e-4, clamp_nonneg=True)
    out = sl.tf_apply_fused(sl.dev(f0), 5e-4, True, impl=impl).numpy()
    assert rel(out, ref) <= 1e-5 and np.max(np.abs(out - ref)) <= 1e-5 * np.max(np.abs(f0))


def test_tf_fused_default_is_the_checked_marching_kernel():
    """tf_apply_fused itself: the library's create-time style self-check (march against tile on a built-in volume) runs on
    the first call and, passing, selects the marching kernel"""
    f = np.random.default_rng(2).standard_normal((9, 31, 45)).astype(np.float32)
    out = sl.tf_apply_fused(sl.dev(f), 0.2, True).numpy()
    assert sl.kernel_log()[-1].startswith("cbct::tf_fused_march_kernel")
    assert sl.lib().tf_apply_fused_describe().decode().startswith("tf_fused_march_kernel (self-check passed)")
    assert np.max(np.abs(out - osv.tf_apply(f.astype(np.float64), 0.2, clamp_nonneg=True))) <= 2e-5 * np.max(np.abs(f))


@pytest.mark.parametrize("shape,fac", [((6, 8, 10), (2, 2, 1)), ((4, 6, 2), (2, 2, 2)), ((70, 64, 32), (2, 2, 1)),
                                       ((3, 5, 8), (2, 1, 1)), ((2, 2, 2), (1, 1, 2)),
                                       # rows of float4 (the vectorised kernels): every factor combination, ragged tiles
                                       ((4, 6, 16), (2, 2, 2)), ((6, 4, 24), (1, 2, 1)), ((2, 6, 8), (2, 1, 2)), ((3, 5, 12), (1, 1, 1)),
                                       ((66, 18, 264), (2, 2, 2)), ((5, 34, 136), (2, 2, 1))])
def test_mg_restrict_prolong_and_extrapolate(shape, fac):
    fx, fy, fz = fac
    rng = np.random.default_rng(5)
    fine = rng.random(shape).astype(np.float32)
    cshape = (shape[0] // fz, shape[1] // fy, shape[2] // fx)
    assert np.max(np.abs(sl.mg_restrict(sl.dev(fine), fx, fy, fz).numpy() - osv.mg_restrict(fine.astype(np.float64), fx, fy, fz))) <= 1e-6
    coarse = rng.random(cshape).astype(np.float32)
    assert np.max(np.abs(sl.mg_prolong(sl.dev(coarse), shape, fx, fy, fz).numpy() - osv.mg_prolong(coarse.astype(np.float64), fx, fy, fz))) <= 1e-6
    b = rng.random(shape).astype(np.float32)
    v = sl.a2_extrapolate(sl.dev(fine), sl.dev(b), 0.2817).numpy()
    assert np.max(np.abs(v - (fine + 0.2817 * (fine.astype(np.float64) - b)))) <= 1e-6


def test_multigrid_a2_driver_two_levels():
    """the whole driver (cbct_tf_reconstruct: cascade, A2, CGLS, fused tight frame) on a small two-level problem"""
    G = syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 48, 16, 3.2, 3.2, 1000.0, 1500.0, tuple(2 * np.pi * k / 12 for k in range(12)))
    f0 = syn.uniform_volume(G, 81)
    g = op.forward(G, f0.astype(np.float64)).astype(np.float32)

    def make_ops(fac):
        return ops(G.coarsen_xy(fac) if fac > 1 else G)

    mu, n_outer, n_cgls = 5e-4, [2, 2], 2
    ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, mu)
    out = sl.tf_reconstruct_volume(G, sl.dev(g), 2, n_outer, n_cgls, mu, True).numpy()
    assert rel(out, ref) <= 1e-4


def test_short_scan_cascade_with_detector_binning():
    """a 200-degree arc (unequal orientation phases, endpoints included) through the
    two-level driver, with and without detector binning at the coarse level, against the oracle's cascade."""
    G = syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 48, 16, 3.2, 3.2, 1000.0, 1500.0, syn.short_scan(11, 200.0, -10.0))
    f0 = syn.uniform_volume(G, 82)
    g = op.forward(G, f0.astype(np.float64)).astype(np.float32)
    mu, n_outer, n_cgls = 5e-4, [2, 2], 2
    for binned in (False, True):
        def make_ops(fac, binned=binned):
            Gl = G.coarsen_xy(fac) if fac > 1 else G
            return ops(Gl.bin_detector(fac) if (binned and fac > 1) else Gl)
        ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, mu, bin_detector=binned)
        out = sl.recon_run(G, sl.dev(g), 2, n_outer, n_cgls, mu, True, bin_detector=binned).numpy()
        assert rel(out, ref) <= 1e-4, binned
    import ctypes as C
    from paper_1008_2042_b200 import binding as cb
    d, _keep = cb.make_desc(syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 47, 16, 3.2, 3.2, 1000.0, 1500.0, (0.0, 1.0)))
    h = C.c_void_p()
    assert sl.lib().cbct_recon_create_ex(C.byref(d), 2, 1, C.byref(h)) == cb.CBCT_E_INVALID      # 47 pixels do not bin by 2
    assert sl.lib().cbct_recon_create_ex(C.byref(d), 2, 6, C.byref(h)) == cb.CBCT_E_INVALID      # unknown flag


@pytest.mark.parametrize("shape", [(6, 20, 24), (1, 9, 33), (5, 1, 7), (3, 4, 1), (1, 1, 1)])
def test_tv_rof_matches_oracle(shape):
    """the ROF descent with its device-resident control state against the oracle's
    loop -- same number of trials and accepted steps (the decisions are taken on fp64 energies on both sides), same
    volume, same final energy; ragged and 1-thick shapes; with and without the positivity clamp."""
    from oracle import tv as otv
    rng = np.random.default_rng(sum(shape))
    u = (rng.random(shape) + 0.3 * rng.standard_normal(shape)).astype(np.float32)
    for mu_tv, eps, max_iter, rel_tol in ((0.3, 0.05, 25, 1e-3), (0.05, 0.02, 8, 0.0), (0.0, 0.05, 5, 1e-3)):
        trace = []
        ref, it = otv.rof(u.astype(np.float64), mu_tv, eps, max_iter, rel_tol, trace=trace)
        out, trials, accepted, energy = sl.tv_rof(sl.dev(u), mu_tv, eps, max_iter, rel_tol)
        assert trials == it and accepted == sum(1 for t in trace if t[0]), (shape, mu_tv, trials, it)
        assert np.max(np.abs(out.numpy() - ref)) <= 2e-5 * max(np.max(np.abs(ref)), 1e-30), (shape, mu_tv)
        e_ref = otv.tv_energy(ref, u.astype(np.float64), mu_tv, eps)
        assert abs(energy - e_ref) <= 1e-5 * max(e_ref, 1e-30)
    out, *_ = sl.tv_rof(sl.dev(u), 0.3, 0.05, 25, 1e-3, clamp=True)
    ref, _ = otv.rof(u.astype(np.float64), 0.3, 0.05, 25, 1e-3)
    assert np.max(np.abs(out.numpy() - np.maximum(ref, 0.0))) <= 2e-5 * np.max(np.abs(ref))
    assert "cbct::tv_trial_kernel" in sl.kernel_log()


def test_tv_cascade_matches_oracle():
    """the TV comparison algorithm on the two-level cascade (cbct_recon_run_tv) against solver.multigrid_a2 with the ROF
    regulariser of oracle/tv.py"""
    from oracle import tv as otv
    G = syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 48, 16, 3.2, 3.2, 1000.0, 1500.0, tuple(2 * np.pi * k / 12 for k in range(12)))
    f0 = syn.uniform_volume(G, 83)
    g = op.forward(G, f0.astype(np.float64)).astype(np.float32)

    def make_ops(fac):
        return ops(G.coarsen_xy(fac) if fac > 1 else G)

    mu_tv, eps, rof_iter, rel_tol, n_outer, n_cgls = 0.02, 0.01, 10, 1e-3, [2, 2], 2
    ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, 0.0,
                           regulariser=otv.tv_regulariser(mu_tv, eps, rof_iter, rel_tol))
    out = sl.recon_run_tv(G, sl.dev(g), 2, n_outer, n_cgls, mu_tv, eps, rof_iter, rel_tol).numpy()
    assert rel(out, ref) <= 1e-4
    import ctypes as C
    from paper_1008_2042_b200 import binding as cb
    d, _keep = cb.make_desc(G)                                  # a handle created without CBCT_RECON_TV has no workspace for it
    h = C.c_void_p()
    sl.check(sl.lib().cbct_recon_create_ex(C.byref(d), 1, 0, C.byref(h)), "create")
    arr = (C.c_int * 1)(1)
    buf = sl.Buf(G.vol_shape)
    assert sl.lib().cbct_recon_run_tv(h, sl.dev(g).ptr, buf.ptr, arr, 1, 0.1, 0.1, 3, 1e-3, 1, None) == cb.CBCT_E_INVALID
    sl.lib().cbct_recon_destroy(h)


def test_microbench_kernels_stay_in_bounds():
    """cbct_microbench (SURVEY.md §8(d) denominators) with its timed loops shortened: every kernel runs under the shim's
    guards and alignment checks; the rates themselves mean nothing on the host."""
    import ctypes as C
    for kind in range(8):
        out = (C.c_double * 3)()
        sl.check(sl.lib().cbct_microbench(kind, 1, out, None), f"cbct_microbench({kind})")
        assert out[2] > 0
    assert sl.lib().cbct_microbench(8, 1, out, None) == -1


def test_cgls_step_takes_its_norms_from_the_projector_launches():
    """SURVEY.md §8(d) "fused minimum": on a handle served by the TMA kernels ||q||^2 comes out of the epilogue of P and
    ||s||^2 out of the conversion pass of P^T -- no separate pass over q or s (the one sumsq_kernel left in a step is the
    rms of the P^T INPUT for its fixed-point reference).  A handle served by the plain kernels reduces q and s itself.
    Either way the scalars are the oracle's."""
    w, _, f0, g = syn.make_inputs(1)
    several_groups = syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 64, 24, 1.6, 1.6, 1000.0, 1500.0, syn.full_circle(12), step_mm=0.5)
    assert "views/group 2" in sl.Geometry(several_groups).describe()      # ||s||^2 must come from the LAST of six conversion passes
    for G, n_sumsq, fwd in ((w.geometry, 1, "cbct::forward_tma_kernel"), (several_groups, 1, "cbct::forward_tma_kernel"),
                            (syn.Geometry(37, 29, 11, 2.0, 3.0, 5.0, 45, 19, 2.3, 3.1, 1000.0, 1500.0, (0.0, 0.4, 2.0, 4.0)), 2, "cbct::forward_")):
        P, PT = ops(G)
        gg = syn.uniform_projections(G, 3) if G is not w.geometry else g
        h = sl.Geometry(G)
        cg = sl.Cgls(h)
        d_x, d_r, d_p = sl.dev(np.zeros(h.vol_shape)), sl.Buf(h.proj_shape), sl.Buf(h.vol_shape)
        cg.init(sl.dev(gg), d_x, d_r, d_p)
        st = osv.cgls_init(P, PT, np.zeros(G.vol_shape), gg.astype(np.float64))
        assert abs(cg.scalars()["gamma"] - st["gamma"]) <= 2e-5 * st["gamma"]
        sl.kernel_log()
        cg.step(d_x, d_r, d_p)
        log = sl.kernel_log()
        assert sum(k == "cbct::sumsq_kernel" for k in log) == n_sumsq and any(k.startswith(fwd) for k in log), log
        st = osv.cgls_step(P, PT, st)
        sc = cg.scalars()
        assert abs(sc["qq"] - st["qq"]) <= 2e-5 * st["qq"] and abs(sc["gamma"] - st["gamma"]) <= 2e-5 * st["gamma"]
        assert abs(sc["alpha"] - st["alpha"]) <= 2e-5 * abs(st["alpha"]) and abs(sc["beta"] - st["beta"]) <= 5e-5 * abs(st["beta"])
