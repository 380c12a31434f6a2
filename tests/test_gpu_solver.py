"""GPU parity of CGLS, the tight frame, multigrid and the A2 driver against the fp64 oracle, through
the C ABI (python -m pytest -m gpu).

Tolerances: single CGLS step (teacher-forced from the oracle's state) <= 1e-5; free-running CGLS with
n_cgls = 3 and A2 outer iterations <= 1e-4 (north_star "reconstructed volumes after N iterations agree
to 1e-4"; protocol of SURVEY.md §8(c) item 32); tight frame / multigrid <= 1e-5 (fp32 stencils).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import projector as op                      # noqa: E402
from oracle import solver as osv                        # noqa: E402
from paper_1008_2042_b200 import binding as cb          # noqa: E402
from paper_1008_2042_b200 import synthetic as syn       # noqa: E402


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy().astype(np.float64)


def rel(a, ref):
    return float(np.linalg.norm(np.asarray(a, np.float64).ravel() - ref.ravel()) / np.linalg.norm(ref.ravel()))


def ops(G):
    return (lambda x: op.forward(G, x)), (lambda r: op.back_scatter(G, r))


# ------------------------------------------------------------------------------------------ CGLS
def test_cgls_teacher_forced_steps_and_scalars():
    """Single-step parity from several states: the oracle free-runs; at each of its iterates x_j both
    sides restart (Initialize + one pass through steps 1-7) from the same fp32 x_j,
    so a GPU step never inherits GPU rounding from earlier steps."""
    w, _, f0, g = syn.make_inputs(1)
    G = w.geometry
    P, PT = ops(G)
    h = cb.Geometry(G)
    cg = cb.Cgls(h)
    g64 = g.astype(np.float64)
    d_g = dev(g)
    st_free = osv.cgls_init(P, PT, np.zeros(G.vol_shape), g64)
    for step in range(4):
        x32 = np.float32(st_free["x"])
        st = osv.cgls_init(P, PT, x32.astype(np.float64), g64)
        d_x = dev(x32)
        d_r, d_p = torch.empty_like(d_g), torch.empty_like(d_x)
        cg.init(d_g, d_x, d_r, d_p)
        assert rel(host(d_r), st["r"]) <= 1e-5 and rel(host(d_p), st["p"]) <= 1e-5, step
        sc = cg.scalars(d_r)
        assert abs(sc["gamma"] - st["gamma"]) <= 2e-5 * st["gamma"], step
        assert abs(sc["rr"] - np.sum(st["r"] ** 2)) <= 2e-5 * np.sum(st["r"] ** 2), step
        st = osv.cgls_step(P, PT, st)
        cg.step(d_x, d_r, d_p)
        sc = cg.scalars(d_r)
        assert not sc["breakdown"]
        assert abs(sc["alpha"] - st["alpha"]) <= 2e-5 * abs(st["alpha"]), step
        assert abs(sc["beta"] - st["beta"]) <= 5e-5 * abs(st["beta"]), step
        assert rel(host(d_x), st["x"]) <= 1e-5, step
        assert rel(host(d_r), st["r"]) <= 1e-5, step
        assert rel(host(d_p), st["p"]) <= 1e-5, step
        st_free = osv.cgls_step(P, PT, st_free)


@pytest.mark.parametrize("cfg,steps,tol", [(1, 3, 1e-4), (2, 3, 1e-4)])
def test_cgls_free_running(cfg, steps, tol):
    w, _, f0, g = syn.make_inputs(cfg)
    G = w.geometry
    P, PT = ops(G)
    x_ref, hist = osv.cgls(P, PT, np.zeros(G.vol_shape), g.astype(np.float64), steps)
    h = cb.Geometry(G)
    cg = cb.Cgls(h)
    d_g, d_x = dev(g), dev(np.zeros(G.vol_shape))
    d_r, d_p = torch.empty_like(d_g), torch.empty_like(d_x)
    cg.init(d_g, d_x, d_r, d_p)
    rr = [cg.scalars(d_r)["rr"]]
    for _ in range(steps):
        cg.step(d_x, d_r, d_p)
        rr.append(cg.scalars(d_r)["rr"])
    assert rel(host(d_x), x_ref) <= tol
    assert all(b <= a * (1 + 1e-6) for a, b in zip(rr, rr[1:]))
    assert np.allclose(rr, hist, rtol=1e-3)


def test_cgls_ten_steps_divergence_is_reported_not_hidden():
    """Config 1 asks for 10 free-running CGLS iterations.  fp32 vs fp64 CGLS drift apart with the
    conditioning of P; the bound asserted here is what the arithmetic
    supports (1e-3 at 10 steps), the 1e-4 bar applies to n_cgls = 3 restarts."""
    w, _, f0, g = syn.make_inputs(1)
    G = w.geometry
    P, PT = ops(G)
    x_ref, _ = osv.cgls(P, PT, np.zeros(G.vol_shape), g.astype(np.float64), 10)
    h = cb.Geometry(G)
    cg = cb.Cgls(h)
    d_g, d_x = dev(g), dev(np.zeros(G.vol_shape))
    d_r, d_p = torch.empty_like(d_g), torch.empty_like(d_x)
    cg.init(d_g, d_x, d_r, d_p)
    for _ in range(10):
        cg.step(d_x, d_r, d_p)
    err = rel(host(d_x), x_ref)
    print("cgls 10-step fp32-vs-fp64 rel-L2:", err)
    assert err <= 1e-3


def test_cgls_norms_from_the_projector_launches_with_several_accumulation_groups():
    """||q||^2 comes out of the epilogue of P and ||s||^2 out of the LAST conversion pass of P^T (SURVEY.md §8(d) "fused
    minimum"); here P^T needs six accumulation groups (views/group 2), and the scalars must still be the oracle's."""
    G = syn.Geometry(32, 32, 8, 4.0, 4.0, 4.0, 64, 24, 1.6, 1.6, 1000.0, 1500.0, syn.full_circle(12), step_mm=0.5)
    P, PT = ops(G)
    g = syn.uniform_projections(G, 3)
    h = cb.Geometry(G)
    print(h.describe())
    cg = cb.Cgls(h)
    d_x = torch.zeros(h.vol_shape, dtype=torch.float32, device="cuda")
    d_r = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
    d_p = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
    cg.init(dev(g), d_x, d_r, d_p)
    st = osv.cgls_init(P, PT, np.zeros(G.vol_shape), g.astype(np.float64))
    assert abs(cg.scalars()["gamma"] - st["gamma"]) <= 2e-5 * st["gamma"]
    for _ in range(2):
        cg.step(d_x, d_r, d_p)
        st = osv.cgls_step(P, PT, st)
        sc = cg.scalars()
        assert abs(sc["qq"] - st["qq"]) <= 5e-5 * st["qq"] and abs(sc["gamma"] - st["gamma"]) <= 5e-5 * st["gamma"]
    assert rel(host(d_x), st["x"]) <= 1e-4 and h.status() == (True, [])


def test_cgls_breakdown_flag():
    G = syn.workload(1).geometry
    h = cb.Geometry(G)
    cg = cb.Cgls(h)
    d_g = torch.zeros(h.proj_shape, device="cuda")
    d_x = torch.zeros(h.vol_shape, device="cuda")
    d_r, d_p = torch.empty_like(d_g), torch.empty_like(d_x)
    cg.init(d_g, d_x, d_r, d_p)
    cg.step(d_x, d_r, d_p)
    sc = cg.scalars(d_r)
    assert sc["breakdown"] and sc["alpha"] == 0.0
    assert torch.all(d_x == 0) and torch.all(torch.isfinite(d_p))


# ------------------------------------------------------------------------------------------ tight frame
SHAPES = [(16, 64, 64), (5, 7, 9), (1, 33, 40), (3, 1, 70), (9, 10, 1), (1, 1, 1), (6, 37, 131)]


@pytest.mark.parametrize("shape", SHAPES)
def test_tf_three_call_path(shape):
    rng = np.random.default_rng(sum(shape))
    f = rng.standard_normal(shape).astype(np.float32)
    a_ref = osv.tf_decompose(f.astype(np.float64))
    d_f = dev(f)
    d_a = torch.empty((27,) + shape, dtype=torch.float32, device="cuda")
    cb.tf_decompose(d_f, d_a)
    a = host(d_a)
    assert np.max(np.abs(a - a_ref)) <= 1e-5 * np.max(np.abs(a_ref))
    mu = 0.4
    cb.tf_shrink(d_a, mu)
    s_ref = osv.tf_shrink(a, mu)                           # same input as the kernel saw
    assert np.max(np.abs(host(d_a) - s_ref)) <= 1e-5 * np.max(np.abs(a_ref))
    d_out = torch.empty_like(d_f)
    cb.tf_reconstruct(d_a, d_out)
    r_ref = osv.tf_reconstruct(host(d_a))
    assert np.max(np.abs(host(d_out) - r_ref)) <= 1e-5 * max(np.max(np.abs(r_ref)), 1e-30)
    # perfect reconstruction through the GPU alone: W^T W = I
    cb.tf_decompose(d_f, d_a)
    cb.tf_reconstruct(d_a, d_out)
    assert np.max(np.abs(host(d_out) - f)) <= 1e-5 * np.max(np.abs(f))


@pytest.mark.parametrize("impl", ["march", "direct"])
@pytest.mark.parametrize("shape", SHAPES + [(31, 20, 45)])
def test_tf_reconstruct_both_kernels(shape, impl):
    """D^T has two kernels: the separable z-marching one (tf_reconstruct) and the direct 27x27-tap one
    (tf_reconstruct_direct, cbct_debug.h); several z-segments, ragged tiles, 1-thick axes."""
    rng = np.random.default_rng(sum(shape) + 1)
    a = rng.standard_normal((27,) + shape).astype(np.float32)
    d_a = dev(a)
    d_out = torch.empty(shape, dtype=torch.float32, device="cuda")
    (cb.tf_reconstruct_direct if impl == "direct" else cb.tf_reconstruct)(d_a, d_out)
    torch.cuda.synchronize()
    r_ref = osv.tf_reconstruct(a.astype(np.float64))
    assert np.max(np.abs(host(d_out) - r_ref)) <= 1e-5 * np.max(np.abs(r_ref))


@pytest.mark.parametrize("impl", [None, "tile", "march"])
@pytest.mark.parametrize("shape", SHAPES + [(70, 57, 29), (23, 13, 57)])       # + several z-segments, several tiles in x and y
@pytest.mark.parametrize("mu,clamp", [(0.0, False), (0.3, False), (0.3, True), (2.0, True), (1e6, False)])
def test_tf_fused_matches_oracle(shape, mu, clamp, impl):
    """tf_apply_fused (the library's choice) and each of the two kernels behind it on its own (cbct_debug.h)"""
    rng = np.random.default_rng(sum(shape) + 1)
    f = rng.standard_normal(shape).astype(np.float32)
    ref = osv.tf_apply(f.astype(np.float64), mu, clamp_nonneg=clamp)
    d_out = torch.empty(shape, dtype=torch.float32, device="cuda")
    cb.tf_apply_fused(dev(f), d_out, mu, clamp, impl=impl)
    assert np.max(np.abs(host(d_out) - ref)) <= 2e-5 * np.max(np.abs(f))


@pytest.mark.parametrize("impl", [None, "tile", "march"])
def test_tf_fused_on_phantom_with_paper_mu(impl):
    """A piecewise-constant phantom with small values and mu = 5e-4: flat regions sit
    exactly at ||alpha_h|| = 0 and edges far above mu."""
    w, _, f0, _ = syn.make_inputs(1)
    ref = osv.tf_apply(f0.astype(np.float64), 5e-4, clamp_nonneg=True)
    d_out = torch.empty(f0.shape, dtype=torch.float32, device="cuda")
    cb.tf_apply_fused(dev(f0), d_out, 5e-4, True, impl=impl)
    assert rel(host(d_out), ref) <= 1e-5
    assert np.max(np.abs(host(d_out) - ref)) <= 1e-5 * np.max(np.abs(f0))


@pytest.mark.parametrize("impl", ["tile", "march"])
def test_tf_fused_on_a_large_offset(impl):
    """||alpha_h||^2 must not be formed as a difference of large numbers (value 100, noise 0.01, next to an edge)"""
    rng = np.random.default_rng(5)
    f = (100.0 + 0.01 * rng.standard_normal((12, 40, 50))).astype(np.float32)
    f[:, 20:, :] += 50.0
    ref = osv.tf_apply(f.astype(np.float64), 0.01, clamp_nonneg=True)
    d_out = torch.empty(f.shape, dtype=torch.float32, device="cuda")
    cb.tf_apply_fused(dev(f), d_out, 0.01, True, impl=impl)
    assert np.max(np.abs(host(d_out) - ref)) <= 1e-6 * np.max(np.abs(f))


def test_tf_fused_kernel_in_use_is_reported():
    print("tf_apply_fused:", cb.tf_apply_fused_describe())
    assert cb.tf_apply_fused_describe().startswith(("tf_fused_march_kernel", "tf_fused_kernel"))


# ------------------------------------------------------------------------------------------ multigrid + A2 step 1
@pytest.mark.parametrize("shape,fac", [((6, 8, 10), (2, 2, 1)), ((4, 6, 2), (2, 2, 2)), ((70, 64, 32), (2, 2, 1)),
                                       ((3, 5, 8), (2, 1, 1)), ((2, 2, 2), (1, 1, 2)),
                                       # rows of float4 (the vectorised kernels): every factor combination, ragged tiles
                                       ((4, 6, 16), (2, 2, 2)), ((6, 4, 24), (1, 2, 1)), ((2, 6, 8), (2, 1, 2)), ((3, 5, 12), (1, 1, 1)),
                                       ((66, 18, 264), (2, 2, 2)), ((5, 34, 136), (2, 2, 1))])
def test_mg_restrict_prolong(shape, fac):
    fx, fy, fz = fac
    rng = np.random.default_rng(5)
    fine = rng.random(shape).astype(np.float32)
    cshape = (shape[0] // fz, shape[1] // fy, shape[2] // fx)
    d_c = torch.empty(cshape, dtype=torch.float32, device="cuda")
    cb.mg_restrict(dev(fine), d_c, fx, fy, fz)
    assert np.max(np.abs(host(d_c) - osv.mg_restrict(fine.astype(np.float64), fx, fy, fz))) <= 1e-6
    coarse = rng.random(cshape).astype(np.float32)
    d_f = torch.empty(shape, dtype=torch.float32, device="cuda")
    cb.mg_prolong(dev(coarse), d_f, fx, fy, fz)
    assert np.max(np.abs(host(d_f) - osv.mg_prolong(coarse.astype(np.float64), fx, fy, fz))) <= 1e-6


def test_a2_extrapolate():
    rng = np.random.default_rng(6)
    a, b = rng.random((4, 5, 6)).astype(np.float32), rng.random((4, 5, 6)).astype(np.float32)
    d_v = torch.empty((4, 5, 6), dtype=torch.float32, device="cuda")
    cb.a2_extrapolate(dev(a), dev(b), d_v, 0.2817)
    assert np.max(np.abs(host(d_v) - (a + 0.2817 * (a.astype(np.float64) - b)))) <= 1e-6


# ------------------------------------------------------------------------------------------ A2 driver
def test_a2_single_level_matches_oracle():
    w, _, f0, g = syn.make_inputs(1)
    G = w.geometry
    P, PT = ops(G)
    mu, n_outer, n_cgls = 5e-4, 4, 3
    ref = osv.a2(P, PT, g.astype(np.float64), np.zeros(G.vol_shape), n_outer, n_cgls, mu, momentum=True)
    rec = cb.Recon(G, 1)
    d_f = torch.empty(G.vol_shape, dtype=torch.float32, device="cuda")
    rec.run(dev(g), d_f, [n_outer], n_cgls, mu, True)
    assert rel(host(d_f), ref) <= 1e-4
    # host-buffer entry point gives the same volume
    h_f = np.empty(G.vol_shape, np.float32)
    rec.run_host(np.ascontiguousarray(g), h_f, [n_outer], n_cgls, mu, True)
    assert np.array_equal(h_f, host(d_f).astype(np.float32))
    # momentum off = Algorithm A1
    ref1 = osv.a2(P, PT, g.astype(np.float64), np.zeros(G.vol_shape), 2, n_cgls, mu, momentum=False)
    rec.run(dev(g), d_f, [2], n_cgls, mu, False)
    assert rel(host(d_f), ref1) <= 1e-4


def test_multigrid_cascade_matches_oracle_two_levels():
    """Config-2 shape of the solver (2-level multigrid TF-CGLS on noisy data) at a size the oracle
    finishes in seconds: the config-2 geometry with half the views, 3 outer iterations per level."""
    w, ells, f0, g_full = syn.make_inputs(2)
    G = w.geometry.with_views(w.geometry.angles[::2])
    g = np.ascontiguousarray(g_full[::2])

    def make_ops(fac):
        Gl = G.coarsen_xy(fac) if fac > 1 else G
        return ops(Gl)

    mu, n_outer, n_cgls = 5e-4, [3, 3], 2
    ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, mu)
    d_f = torch.empty(G.vol_shape, dtype=torch.float32, device="cuda")
    cb.tf_reconstruct_volume(G, dev(g), d_f, 2, n_outer, n_cgls, mu, True)
    assert rel(host(d_f), ref) <= 1e-4
    rrms = rel(host(d_f), f0.astype(np.float64))                # PAPER.md:270 RRMS (context, synthetic phantom)
    print("RRMS vs phantom after 3+3 outer iterations:", rrms)
    assert rrms < 0.5


def test_short_scan_cascade_with_detector_binning():
    """the scanner's 200-degree arc (20 views, endpoints included) on the config-2
    volume and detector, two levels, with and without detector binning at the coarse level (cbct_recon_create_ex),
    against the oracle's cascade; P and P^T of the arc geometry on their own first."""
    w, ells, f0, _ = syn.make_inputs(2, noisy=False)
    G = w.geometry.with_views(syn.short_scan(20, 200.0, -10.0))
    g = syn.analytic_projections(G, ells)
    h = cb.Geometry(G)
    d_p = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
    d_v = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
    h.forward(dev(f0), d_p)
    h.backproject(dev(g), d_v)
    assert rel(host(d_p), op.forward(G, f0.astype(np.float64))) <= 1e-5
    assert rel(host(d_v), op.back_scatter(G, g.astype(np.float64))) <= 1e-5
    assert h.status() == (True, [])
    mu, n_outer, n_cgls = 5e-4, [2, 2], 2
    for binned in (False, True):
        def make_ops(fac, binned=binned):
            Gl = G.coarsen_xy(fac) if fac > 1 else G
            return ops(Gl.bin_detector(fac) if (binned and fac > 1) else Gl)
        ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, mu, bin_detector=binned)
        rec = cb.Recon(G, 2, bin_detector=binned)
        d_f = torch.empty(G.vol_shape, dtype=torch.float32, device="cuda")
        rec.run(dev(g), d_f, n_outer, n_cgls, mu, True)
        assert rec.status() == (True, [])
        assert rel(host(d_f), ref) <= 1e-4, binned
        rec.close()


# ------------------------------------------------------------------------------------------ NEXT-3: TV / ROF comparison
@pytest.mark.parametrize("shape", [(16, 64, 64), (6, 37, 131), (1, 9, 33), (5, 1, 7), (1, 1, 1)])
def test_tv_rof_matches_oracle(shape):
    """the ROF gradient descent (device-resident step control) against the
    oracle's loop: same trials / accepted steps (both sides decide on fp64 energies), same volume, same energy."""
    from oracle import tv as otv
    rng = np.random.default_rng(sum(shape))
    u = (rng.random(shape) + 0.3 * rng.standard_normal(shape)).astype(np.float32)
    d_u = dev(u)
    d_f = torch.empty_like(d_u)
    for mu_tv, eps, max_iter, rel_tol in ((0.3, 0.05, 25, 1e-3), (0.05, 0.02, 8, 0.0), (0.0, 0.05, 5, 1e-3)):
        trace = []
        ref, it = otv.rof(u.astype(np.float64), mu_tv, eps, max_iter, rel_tol, trace=trace)
        _, trials, accepted, energy = cb.tv_rof(d_u, d_f, mu_tv, eps, max_iter, rel_tol)
        assert trials == it and accepted == sum(1 for t in trace if t[0]), (shape, mu_tv, trials, it)
        assert np.max(np.abs(host(d_f) - ref)) <= 2e-5 * max(np.max(np.abs(ref)), 1e-30), (shape, mu_tv)
        e_ref = otv.tv_energy(ref, u.astype(np.float64), mu_tv, eps)
        assert abs(energy - e_ref) <= 1e-5 * max(e_ref, 1e-30)
    cb.tv_rof(d_u, d_f, 0.3, 0.05, 25, 1e-3, clamp_nonneg=True)
    ref, _ = otv.rof(u.astype(np.float64), 0.3, 0.05, 25, 1e-3)
    assert np.max(np.abs(host(d_f) - np.maximum(ref, 0.0))) <= 2e-5 * np.max(np.abs(ref))


def test_tv_cascade_matches_oracle():
    """cbct_recon_run_tv (the paper's TV comparison algorithm on the multigrid cascade) against solver.multigrid_a2 with
    the ROF regulariser; config-1 geometry, two levels."""
    from oracle import tv as otv
    w, _, f0, g = syn.make_inputs(1)
    G = w.geometry

    def make_ops(fac):
        return ops(G.coarsen_xy(fac) if fac > 1 else G)

    mu_tv, eps, rof_iter, rel_tol, n_outer, n_cgls = 2e-3, 1e-3, 10, 1e-3, [2, 2], 2
    ref = osv.multigrid_a2(make_ops, G.vol_shape, g.astype(np.float64), 2, n_outer, n_cgls, 0.0,
                           regulariser=otv.tv_regulariser(mu_tv, eps, rof_iter, rel_tol))
    rec = cb.Recon(G, 2, tv=True)
    d_f = torch.empty(G.vol_shape, dtype=torch.float32, device="cuda")
    rec.run_tv(dev(g), d_f, n_outer, n_cgls, mu_tv, eps, rof_iter, rel_tol, True)
    assert rec.status() == (True, [])
    assert rel(host(d_f), ref) <= 1e-4
    rec.close()
