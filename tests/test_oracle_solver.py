"""Pins for the fp64 numpy oracle of the tight frame, CGLS, A2 and multigrid (oracle/solver.py).

PAPER.md:115 (filters, f = D^T alpha), PAPER.md:123-129 (Eq. 2), PAPER.md:430-470 (CGLS, residual
never grows), PAPER.md:159-169 (A2), PAPER.md:232 (multigrid); SURVEY.md §8(c) pin table.
"""
import math

import numpy as np
import pytest

from oracle import projector as op
from oracle import solver as osv
from paper_1008_2042_b200 import synthetic as syn


# ---------------------------------------------------------------- tight frame
def test_filters_are_the_papers_and_form_a_tight_frame():
    """PAPER.md:115 values; sum_l h_l[a] h_l[b] = delta_ab * (1/4, 1/2, 1/4)[a] (unitary extension)."""
    s = math.sqrt(2.0) / 4.0
    assert np.allclose(osv.H, [[0.25, 0.5, 0.25], [s, 0.0, -s], [-0.25, 0.5, -0.25]], rtol=0, atol=1e-16)
    assert np.allclose(osv.H.T @ osv.H, np.diag([0.25, 0.5, 0.25]), rtol=0, atol=1e-16)


@pytest.mark.parametrize("shape", [(5, 6, 7), (1, 4, 9), (3, 1, 2), (2, 2, 2)])
def test_perfect_reconstruction_and_parseval(shape):
    """W^T W = I (north_star check 4) and sum_i ||alpha_i||^2 = ||f||^2, boundaries included."""
    rng = np.random.default_rng(7)
    f = rng.standard_normal(shape)
    a = osv.tf_decompose(f)
    assert a.shape == (27,) + shape
    assert np.max(np.abs(osv.tf_reconstruct(a) - f)) < 1e-14
    assert abs(np.sum(a * a) - np.sum(f * f)) < 1e-12 * np.sum(f * f)


def test_reconstruct_is_the_matrix_transpose_of_decompose():
    """Explicit matrices on a 3x4x5 volume: <D e_j, e_i> == <e_j, D^T e_i> for every pair."""
    shape = (3, 4, 5)
    n = int(np.prod(shape))
    Dm = np.zeros((27 * n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        Dm[:, j] = osv.tf_decompose(e.reshape(shape)).ravel()
    DTm = np.zeros((n, 27 * n))
    for i in range(27 * n):
        e = np.zeros(27 * n)
        e[i] = 1.0
        DTm[:, i] = osv.tf_reconstruct(e.reshape((27,) + shape)).ravel()
    assert np.max(np.abs(DTm - Dm.T)) < 1e-15
    assert np.max(np.abs(Dm.T @ Dm - np.eye(n))) < 1e-14


def test_band_order_and_convolution_sign():
    """i = l + 3m + 9n with l along x: band 1 of an x-ramp is sqrt(2)/4 * (f[x+1]-f[x-1]) = sqrt(2)/2,
    band 3 (m=1) sees only y, band 9 (n=1) only z; band 0 of a constant is the constant."""
    z, y, x = np.meshgrid(np.arange(6.0), np.arange(7.0), np.arange(8.0), indexing="ij")
    for ramp, band in ((x, 1), (y, 3), (z, 9)):
        a = osv.tf_decompose(ramp)
        inner = a[:, 1:-1, 1:-1, 1:-1]
        assert np.allclose(inner[band], math.sqrt(2.0) / 2.0, atol=1e-14)
        others = [b for b in (1, 3, 9) if b != band]
        assert np.max(np.abs(inner[others])) < 1e-14
        assert np.allclose(inner[0], ramp[1:-1, 1:-1, 1:-1], atol=1e-13)   # low-pass keeps affine data
    a = osv.tf_decompose(np.full((4, 4, 4), 3.5))
    assert np.allclose(a[0], 3.5, atol=1e-14) and np.max(np.abs(a[1:])) < 1e-14


def test_shrinkage_eq2_special_cases():
    rng = np.random.default_rng(8)
    f = rng.standard_normal((5, 6, 7))
    a = osv.tf_decompose(f)
    assert np.array_equal(osv.tf_shrink(a, 0.0), a)                               # mu = 0: identity
    big = osv.tf_shrink(a, 1e9)
    assert np.array_equal(big[0], a[0]) and np.all(big[1:] == 0.0)                # mu -> inf: alpha_0 only
    norm = np.sqrt(np.sum(a[1:] ** 2, axis=0))
    mu = float(np.median(norm))
    sh = osv.tf_shrink(a, mu)
    assert np.all(sh[1:, norm < mu] == 0.0)
    keep = norm > mu
    assert np.allclose(np.sqrt(np.sum(sh[1:] ** 2, axis=0))[keep], norm[keep] - mu, rtol=1e-12)
    assert np.array_equal(sh[0], a[0])
    zero = osv.tf_shrink(np.zeros((27, 2, 2, 2)), 0.1)                            # ||alpha_h|| = 0: no NaN
    assert np.all(zero == 0.0)


def _lowpass(f):
    return osv.tf_decompose(f)[0]


def _lowpass_T(a0):
    a = np.zeros((27,) + a0.shape)
    a[0] = a0
    return osv.tf_reconstruct(a)


@pytest.mark.parametrize("mu", [0.05, 0.5, 5.0])
def test_collapse_identity_is_a_second_route(mu):
    """||alpha_h||^2 = W0 f^2 - (W0 f)^2 and D^T T_mu D f = f * W0^T s + W0^T((1-s) * W0 f)
    (SURVEY.md §8(c) TF pin 4): an independent route to the fused result, boundaries included."""
    rng = np.random.default_rng(9)
    f = rng.standard_normal((6, 7, 8))
    a = osv.tf_decompose(f)
    nh2 = np.sum(a[1:] ** 2, axis=0)
    var = _lowpass(f * f) - _lowpass(f) ** 2
    assert np.max(np.abs(nh2 - var)) < 1e-13
    nh = np.sqrt(np.maximum(var, 0.0))
    s = np.where(nh > 0, np.maximum(1.0 - mu / np.where(nh > 0, nh, 1.0), 0.0), 0.0)
    route2 = f * _lowpass_T(s) + _lowpass_T((1.0 - s) * _lowpass(f))
    assert np.max(np.abs(osv.tf_apply(f, mu) - route2)) < 1e-13


def _filt(g, axis, l):
    """h_l along one axis with edge-replicate extension, written out tap by tap (alpha[x] = sum_a h_l[a] g[x - a])"""
    n = g.shape[axis]
    pad = [(0, 0)] * g.ndim
    pad[axis] = (1, 1)
    e = np.pad(g, pad, mode="edge")
    sl = lambda k: tuple(slice(k, k + n) if ax == axis else slice(None) for ax in range(g.ndim))
    return osv.H[l][0] * e[sl(2)] + osv.H[l][1] * e[sl(1)] + osv.H[l][2] * e[sl(0)]        # taps a = -1, 0, +1


def test_high_band_energy_from_separable_difference_terms():
    """The route tf_fused_march_kernel takes: per axis sum_l (h_l * g)^2 = h0 * g^2, hence
        ||alpha_h||^2 = Wz[ Wy[X_1^2 + X_2^2] + Y_01^2 + Y_02^2 ] + alpha_001^2 + alpha_002^2
    with X_l = h_l *x f, Y_0m = h_m *y X_0, alpha_00n = h_n *z Y_00 -- a sum of non-negative terms made of difference
    filters.  Checked against the 26 high bands of the oracle's plain decomposition, faces and 1-thick axes included."""
    rng = np.random.default_rng(11)
    for shape in ((6, 7, 8), (1, 5, 9), (4, 1, 3), (2, 2, 1)):
        f = rng.standard_normal(shape) + 50.0                       # a large offset: the terms below never see it
        a = osv.tf_decompose(f)
        X = [_filt(f, 2, l) for l in range(3)]                      # axes: volumes are f[z][y][x], l runs on x
        assert np.max(np.abs(sum(x * x for x in X) - _filt(f * f, 2, 0))) < 1e-9
        Y0 = [_filt(X[0], 1, m) for m in range(3)]
        A00 = [_filt(Y0[0], 0, n) for n in range(3)]
        t = _filt(X[1] ** 2 + X[2] ** 2, 1, 0) + Y0[1] ** 2 + Y0[2] ** 2
        energy = _filt(t, 0, 0) + A00[1] ** 2 + A00[2] ** 2
        assert np.max(np.abs(A00[0] - a[0])) < 1e-12 and np.max(np.abs(A00[2] - a[18])) < 1e-12      # band i = l + 3m + 9n
        ref = np.sum(a[1:] ** 2, axis=0)
        assert np.max(np.abs(energy - ref)) <= 1e-12 * max(np.max(ref), 1.0), shape
        assert np.all(energy >= 0.0)


def test_tf_apply_limits():
    rng = np.random.default_rng(10)
    f = rng.standard_normal((4, 5, 6))
    assert np.max(np.abs(osv.tf_apply(f, 0.0) - f)) < 1e-14                       # mu = 0
    c = np.full((4, 5, 6), -2.25)
    assert np.max(np.abs(osv.tf_apply(c, 0.3) - c)) < 1e-14                       # constants pass
    assert np.all(osv.tf_apply(c, 0.3, clamp_nonneg=True) == 0.0)                 # H
    lp = _lowpass_T(_lowpass(f))
    assert np.max(np.abs(osv.tf_apply(f, 1e9) - lp)) < 1e-14                      # mu -> inf


# ---------------------------------------------------------------- CGLS
def _tiny_system():
    """8x8x4 volume of 4 mm voxels, 24x12 detector at 2.2 mm, 24 views: 6912 rays x 256 unknowns,
    full rank, cond ~ 24 (SURVEY.md §8(c) CGLS pin 2)."""
    G = syn.Geometry(8, 8, 4, 4.0, 4.0, 4.0, 24, 12, 2.2, 2.2, 1000.0, 1500.0, syn.full_circle(24))
    n = G.nx * G.ny * G.nz
    A = np.zeros((G.n_views * G.nv * G.nu, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        A[:, j] = op.forward(G, e.reshape(G.vol_shape)).ravel()
    return G, A


def test_cgls_reaches_dense_least_squares_and_residual_never_grows():
    G, A = _tiny_system()
    assert np.linalg.cond(A) < 100
    rng = np.random.default_rng(12)
    y = rng.random(G.proj_shape)
    P = lambda x: op.forward(G, x)
    PT = lambda r: op.back_scatter(G, r)
    x0 = rng.random(G.vol_shape)
    x, hist = osv.cgls(P, PT, x0, y, 256)
    ref = np.linalg.lstsq(A, y.ravel(), rcond=None)[0].reshape(G.vol_shape)
    assert np.max(np.abs(x - ref)) < 1e-12 * np.max(np.abs(ref))
    assert all(b <= a * (1 + 1e-12) for a, b in zip(hist, hist[1:]))
    # one step from a given state equals the textbook formulas evaluated with the dense matrix
    st = osv.cgls_init(P, PT, x0, y)
    r0 = y.ravel() - A @ x0.ravel()
    s0 = A.T @ r0
    assert np.allclose(st["p"].ravel(), s0, rtol=1e-12) and abs(st["gamma"] - s0 @ s0) < 1e-10 * (s0 @ s0)
    st = osv.cgls_step(P, PT, st)
    q = A @ s0
    al = (s0 @ s0) / (q @ q)
    assert np.allclose(st["x"].ravel(), x0.ravel() + al * s0, rtol=1e-12)
    s1 = A.T @ (r0 - al * q)
    assert abs(s1 @ s0) < 1e-10 * (s0 @ s0)                                        # s_{k+1} _|_ s_k
    assert np.allclose(st["p"].ravel(), s1 + (s1 @ s1) / (s0 @ s0) * s0, rtol=1e-10, atol=1e-12)


def test_cgls_breakdown_is_flagged_not_nan():
    G, _ = _tiny_system()
    P = lambda x: op.forward(G, x)
    PT = lambda r: op.back_scatter(G, r)
    y = np.zeros(G.proj_shape)
    st = osv.cgls_init(P, PT, np.zeros(G.vol_shape), y)
    st = osv.cgls_step(P, PT, st)
    assert st["breakdown"] and np.all(st["x"] == 0.0)


# ---------------------------------------------------------------- A2
def test_a2_t_sequence_closed_form():
    """t0=1, t1=(1+sqrt5)/2=1.6180, t2=2.1935; coefficient (t^(k-1)-1)/t^k = 0, 0, 0.2817 (item 11)."""
    t0 = 1.0
    t1 = osv.a2_t_next(t0)
    t2 = osv.a2_t_next(t1)
    assert abs(t1 - (1 + math.sqrt(5)) / 2) < 1e-15
    assert abs(t2 - 2.193527085331054) < 1e-12
    assert abs((t1 - 1) / t2 - 0.2817) < 1e-4


def test_a2_momentum_coefficients_and_a1_reduction():
    G = syn.Geometry(8, 8, 4, 4.0, 4.0, 4.0, 12, 6, 4.4, 4.4, 1000.0, 1500.0, syn.full_circle(6))
    P = lambda x: op.forward(G, x)
    PT = lambda r: op.back_scatter(G, r)
    f0 = syn.voxelise(G, [syn.Ellipsoid(1.0, -2.0, 0.5, 9.0, 7.0, 5.0, 0.05)], dtype=np.float64)
    g = P(f0)
    tr = []
    f_a2 = osv.a2(P, PT, g, np.zeros(G.vol_shape), 4, 2, 1e-4, momentum=True, trace=tr)
    phi = (1 + math.sqrt(5)) / 2
    t2 = 0.5 * (1 + math.sqrt(1 + 4 * phi * phi))
    t3 = 0.5 * (1 + math.sqrt(1 + 4 * t2 * t2))
    assert np.allclose([t["coef"] for t in tr], [0.0, 0.0, (phi - 1) / t2, (t2 - 1) / t3], rtol=1e-14, atol=0)
    for t in tr:                                   # CGLS output never worse than its input
        assert t["rr"][-1] <= t["rr"][0] * (1 + 1e-12)
    # momentum off: A1 written out by hand
    f = np.zeros(G.vol_shape)
    for _ in range(3):
        f, _h = osv.cgls(P, PT, f, g, 2)
        f = np.maximum(osv.tf_reconstruct(osv.tf_shrink(osv.tf_decompose(f), 1e-4)), 0.0)
    assert np.array_equal(osv.a2(P, PT, g, np.zeros(G.vol_shape), 3, 2, 1e-4, momentum=False), f)
    assert f_a2.min() >= 0.0


# ---------------------------------------------------------------- multigrid
def test_prolong_reproduces_affine_and_restrict_preserves_mean():
    z, y, x = np.meshgrid(np.arange(5.0), np.arange(6.0), np.arange(7.0), indexing="ij")
    coarse = 2.0 + 0.5 * x - 0.25 * y + 0.125 * z
    fine = osv.mg_prolong(coarse, 2, 2, 1)
    assert fine.shape == (5, 12, 14)
    zf, yf, xf = np.meshgrid(np.arange(5.0), np.arange(12.0), np.arange(14.0), indexing="ij")
    expect = 2.0 + 0.5 * (xf / 2 - 0.25) - 0.25 * (yf / 2 - 0.25) + 0.125 * zf    # fine cell i at coarse i/2 - 1/4
    assert np.max(np.abs(fine[:, 1:-1, 1:-1] - expect[:, 1:-1, 1:-1])) < 1e-14
    back = osv.mg_restrict(fine, 2, 2, 1)
    assert np.max(np.abs(back[:, 1:-1, 1:-1] - coarse[:, 1:-1, 1:-1])) < 1e-14    # restrict o prolong = id
    rng = np.random.default_rng(13)
    r = rng.random((4, 6, 8))
    assert abs(osv.mg_restrict(r, 2, 2, 2).mean() - r.mean()) < 1e-15
    assert np.all(osv.mg_restrict(np.full((4, 6, 8), 1.75), 2, 2, 1) == 1.75)
    assert np.all(osv.mg_prolong(np.full((4, 3, 4), 1.75), 2, 2, 2) == 1.75)
    # hand values at a face: weights 3/4, 1/4 with the neighbour clamped
    p = osv.mg_prolong(np.array([[[1.0, 5.0]]]), 2, 1, 1)
    assert np.allclose(p, [[[1.0, 2.0, 4.0, 5.0]]])


def test_multigrid_cascade_runs_and_reduces_error():
    G = syn.Geometry(16, 16, 4, 4.0, 4.0, 4.0, 24, 8, 4.2, 4.2, 1000.0, 1500.0, syn.full_circle(12))
    f0 = syn.voxelise(G, [syn.Ellipsoid(3.0, -5.0, 0.0, 20.0, 14.0, 6.0, 0.04),
                          syn.Ellipsoid(-9.0, 8.0, 1.0, 8.0, 9.0, 4.0, 0.03)], dtype=np.float64)
    g = op.forward(G, f0)

    def make_ops(fac):
        Gl = G.coarsen_xy(fac) if fac > 1 else G
        # the sampling step stays that of the finest grid only if asked; here each level uses its default
        return (lambda x: op.forward(Gl, x)), (lambda r: op.back_scatter(Gl, r))

    f = osv.multigrid_a2(make_ops, G.vol_shape, g, 2, [3, 3], 2, 1e-5)
    assert f.shape == G.vol_shape
    rrms = np.linalg.norm(f - f0) / np.linalg.norm(f0)          # PAPER.md:270 RRMS definition
    assert rrms < 0.35, rrms


# ---------------------------------------------------------------- short scan, detector binning
def test_bin_projections_is_the_block_mean_and_matches_the_binned_detector_geometry():
    """bin_projections: hand values; mean preserved; views kept.  And the geometric pin: the mean of the 2x2 (4x4) pixel
    centres' line integrals of a smooth object equals the line integral at the block centre -- the pixel of the binned
    detector geometry -- up to second order in the pixel pitch (analytic ellipsoid chords on both detectors), and the
    error falls 4x when the pitch is halved; a wrong centre / pitch in Geometry.bin_detector would be first order."""
    g = np.arange(2 * 4 * 6, dtype=np.float64).reshape(2, 4, 6)
    b = osv.bin_projections(g, 2)
    assert b.shape == (2, 2, 3)
    assert b[0, 0, 0] == np.mean([0, 1, 6, 7]) and b[1, 1, 2] == np.mean([40, 41, 46, 47])
    assert abs(b.mean() - g.mean()) < 1e-13
    assert np.array_equal(osv.bin_projections(g, 1), g)
    e = [syn.Ellipsoid(4.0, -6.0, 2.0, 40.0, 28.0, 22.0, 0.03)]
    errs = []
    for pitch in (2.0, 1.0):
        n = int(round(192 / pitch))
        G = syn.Geometry(8, 8, 8, 1.0, 1.0, 1.0, n, n // 2, pitch, pitch, 1000.0, 1500.0, (0.3, 2.0, 4.4), u0=3.0, v0=-2.0)
        fine = syn.analytic_projections(G, e, np.float64)
        for fac in (2, 4):
            coarse = syn.analytic_projections(G.bin_detector(fac), e, np.float64)
            inner = coarse > 0.5 * coarse.max()                       # away from the silhouette, where chords are smooth
            errs.append(np.max(np.abs(osv.bin_projections(fine, fac)[inner] - coarse[inner])) / coarse.max())
    assert errs[0] < 6e-3 and errs[1] < 3e-2, errs
    assert errs[0] / errs[2] > 3.5 and errs[1] / errs[3] > 3.5, errs     # second order in the pitch ...
    assert 4.0 < errs[1] / errs[0] < 6.0 and 4.0 < errs[3] / errs[2] < 6.0, errs   # ... and (f^2 - 1) in the factor: 15 / 3


def test_short_scan_angles_and_cascade_with_detector_binning():
    """200-degree arc, endpoints included; the oracle's cascade with detector binning at the coarse
    level: the coarse level works on block-mean data with the binned detector's operators and still delivers a useful
    initial guess (the error after the cascade is within 10 % of the cascade on unbinned data)."""
    ang = syn.short_scan(21, 200.0, -10.0)
    assert len(ang) == 21 and abs(math.degrees(ang[0]) + 10.0) < 1e-12 and abs(math.degrees(ang[-1]) - 190.0) < 1e-12
    assert np.allclose(np.diff(ang), math.radians(10.0))
    G = syn.Geometry(16, 16, 4, 4.0, 4.0, 4.0, 24, 8, 4.2, 4.2, 1000.0, 1500.0, ang)
    f0 = syn.voxelise(G, [syn.Ellipsoid(3.0, -5.0, 0.0, 20.0, 14.0, 6.0, 0.04),
                          syn.Ellipsoid(-9.0, 8.0, 1.0, 8.0, 9.0, 4.0, 0.03)], dtype=np.float64)
    g = op.forward(G, f0)

    def make_ops(binned):
        def ops(fac):
            Gl = G.coarsen_xy(fac) if fac > 1 else G
            if binned and fac > 1:
                Gl = Gl.bin_detector(fac)
            return (lambda x: op.forward(Gl, x)), (lambda r: op.back_scatter(Gl, r))
        return ops

    rr = {}
    for binned in (False, True):
        f = osv.multigrid_a2(make_ops(binned), G.vol_shape, g, 2, [3, 3], 2, 1e-5, bin_detector=binned)
        rr[binned] = np.linalg.norm(f - f0) / np.linalg.norm(f0)
    assert rr[False] < 0.45 and rr[True] < 1.1 * rr[False], rr
    # the binned coarse level alone: its CGLS objective is that of the binned problem (residual never grows)
    P, PT = make_ops(True)(2)
    _x, hist = osv.cgls(P, PT, np.zeros(G.coarsen_xy(2).vol_shape), osv.bin_projections(g, 2), 4)
    assert all(b <= a * (1 + 1e-12) for a, b in zip(hist, hist[1:]))
