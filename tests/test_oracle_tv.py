"""Pins for the fp64 oracle of the paper's comparison regulariser, TV through the ROF sub-problem (oracle/tv.py;
PAPER.md:236-238).  Each pin is something the mathematics fixes, not a re-typing of the formula:
an explicit matrix for D and D^T, finite differences of the energy, a closed-form minimiser, an independent optimiser."""
import numpy as np
import pytest

from oracle import solver as osv
from oracle import tv


def test_forward_difference_and_its_transpose_as_explicit_matrices():
    """D built column by column on a 3x4x2 volume: rows at the last index of an axis are zero (Neumann, T1), D of a constant is
    zero, and tv_forward_diff_transpose is D^T entry for entry; D^T D has zero row sums (a Neumann Laplacian)."""
    shape = (3, 4, 2)
    n = int(np.prod(shape))
    D = np.zeros((3 * n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        D[:, j] = np.concatenate([g.ravel() for g in tv.tv_forward_diff(e.reshape(shape))])
    assert np.all(D @ np.ones(n) == 0.0)
    gz, gy, gx = tv.tv_forward_diff(np.arange(n, dtype=float).reshape(shape))
    assert np.all(gx[:, :, :-1] == 1.0) and np.all(gx[:, :, -1] == 0.0)
    assert np.all(gy[:, :-1, :] == 2.0) and np.all(gy[:, -1, :] == 0.0)
    assert np.all(gz[:-1] == 8.0) and np.all(gz[-1] == 0.0)
    rng = np.random.default_rng(1)
    p = rng.standard_normal((3,) + shape)
    assert np.max(np.abs(tv.tv_forward_diff_transpose(p).ravel() - D.T @ p.reshape(-1))) < 1e-14
    assert np.max(np.abs((D.T @ D).sum(axis=1))) < 1e-13


@pytest.mark.parametrize("shape", [(3, 4, 5), (1, 6, 7), (4, 1, 1)])
def test_gradient_is_the_derivative_of_the_energy(shape):
    """central finite differences of tv_energy in every coordinate against tv_energy_gradient (T3, T4): a dropped factor 2,
    a wrong sign in D^T or a missing eps would each be far outside 1e-6."""
    rng = np.random.default_rng(2)
    f, u = rng.standard_normal(shape), rng.standard_normal(shape)
    mu, eps, h = 0.7, 0.3, 1e-6
    g = tv.tv_energy_gradient(f, u, mu, eps)
    num = np.zeros(shape)
    for idx in np.ndindex(*shape):
        fp, fm = f.copy(), f.copy()
        fp[idx] += h
        fm[idx] -= h
        num[idx] = (tv.tv_energy(fp, u, mu, eps) - tv.tv_energy(fm, u, mu, eps)) / (2 * h)
    assert np.max(np.abs(num - g)) < 1e-6 * max(1.0, np.max(np.abs(g)))


def test_rof_special_cases_and_monotone_energy():
    rng = np.random.default_rng(3)
    u = rng.random((4, 5, 6))
    f, it = tv.rof(u, 0.0, 1e-3)
    assert it == 0 and np.array_equal(f, u)                                  # mu = 0: nothing to do (T6)
    c = np.full((3, 3, 3), 1.75)
    f, it = tv.rof(c, 0.5, 1e-3, max_iter=20)
    assert np.max(np.abs(f - c)) < 1e-15                                     # a constant is a fixed point (gradient 0)
    trace = []
    f, it = tv.rof(u, 0.4, 1e-2, max_iter=60, rel_tol=1e-6, trace=trace)
    e = [tv.tv_energy(u, u, 0.4, 1e-2)] + [t[2] for t in trace if t[0]]
    assert all(b < a for a, b in zip(e, e[1:])) and len(e) > 5               # accepted steps strictly lower E (T5)
    assert any(not t[0] for t in trace) or max(t[1] for t in trace) > 0.25   # the step length did adapt
    assert abs(f.mean() - u.mean()) < 1e-12                                  # D^T p sums to zero: the mean is preserved
    # the stopping rule: with rel_tol = 0.5 the first accepted step whose decrease is below 50 % ends the descent
    tr2 = []
    f2, it2 = tv.rof(u, 0.4, 1e-2, max_iter=60, rel_tol=0.5, trace=tr2)
    acc = [t for t in tr2 if t[0]]
    e2 = [tv.tv_energy(u, u, 0.4, 1e-2)] + [t[2] for t in acc]
    rel = [(a - b) / a for a, b in zip(e2, e2[1:])]
    assert rel[-1] < 0.5 and all(r >= 0.5 for r in rel[:-1]) and it2 == len(tr2)


def test_rof_step_edge_closed_form():
    """1-D two-level signal (plateaus of n1 and n2 samples, jump h): the minimiser of sum (f-u)^2 + mu |jump| moves the
    plateaus towards each other by mu / (2 n1) and mu / (2 n2) (set the derivative of n1 a^2 + n2 b^2 + mu (h - a - b) to
    zero).  With a small eps the descent must land there: pins mu, the missing 1/2 of T3 and the boundary rows."""
    n1, n2, h, mu = 6, 10, 2.0, 1.2
    u = np.concatenate([np.zeros(n1), np.full(n2, h)]).reshape(1, 1, -1)
    f, it = tv.rof(u, mu, 0.02, max_iter=20000, rel_tol=1e-15)
    a, b = mu / (2 * n1), mu / (2 * n2)
    # the smoothing rounds the plateaus next to the jump (a few eps) but does not move their means
    assert abs(f[0, 0, :n1].mean() - a) < 2e-3 and abs(f[0, 0, n1:].mean() - (h - b)) < 2e-3
    assert np.ptp(f[0, 0, :n1]) < 0.1 and np.ptp(f[0, 0, n1:]) < 0.1


def test_rof_reaches_the_minimiser_found_by_an_independent_optimiser():
    from scipy.optimize import minimize
    rng = np.random.default_rng(5)
    shape = (2, 3, 3)
    u = rng.random(shape)
    mu, eps = 0.3, 0.05
    res = minimize(lambda x: tv.tv_energy(x.reshape(shape), u, mu, eps), u.ravel(), method="BFGS", options=dict(gtol=1e-10))
    f, it = tv.rof(u, mu, eps, max_iter=5000, rel_tol=1e-15)
    assert np.max(np.abs(f.ravel() - res.x)) < 1e-5
    assert tv.tv_energy(f, u, mu, eps) <= res.fun * (1 + 1e-9)


def test_a2_with_the_tv_regulariser_reduces_to_a1_structure():
    """solver.a2(regulariser=...) replaces step 3 only ("akin to the Algorithm A1 ... the Step 2 becomes"):
    with the identity as regulariser it is plain CGLS + positivity; with ROF it equals the loop written out by hand."""
    rng = np.random.default_rng(6)
    A = rng.standard_normal((40, 18))
    shape = (2, 3, 3)
    P, PT = (lambda x: A @ x.ravel()), (lambda r: (A.T @ r).reshape(shape))
    g = A @ rng.random(18)
    reg = tv.tv_regulariser(0.05, 1e-3, max_iter=15)
    out = osv.a2(P, PT, g, np.zeros(shape), 3, 2, 0.0, momentum=False, regulariser=reg)
    f = np.zeros(shape)
    for _ in range(3):
        x, _h = osv.cgls(P, PT, f, g, 2)
        f = np.maximum(reg(x), 0.0)
    assert np.array_equal(out, f)
    ident = osv.a2(P, PT, g, np.zeros(shape), 1, 4, 0.0, momentum=False, regulariser=lambda x: x)
    assert np.array_equal(ident, np.maximum(osv.cgls(P, PT, np.zeros(shape), g, 4)[0], 0.0))
