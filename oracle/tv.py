"""TEST INFRASTRUCTURE -- fp64 numpy oracle of the paper's COMPARISON regulariser: total
variation through the Rudin-Osher-Fatemi (ROF) sub-problem, PAPER.md:236-238 (§2.3).  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline leg may import this; it shares no code with paper_1008_2042_b200/.

PAPER.md:236: "f = argmin 1/2 ||Pf - g||^2 + mu_TV ||f||_TV, where ||f||_TV = int |grad f| dx ... a forward-backward
splitting algorithm akin to the Algorithm A1 is used ... the Step 2 becomes solving a sub-problem of
argmin_f ||f - f^(k+1)||^2 + mu_TV ||f||_TV, also known as a Rudin-Osher-Fatemi (ROF) model ... achieved by a simple
gradient descent method ... along the negative gradient direction in each step with an adaptively adjusted step length.
This process terminates when the energy function value decreases less than a certain amount, for instance, 0.1%, in two
successive steps."

The paper gives no discretisation; the readings (listed in DESIGN.md §1b) are:
  T1  grad f by FORWARD differences, zero across the last face (Neumann): (Df)_x[i] = f[i+1] - f[i], 0 at i = n-1;
      isotropic TV (PAPER.md:402 writes the square root of the three squared partials).
  T2  |grad f| is smoothed, sqrt(|Df|^2 + eps^2), eps an explicit parameter: TV is not differentiable at 0 and the paper
      descends along "the negative gradient".
  T3  E(f) = sum (f - u)^2 + mu_TV sum sqrt(|Df|^2 + eps^2)            (no 1/2 in front of the fidelity: as printed).
  T4  grad E = 2 (f - u) + mu_TV D^T( Df / sqrt(|Df|^2 + eps^2) ),  D^T the exact matrix transpose of D.
  T5  "adaptively adjusted step length": a trial step f - tau grad E is ACCEPTED iff it lowers E, then tau <- 1.2 tau;
      otherwise it is rejected and tau <- tau / 2 (the iterate and its gradient are kept).  tau starts at 0.25; descent
      starts from f = u.  Rejected trials count as iterations.
  T6  stop after the first accepted step whose relative decrease (E_k - E_{k+1}) / E_k is below rel_tol (0.1 %: "in two
      successive steps" read as "between two successive iterates"), or after max_iter trials, or at once if E(u) = 0.
"""
from __future__ import annotations

import numpy as np


def tv_forward_diff(f):
    """(Df)_a[i] = f[i + e_a] - f[i], zero at the last index of axis a (T1).  Returns (gz, gy, gx) for f[z][y][x]."""
    f = np.asarray(f, dtype=np.float64)
    out = []
    for ax in range(3):
        g = np.zeros_like(f)
        n = f.shape[ax]
        if n > 1:
            sl_lo = [slice(None)] * 3
            sl_hi = [slice(None)] * 3
            sl_lo[ax] = slice(0, n - 1)
            sl_hi[ax] = slice(1, n)
            g[tuple(sl_lo)] = f[tuple(sl_hi)] - f[tuple(sl_lo)]
        out.append(g)
    return out


def tv_forward_diff_transpose(p):
    """D^T p, the exact matrix transpose of tv_forward_diff: (D^T p)[i] = sum_a ( p_a[i - e_a] - p_a[i] ), with p_a taken
    as 0 at the last index (where D has no row) and the first term dropped at i = 0."""
    out = np.zeros_like(np.asarray(p[0], dtype=np.float64))
    for ax in range(3):
        pa = np.asarray(p[ax], dtype=np.float64)
        n = pa.shape[ax]
        if n > 1:
            sl_lo = [slice(None)] * 3
            sl_hi = [slice(None)] * 3
            sl_lo[ax] = slice(0, n - 1)
            sl_hi[ax] = slice(1, n)
            out[tuple(sl_lo)] -= pa[tuple(sl_lo)]
            out[tuple(sl_hi)] += pa[tuple(sl_lo)]
    return out


def tv_energy(f, u, mu_tv, eps):
    """E(f) of T3."""
    gz, gy, gx = tv_forward_diff(f)
    d = np.asarray(f, dtype=np.float64) - np.asarray(u, dtype=np.float64)
    return float(np.sum(d * d) + mu_tv * np.sum(np.sqrt(gx * gx + gy * gy + gz * gz + eps * eps)))


def tv_energy_gradient(f, u, mu_tv, eps):
    """grad E of T4."""
    gz, gy, gx = tv_forward_diff(f)
    inv = 1.0 / np.sqrt(gx * gx + gy * gy + gz * gz + eps * eps)
    return 2.0 * (np.asarray(f, dtype=np.float64) - np.asarray(u, dtype=np.float64)) + mu_tv * tv_forward_diff_transpose(
        (gz * inv, gy * inv, gx * inv))


def rof(u, mu_tv, eps, max_iter=30, rel_tol=1e-3, tau0=0.25, trace=None):
    """The ROF sub-problem by gradient descent with the adaptive step of T5 and the stopping rule of T6.
    Returns (f, trials used).  trace, if a list, receives (accepted, tau, E) per trial."""
    u = np.asarray(u, dtype=np.float64)
    f = u.copy()
    E = tv_energy(f, u, mu_tv, eps)
    tau, it = float(tau0), 0
    if E == 0.0:
        return f, 0
    while it < max_iter:
        it += 1
        ft = f - tau * tv_energy_gradient(f, u, mu_tv, eps)
        Et = tv_energy(ft, u, mu_tv, eps)
        if Et < E:
            rel = (E - Et) / E
            f, E = ft, Et
            if trace is not None:
                trace.append((True, tau, E))
            tau *= 1.2
            if rel < rel_tol:
                break
        else:
            if trace is not None:
                trace.append((False, tau, E))
            tau *= 0.5
    return f, it


def tv_regulariser(mu_tv, eps, max_iter=30, rel_tol=1e-3):
    """x -> ROF(x): plugs into solver.a2(..., regulariser=...) in the place of the tight-frame shrinkage (PAPER.md:236:
    "akin to the Algorithm A1 ... the Step 2 becomes ...")."""
    return lambda x: rof(x, mu_tv, eps, max_iter, rel_tol)[0]
