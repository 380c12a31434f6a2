"""fp64 numpy oracle for CGLS, the tight frame, multigrid and Algorithm A2.  TEST INFRASTRUCTURE ONLY.

Every function follows the cited passage of /root/reference/PAPER.md step by step, in the
paper's order and notation; readings of silent/garbled points are those of SURVEY.md §8(c)
(item numbers quoted).  Nothing here is imported by the CUDA path.

Pins (tests/test_oracle_solver.py): W^T W = I, Parseval, explicit-matrix transpose of D,
shrinkage special cases, the collapse identity, CGLS vs dense least squares on a cond~24
system, residual monotonicity, A2 t-sequence closed form, multigrid affine reproduction.
"""
from __future__ import annotations

import math

import numpy as np

# PAPER.md:115 (§2.1): h0 = 1/4 [1,2,1], h1 = sqrt(2)/4 [1,0,-1], h2 = 1/4 [-1,2,-1]; h[a+1], a in {-1,0,1}
H = np.array([[0.25, 0.5, 0.25],
              [math.sqrt(2.0) / 4.0, 0.0, -math.sqrt(2.0) / 4.0],
              [-0.25, 0.5, -0.25]], dtype=np.float64)


# --------------------------------------------------------------------------------------
# tight frame: alpha = D f, T_mu, f = D^T alpha          (Eq. 2)
# --------------------------------------------------------------------------------------
def tf_decompose(f):
    """alpha_i = psi_i (x) f, psi_i = h_l(x) h_m(y) h_n(z), i = l + 3m + 9n (item 17),
    true convolution (item 16): alpha_i[x] = sum_{a,b,c} h_l[a]h_m[b]h_n[c] f[x-a,y-b,z-c],
    half-sample symmetric (edge-replicate) extension of f (item 15).  Returns [27][nz][ny][nx]."""
    f = np.asarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    fp = np.pad(f, 1, mode="edge")
    alpha = np.zeros((27, nz, ny, nx), dtype=np.float64)
    for n in range(3):
        for m in range(3):
            for l in range(3):
                i = l + 3 * m + 9 * n
                for c in (-1, 0, 1):
                    for b in (-1, 0, 1):
                        for a in (-1, 0, 1):
                            w = H[l, a + 1] * H[m, b + 1] * H[n, c + 1]
                            if w == 0.0:
                                continue
                            alpha[i] += w * fp[1 - c:1 - c + nz, 1 - b:1 - b + ny, 1 - a:1 - a + nx]
    return alpha


def tf_reconstruct(alpha):
    """f = D^T alpha: the exact matrix transpose of tf_decompose, boundary included (item 15).
    D = S E with E the edge-replicate padding and S the valid convolution, so D^T = E^T S^T:
    scatter every tap back into the padded array, then fold each padding layer onto the face
    it was replicated from."""
    alpha = np.asarray(alpha, dtype=np.float64)
    _, nz, ny, nx = alpha.shape
    acc = np.zeros((nz + 2, ny + 2, nx + 2), dtype=np.float64)
    for n in range(3):
        for m in range(3):
            for l in range(3):
                i = l + 3 * m + 9 * n
                for c in (-1, 0, 1):
                    for b in (-1, 0, 1):
                        for a in (-1, 0, 1):
                            w = H[l, a + 1] * H[m, b + 1] * H[n, c + 1]
                            if w == 0.0:
                                continue
                            acc[1 - c:1 - c + nz, 1 - b:1 - b + ny, 1 - a:1 - a + nx] += w * alpha[i]
    # E^T, one axis at a time (E is separable)
    acc[1, :, :] += acc[0, :, :]
    acc[-2, :, :] += acc[-1, :, :]
    acc = acc[1:-1]
    acc[:, 1, :] += acc[:, 0, :]
    acc[:, -2, :] += acc[:, -1, :]
    acc = acc[:, 1:-1]
    acc[:, :, 1] += acc[:, :, 0]
    acc[:, :, -2] += acc[:, :, -1]
    return np.ascontiguousarray(acc[:, :, 1:-1])


def tf_shrink(alpha, mu):
    """Vector shrinkage T_mu, Eq. 2: alpha_0 kept; alpha_i, i>=1, scaled by
    max(1 - mu/||alpha_h||, 0) with ||alpha_h|| the l2 norm over the 26 high bands.
    Factor := 0 where ||alpha_h|| = 0 (item 14)."""
    alpha = np.array(alpha, dtype=np.float64, copy=True)
    norm = np.sqrt(np.sum(alpha[1:] ** 2, axis=0))
    factor = np.zeros_like(norm)
    nzm = norm > 0.0
    factor[nzm] = np.maximum(1.0 - mu / norm[nzm], 0.0)
    alpha[1:] *= factor[None]
    return alpha


def positivity(f):
    """H f: voxel-wise truncation of negative values."""
    return np.maximum(f, 0.0)


def tf_apply(f, mu, clamp_nonneg=False):
    """f <- D^T T_mu D f, optionally followed by H (A2 step 4, item 26)."""
    out = tf_reconstruct(tf_shrink(tf_decompose(f), mu))
    return positivity(out) if clamp_nonneg else out


# --------------------------------------------------------------------------------------
# CGLS                                                   (Appendix 1)
# --------------------------------------------------------------------------------------
def cgls_init(P, PT, x0, y):
    """Initialize: r = y - P x0; p = s = P^T r; gamma = ||s||^2."""
    x = np.array(x0, dtype=np.float64, copy=True)
    r = np.asarray(y, dtype=np.float64) - P(x)
    s = PT(r)
    p = s.copy()
    gamma = float(np.sum(s * s))
    return dict(x=x, r=r, p=p, gamma=gamma, breakdown=False, qq=0.0, alpha=0.0, beta=0.0)


def cgls_step(P, PT, st):
    """One pass through steps 1-7.  Breakdown (gamma == 0 or ||q||^2 == 0)
    leaves the state untouched and raises the flag (item 13)."""
    if st["gamma"] == 0.0:
        st["breakdown"] = True
        return st
    q = P(st["p"])                                   # 1. q = P p
    qq = float(np.sum(q * q))
    if qq == 0.0:
        st["breakdown"] = True
        return st
    alpha = st["gamma"] / qq                         # 2. alpha = gamma / ||q||^2
    st["x"] = st["x"] + alpha * st["p"]              # 3. x += alpha p
    st["r"] = st["r"] - alpha * q                    #    r -= alpha q
    s = PT(st["r"])                                  # 4. s = P^T r
    gamma_new = float(np.sum(s * s))                 # 5. gamma' = ||s||^2
    beta = gamma_new / st["gamma"]                   # 6. beta = gamma'/gamma
    st["p"] = s + beta * st["p"]                     # 7. p = s + beta p
    st.update(gamma=gamma_new, qq=qq, alpha=alpha, beta=beta)
    return st


def cgls(P, PT, x0, y, n_steps):
    """x = CGLS[x0] with n_steps passes through steps 1-7 (item 12).  Returns (x, history of ||r||^2)."""
    st = cgls_init(P, PT, x0, y)
    hist = [float(np.sum(st["r"] ** 2))]
    for _ in range(n_steps):
        st = cgls_step(P, PT, st)
        if st["breakdown"]:
            break
        hist.append(float(np.sum(st["r"] ** 2)))
    return st["x"], hist


# --------------------------------------------------------------------------------------
# multigrid transfer operators                           (§2.2.3; items 20, 22)
# --------------------------------------------------------------------------------------
def _axis_of(name):
    return {"z": 0, "y": 1, "x": 2}[name]


def mg_restrict(fine, fx=2, fy=2, fz=1):
    """Mean of the fx*fy*fz children (item 22)."""
    out = np.asarray(fine, dtype=np.float64)
    for name, fac in (("x", fx), ("y", fy), ("z", fz)):
        assert fac in (1, 2)
        if fac == 2:
            ax = _axis_of(name)
            assert out.shape[ax] % 2 == 0
            ev = np.take(out, np.arange(0, out.shape[ax], 2), axis=ax)
            od = np.take(out, np.arange(1, out.shape[ax], 2), axis=ax)
            out = 0.5 * (ev + od)
    return np.ascontiguousarray(out)


def mg_prolong(coarse, fx=2, fy=2, fz=1):
    """Cell-centred linear interpolation ("smoothly extend ... linear interpolation"):
    fine cell 2j sits at coarse coordinate j - 1/4, fine cell 2j+1 at j + 1/4, so the weights are
    3/4 (own parent) and 1/4 (nearer neighbour); the neighbour is clamped at the faces (item 22)."""
    out = np.asarray(coarse, dtype=np.float64)
    for name, fac in (("x", fx), ("y", fy), ("z", fz)):
        assert fac in (1, 2)
        if fac == 2:
            ax = _axis_of(name)
            n = out.shape[ax]
            idx = np.arange(n)
            left = np.take(out, np.maximum(idx - 1, 0), axis=ax)
            right = np.take(out, np.minimum(idx + 1, n - 1), axis=ax)
            even = 0.75 * out + 0.25 * left
            odd = 0.75 * out + 0.25 * right
            shape = list(out.shape)
            shape[ax] = 2 * n
            fine = np.empty(shape, dtype=np.float64)
            sl_e = [slice(None)] * 3
            sl_o = [slice(None)] * 3
            sl_e[ax] = slice(0, None, 2)
            sl_o[ax] = slice(1, None, 2)
            fine[tuple(sl_e)] = even
            fine[tuple(sl_o)] = odd
            out = fine
    return np.ascontiguousarray(out)


# --------------------------------------------------------------------------------------
# Algorithm A2 and the multigrid cascade
# --------------------------------------------------------------------------------------
def a2_t_next(t):
    """Step 5: t^(k+1) = (1 + sqrt(1 + 4 t^(k)^2)) / 2."""
    return 0.5 * (1.0 + math.sqrt(1.0 + 4.0 * t * t))


def a2(P, PT, g, f_init, n_outer, n_cgls, mu, momentum=True, trace=None, regulariser=None):
    """Algorithm A2; momentum=False gives Algorithm A1.
    Step 1 is garbled in PAPER.md:165; reading of item 11:
        v = f^k + ((t^(k-1) - 1)/t^k) (f^k - f^(k-1)),  t^(-1) = t^(0) = 1, f^(-1) = f^(0) = f_init.
    CGLS restarts from x0 = v every outer iteration (item 23).
    regulariser: a callable x -> x' that replaces the tight-frame shrinkage of step 3 (the TV comparison
    algorithm is "akin to the Algorithm A1", with the ROF sub-problem in that place; oracle/tv.py); mu is then unused."""
    f_prev = np.array(f_init, dtype=np.float64, copy=True)
    f_cur = f_prev.copy()
    t_prev, t_cur = 1.0, 1.0
    for k in range(n_outer):
        coef = (t_prev - 1.0) / t_cur if momentum else 0.0
        v = f_cur + coef * (f_cur - f_prev)                    # 1. extrapolate
        x, hist = cgls(P, PT, v, g, n_cgls)                     # 2. f = CGLS[v]
        x = tf_apply(x, mu, clamp_nonneg=False) if regulariser is None else regulariser(x)   # 3. shrinkage (or ROF)
        x = positivity(x)                                       # 4. correct
        if trace is not None:
            trace.append(dict(k=k, coef=coef, t=t_cur, rr=hist))
        f_prev, f_cur = f_cur, x
        t_prev, t_cur = t_cur, a2_t_next(t_cur)                 # 5. t update
    return f_cur


def bin_projections(g, factor):
    """Detector binning: every factor x factor block of pixels of each view is replaced by
    its mean, i.e. the line integral averaged over the block; `factor` a power of two.  g[view][v][u]."""
    out = np.asarray(g, dtype=np.float64)
    while factor > 1:
        assert factor % 2 == 0
        out = mg_restrict(out, 2, 2, 1)          # the "volume" axes (z, y, x) are (view, v, u) here: views are kept
        factor //= 2
    return out


def multigrid_a2(make_ops, finest_shape, g, n_levels, n_outer, n_cgls, mu, momentum=True, bin_detector=False, regulariser=None):
    """Coarse-to-fine cascade Omega_{2^(L-1) h} -> ... -> Omega_h: x,y coarsened by 2 per
    level, z kept (item 20); g at full resolution on every level (item 21) unless bin_detector (NEXT-4: the level
    coarsened by `fac` then works on g binned by `fac`, and make_ops must return the operators of the binned
    detector); the prolonged solution is the initial guess and t, f^(k-1) are reset on each level (item 23).
    make_ops(level_factor) -> (P, PT) for the grid coarsened by `level_factor` in x and y."""
    nz, ny, nx = finest_shape
    fac = 2 ** (n_levels - 1)
    f = np.zeros((nz, ny // fac, nx // fac), dtype=np.float64)
    for lev in range(n_levels):
        P, PT = make_ops(fac)
        g_lev = bin_projections(g, fac) if bin_detector else g
        f = a2(P, PT, g_lev, f, n_outer[lev], n_cgls, mu, momentum, regulariser=regulariser)
        if lev + 1 < n_levels:
            f = mg_prolong(f, 2, 2, 1)
            fac //= 2
    return f
