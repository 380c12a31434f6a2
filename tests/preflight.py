"""Device pre-flight: every kernel variant of libcbct_b200 once, at sizes that finish in seconds, through the C ABI,
each checked against the fp64 oracle and against the handle's device error word.

    compute-sanitizer --tool memcheck --error-exitcode 7 python tests/preflight.py        # first, on any kernel change
    python tests/preflight.py                                                              # plain

This is the GPU half of the gate in DESIGN.md §5c (the CPU half is `pytest -m "not gpu"`, which runs the same kernel
sources under tests/cpu_shim): nothing larger than this runs on a device before this has passed under memcheck.
It stops at the FIRST failure (a later kernel must not run on a context that may already be poisoned).
"""
from __future__ import annotations

import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TOL = 1e-5


def main() -> int:
    import torch

    from oracle import projector as op
    from oracle import solver as osv
    from paper_1008_2042_b200 import binding as cb
    from paper_1008_2042_b200 import synthetic as syn

    assert torch.cuda.is_available(), "preflight needs cuda:0"
    torch.cuda.set_device(0)

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()

    def rel(a, ref):
        return float(np.linalg.norm(np.asarray(a, np.float64).ravel() - ref.ravel()) / max(np.linalg.norm(ref.ravel()), 1e-300))

    def say(what, err, tol=TOL):
        ok = err <= tol
        print(f"{'ok  ' if ok else 'FAIL'} {what}: {err:.2e}", flush=True)
        if not ok:
            raise SystemExit(1)

    def clean(h, what):
        ok, bits = h.status()
        if not ok:
            print(f"FAIL {what}: device error word {bits}", flush=True)
            raise SystemExit(1)

    TINY = syn.workload(1).geometry
    RAGGED = syn.Geometry(44, 36, 12, 2.0, 2.5, 4.0, 53, 27, 2.1, 2.9, 1000.0, 1500.0,
                          (0.0, 0.3, math.pi / 4, 1.2, math.pi / 2, 2.2, 3 * math.pi / 4, math.pi, 3.9, 5.0, 5.9),
                          ox=-3.0, oy=5.0, oz=1.5, u0=-2.2, v0=3.3, step_mm=0.9)
    ODD = syn.Geometry(37, 29, 11, 2.0, 3.0, 5.0, 45, 19, 2.3, 3.1, 1000.0, 1500.0,
                       (0.0, 0.4, math.pi / 4, math.pi / 2, 2.0, math.pi, 4.0, 5.5), ox=3.0, oy=-4.0, oz=2.0, u0=1.7, v0=-2.9,
                       step_mm=0.7)
    refs = {}

    def oracle(kind, G, a):
        key = (kind, id(G), a.tobytes()[:64], a.shape)
        if key not in refs:
            fn = {"P": op.forward, "PT": op.back_scatter, "EQ3": op.back_eq3, "SF": op.siddon_forward, "SB": op.siddon_back}[kind]
            refs[key] = fn(G, a.astype(np.float64))
        return refs[key]

    def with_env(env):
        for k in ("CBCT_FORWARD_IMPL", "CBCT_BACKPROJECT_IMPL", "CBCT_FW_PACKED", "CBCT_BT_PACKED", "CBCT_BT_LANES"):
            os.environ.pop(k, None)
        os.environ.update(env)

    with_env({})
    h0 = cb.Geometry(TINY)                                   # first create: runs the library's self-check of the fast variants
    print("default kernels:", h0.describe(), flush=True)
    fast_ok = "rejected" not in h0.describe()
    h0.close()
    if not fast_ok:
        print("NOTE fast variants rejected by the create-time self-check: they are skipped below", flush=True)
    # ---- P: every forward kernel -----------------------------------------------------------------------------------
    fw_variants = [({"CBCT_FORWARD_IMPL": "global"}, (TINY, ODD)), ({"CBCT_FORWARD_IMPL": "tiled"}, (TINY, ODD)),
                   ({"CBCT_FORWARD_IMPL": "tma", "CBCT_FW_PACKED": "0"}, (TINY, RAGGED)),
                   ({"CBCT_FORWARD_IMPL": "tma", "CBCT_FW_PACKED": "1"}, (TINY, RAGGED))]
    for env, geoms in fw_variants:
        if env.get("CBCT_FW_PACKED") == "1" and not fast_ok:
            continue
        with_env(env)
        for G in geoms:
            x = syn.uniform_volume(G, 5)
            h = cb.Geometry(G)
            out = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
            h.forward(dev(x), out)
            torch.cuda.synchronize()
            clean(h, "forward")
            say(f"P   {h.describe().split(';')[0]} {G.nx}x{G.ny}x{G.nz}", rel(out.cpu().numpy(), oracle("P", G, x)))
            h.close()
    # ---- P^T: every backprojection kernel ---------------------------------------------------------------------------
    bp_variants = [({"CBCT_BACKPROJECT_IMPL": "gather"}, (TINY, ODD)), ({"CBCT_BACKPROJECT_IMPL": "cell"}, (TINY, ODD))]
    for lanes in ("1", "0"):
        for packed in ("0", "1"):
            bp_variants.append(({"CBCT_BACKPROJECT_IMPL": "scatter", "CBCT_BT_LANES": lanes, "CBCT_BT_PACKED": packed}, (TINY, RAGGED)))
    for env, geoms in bp_variants:
        if (env.get("CBCT_BT_PACKED") == "1" or env.get("CBCT_BT_LANES") == "0") and not fast_ok:
            continue
        with_env(env)
        for G in geoms:
            y = syn.uniform_projections(G, 6) - 0.4
            h = cb.Geometry(G)
            out = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
            h.backproject(dev(y), out)
            torch.cuda.synchronize()
            clean(h, "backproject")
            say(f"P^T {h.describe().split('; ')[1]} {G.nx}x{G.ny}x{G.nz}", rel(out.cpu().numpy(), oracle("PT", G, y)))
            h.close()
    with_env({})
    # ---- the paper's own pair: Eq. 3, Siddon ------------------------------------------------------------------------------
    for G in (TINY, ODD):
        x, y = syn.uniform_volume(G, 7), syn.uniform_projections(G, 7) - 0.3
        h = cb.Geometry(G)
        vol = torch.empty(h.vol_shape, dtype=torch.float32, device="cuda")
        proj = torch.empty(h.proj_shape, dtype=torch.float32, device="cuda")
        h.backproject_eq3(dev(y), vol)
        torch.cuda.synchronize()
        say(f"Eq.3 backprojector {G.nx}x{G.ny}x{G.nz}", rel(vol.cpu().numpy(), oracle("EQ3", G, y)))
        h.siddon_forward(dev(x), proj)
        h.siddon_backproject(dev(y), vol)
        torch.cuda.synchronize()
        say(f"Siddon P   {G.nx}x{G.ny}x{G.nz}", rel(proj.cpu().numpy(), oracle("SF", G, x)))
        say(f"Siddon P^T {G.nx}x{G.ny}x{G.nz}", rel(vol.cpu().numpy(), oracle("SB", G, y)))
        clean(h, "siddon / eq3")
        h.close()
    # ---- tight frame, multigrid, A2 extrapolation ------------------------------------------------------------------------
    rng = np.random.default_rng(3)
    for shape in ((16, 64, 64), (5, 7, 9), (1, 33, 40), (6, 37, 131), (40, 30, 29)):
        f = rng.standard_normal(shape).astype(np.float32)
        d_f = dev(f)
        d_a = torch.empty((27,) + shape, dtype=torch.float32, device="cuda")
        d_o = torch.empty(shape, dtype=torch.float32, device="cuda")
        cb.tf_decompose(d_f, d_a)
        torch.cuda.synchronize()
        a_ref = osv.tf_decompose(f.astype(np.float64))
        say(f"tf_decompose {shape}", float(np.max(np.abs(d_a.cpu().numpy() - a_ref)) / np.max(np.abs(a_ref))))
        cb.tf_shrink(d_a, 0.4)
        torch.cuda.synchronize()
        a_s = d_a.cpu().numpy().astype(np.float64)
        say(f"tf_shrink {shape}", float(np.max(np.abs(a_s - osv.tf_shrink(a_ref, 0.4))) / np.max(np.abs(a_ref))), 2e-5)
        r_ref = osv.tf_reconstruct(a_s)
        for name, fn in (("tf_reconstruct (march)", cb.tf_reconstruct), ("tf_reconstruct_direct", cb.tf_reconstruct_direct)):
            fn(d_a, d_o)
            torch.cuda.synchronize()
            say(f"{name} {shape}", float(np.max(np.abs(d_o.cpu().numpy() - r_ref)) / np.max(np.abs(r_ref))))
        ref = osv.tf_apply(f.astype(np.float64), 0.3, clamp_nonneg=True)
        for impl in ("tile", "march", None):                  # each kernel on its own, then the library's choice
            cb.tf_apply_fused(d_f, d_o, 0.3, True, impl=impl)
            torch.cuda.synchronize()
            say(f"tf_apply_fused[{impl or cb.tf_apply_fused_describe()}] {shape}", float(np.max(np.abs(d_o.cpu().numpy() - ref)) / np.max(np.abs(f))), 2e-5)
    from oracle import tv as otv
    for shape in ((6, 20, 24), (1, 9, 33)):
        u = (rng.random(shape) + 0.3 * rng.standard_normal(shape)).astype(np.float32)
        d_u = dev(u)
        d_o = torch.empty_like(d_u)
        _, trials, accepted, energy = cb.tv_rof(d_u, d_o, 0.3, 0.05, 25, 1e-3)
        ref, it = otv.rof(u.astype(np.float64), 0.3, 0.05, 25, 1e-3)
        say(f"tv_rof {shape} ({trials} trials, oracle {it})", float(np.max(np.abs(d_o.cpu().numpy() - ref)) / np.max(np.abs(ref))) + (0.0 if trials == it else 1.0), 2e-5)
    # scalar kernels (ragged rows) and the float4 kernels (rows of whole float4s), every factor pattern the driver uses
    for shape, (fx, fy, fz) in (((6, 8, 10), (2, 2, 1)), ((4, 6, 16), (2, 2, 2)), ((6, 4, 24), (1, 2, 1)), ((5, 34, 136), (2, 2, 1))):
        fine = rng.random(shape).astype(np.float32)
        d_c = torch.empty((shape[0] // fz, shape[1] // fy, shape[2] // fx), dtype=torch.float32, device="cuda")
        d_fine = torch.empty(shape, dtype=torch.float32, device="cuda")
        cb.mg_restrict(dev(fine), d_c, fx, fy, fz)
        cb.mg_prolong(d_c, d_fine, fx, fy, fz)
        torch.cuda.synchronize()
        say(f"mg_restrict {shape} /{fx}{fy}{fz}", float(np.max(np.abs(d_c.cpu().numpy() - osv.mg_restrict(fine.astype(np.float64), fx, fy, fz)))), 1e-6)
        say(f"mg_prolong  {shape} x{fx}{fy}{fz}",
            float(np.max(np.abs(d_fine.cpu().numpy() - osv.mg_prolong(d_c.cpu().numpy().astype(np.float64), fx, fy, fz)))), 1e-6)
    # ---- CGLS + the A2 driver (default kernels) ---------------------------------------------------------------------------
    w, _e, f0, g = syn.make_inputs(1)
    G = w.geometry
    P, PT = (lambda v: op.forward(G, v)), (lambda r: op.back_scatter(G, r))
    rec = cb.Recon(G, 1)
    d_out = torch.empty(G.vol_shape, dtype=torch.float32, device="cuda")
    rec.run(dev(g), d_out, [1], 2, 5e-4, True)
    torch.cuda.synchronize()
    say("A2 outer iteration (CGLS init + 2 steps, fused TF, clamp)",
        rel(d_out.cpu().numpy(), osv.a2(P, PT, g.astype(np.float64), np.zeros(G.vol_shape), 1, 2, 5e-4, True)), 1e-4)
    rec.close()
    # ---- micro-benchmarks with short loops (bounds only; rates are meaningless at this length) ----------------------------
    r = cb.microbench(iters=4)
    print("ok   cbct_microbench (iters=4):", {k: round(v[0], 3) for k, v in r.items()}, flush=True)
    print(f"preflight ok: {cb.launch_count()} kernel launches", flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
