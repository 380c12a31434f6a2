#!/usr/bin/env python
"""bench.py -- whole-hot-path benchmark of the B200 CBCT library (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 4]
    python bench.py --kernels-only      # P, P^T, fused TF, Siddon pair a few times (the command ncu wraps)
    python bench.py --peaks             # cbct_microbench alone: the per-SM rates that bound P / P^T on this device

A *step* is one pass of the whole hot path (every row) over one batch of synthetic
input at BASELINE.json's paper-size config (512x512x70 volume, 40 views of 512x384, step 0.25 mm):
  * one Algorithm-A2 outer iteration at the finest level through the driver (cbct_recon_run):
    extrapolation (a8), CGLS Initialize + 3 CGLS steps = 4 P (a1) + 4 P^T (a2) + the vector kernels
    (a3), the fused tight-frame shrinkage + positivity (a7);
  * the three-call tight frame on the result: tf_decompose, tf_shrink, tf_reconstruct (a4-a6);
  * mg_restrict + mg_prolong of the result (a9).
`value` = projector samples processed per second over the whole step (8 projector calls x the
algorithmic sample count of cbct_geometry_info), inputs resident in HBM.  `e2e` = the same step driven
through cbct_recon_run_host with HOST buffers (H2D of g, D2H of f inside the timed region).
Multi-GPU: the path does not shard (north_star: one GPU) -> N independent replicas, weak scaling.

Everything in the `roofline` object can be recomputed from the line itself: `launch_ms` is the mean CUDA-event time of the
dominant projector inside the timed steps (events recorded by the library on the launching stream), `samples_per_launch`
the algorithmic sample count, and the two ceilings of SURVEY.md §8(d) -- shared-memory wavefronts (8 per warp-sample) and
thread-instruction issue (40 per sample) -- are formed from rates that cbct_microbench measures IN THIS PROCESS (conflict-
free LDS / ATOMS wavefronts and FFMA issue per clock per SM) times the SM clock sampled during the timed region.
`traffic` is null: it may only come from an ncu capture of the kernels now timed, and none exists for this build.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "P+P^T projector throughput over one A2 outer iteration + TF + MG at 512x512x70x40 (Gsamples/s)"
UNIT = "Gsamples/s"
N_CGLS = 3
MU = 5e-4
# algorithmic thread-instructions per trilinear sample: 3 position FMAs, 3 floor,
# 3 frac, 3 address, 8 loads, 14 lerp ops, 1 accumulate, ~5 loop/convert = 40
INSTR_PER_SAMPLE = 40.0
ACCESSES_PER_SAMPLE = 8.0          # shared-memory loads (P) / integer reductions (P^T) per sample: 8 wavefronts per warp-sample
N_SM, SMSP_PER_SM = 148, 4


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        rows = [l.strip().split(",") for l in open(self.tmp.name) if l.strip()]
        os.unlink(self.tmp.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, val in zip(names, r[4:8]):
                if val.strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            hot = [s for s in sm if s > 0.5 * max(sm)]        # samples under load
            out.update(sm_mhz=float(np.median(hot)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def time_oracle_sample(G, f0, g, views):
    """The oracle as it stands on a bounded sample: P and P^T on `views` of the workload's views."""
    from oracle import projector as op
    sub = G.with_views([G.angles[i] for i in views])
    samples = op.sample_count(sub)
    f64 = f0.astype(np.float64)
    g64 = np.ascontiguousarray(g[list(views)].astype(np.float64))
    t0 = time.perf_counter()
    op.forward(sub, f64)
    t1 = time.perf_counter()
    op.back_scatter(sub, g64)
    t2 = time.perf_counter()
    return dict(samples=2.0 * samples, seconds=t2 - t0, t_forward=t1 - t0, t_back=t2 - t1)


def omp_threads():
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def run_reference(args, rank, world):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import build as ob
    ob.build()
    from paper_1008_2042_b200 import synthetic as syn
    w = syn.workload(args.workload)
    G = w.geometry
    f0 = syn.voxelise(G, syn.ellipsoids_for(w))
    g = syn.uniform_projections(G, w.seed)
    views = [0]                                               # one of the 40 views per step
    for _ in range(args.warmup):
        time_oracle_sample(G, f0, g, views)
    tot_s, tot_t = 0.0, 0.0
    for k in range(args.steps):
        r = time_oracle_sample(G, f0, g, [(k * 7) % G.n_views])
        tot_s += r["samples"]; tot_t += r["seconds"]
    val = tot_s / tot_t / 1e9
    sample = f"P + P^T (scatter form) on 1 of {G.n_views} views of workload {args.workload} per step, fp64, OpenMP"
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * tot_t / max(args.steps, 1), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=f"cfg{args.workload}:{w.name} {G.nx}x{G.ny}x{G.nz} vol, {G.n_views}x{G.nv}x{G.nu} proj",
                            step_mm=G.step, sample=sample),
                cpu_baseline=dict(value=val, unit=UNIT, cores=omp_threads(), kind="oracle", sample=sample),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=4)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernels-only", action="store_true", help="run P, P^T, fused TF 3x and exit (for ncu)")
    ap.add_argument("--peaks", action="store_true", help="run the library's micro-benchmarks (cbct_microbench) and exit")
    ap.add_argument("--no-full-recon", action="store_true", help="skip the one-off 3-level 5/10/15 reconstruction timing")
    ap.add_argument("--no-variants", action="store_true", help="skip the A/B timings of the other kernel variants")
    ap.add_argument("--full-recon-outer", default="5,10,15",
                    help="A2 outer iterations per level (coarse to fine) of the one-off full reconstruction; PAPER.md:288: 5,10,15")
    args = ap.parse_args()

    from paper_1008_2042_b200 import replicas
    rank, world, local_rank = replicas.world()
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    from paper_1008_2042_b200 import binding as cb
    from paper_1008_2042_b200 import synthetic as syn

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    replicas.init("nccl", torch.device("cuda", local_rank))

    def barrier():
        replicas.barrier("cuda")

    w = syn.workload(args.workload)
    G = w.geometry
    ells = syn.ellipsoids_for(w)
    f0 = syn.voxelise(G, ells)
    g = syn.analytic_projections(G, ells)
    if w.photons:
        g = syn.add_poisson_noise(g, w.photons, w.seed + rank)          # every replica its own noise draw

    def measure_peaks():
        """per-SM rates of cbct_microbench; per-clock rates need no clock assumption"""
        res = cb.microbench()
        return {name: dict(value=rate, unit=unit) for name, (rate, unit) in res.items()}

    if args.peaks:
        line = dict(peaks=True, n_sm=N_SM, **measure_peaks())
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "peaks_local.json"), "w") as fh:
            json.dump(line, fh, indent=1)
        print(json.dumps(line), flush=True)
        return

    if args.kernels_only:
        # short command for `ncu --set full`: 3 x (P, P^T, fused TF) on the workload, nothing else
        geom = cb.Geometry(G)
        d_vol = torch.from_numpy(f0).cuda()
        d_g = torch.from_numpy(g).cuda()
        d_proj = torch.empty(geom.proj_shape, dtype=torch.float32, device="cuda")
        d_out = torch.empty(geom.vol_shape, dtype=torch.float32, device="cuda")
        evs = []
        for _ in range(3):
            e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            e[0].record(); geom.forward(d_vol, d_proj)
            e[1].record(); geom.backproject(d_g, d_out)
            e[2].record(); cb.tf_apply_fused(d_vol, d_out, MU, True)
            e[3].record()
            evs.append(e)
        s = [torch.cuda.Event(enable_timing=True) for _ in range(3)]     # the paper's own pair (Siddon), warm then timed
        geom.siddon_forward(d_vol, d_proj); geom.siddon_backproject(d_g, d_out)
        s[0].record(); geom.siddon_forward(d_vol, d_proj)
        s[1].record(); geom.siddon_backproject(d_g, d_out)
        s[2].record()
        torch.cuda.synchronize()
        ok, bits = geom.status()
        e = evs[-1]
        print(json.dumps(dict(kernels_only=True, workload=args.workload, kernels=geom.describe(), device_status=bits,
                              p_ms=e[0].elapsed_time(e[1]),
                              pt_ms=e[1].elapsed_time(e[2]), tf_fused_ms=e[2].elapsed_time(e[3]),
                              siddon_p_ms=s[0].elapsed_time(s[1]), siddon_pt_ms=s[1].elapsed_time(s[2]),
                              samples=geom.n_samples)), flush=True)
        if not ok:
            raise SystemExit(3)
        return

    geom = cb.Geometry(G)                                                 # for the standalone P / P^T timing
    rec = cb.Recon(G, 1)
    n_proj_calls = 2 * (N_CGLS + 1)
    samples_per_step = n_proj_calls * geom.n_samples

    d_g = torch.from_numpy(g).cuda()
    d_f = torch.empty(geom.vol_shape, dtype=torch.float32, device="cuda")
    d_alpha = torch.empty((27,) + geom.vol_shape, dtype=torch.float32, device="cuda")
    d_tmp = torch.empty(geom.vol_shape, dtype=torch.float32, device="cuda")
    d_coarse = torch.empty((G.nz, G.ny // 2, G.nx // 2), dtype=torch.float32, device="cuda")
    h_g = torch.from_numpy(g).pin_memory()
    h_f = torch.empty(geom.vol_shape, dtype=torch.float32).pin_memory()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 256 MiB > 126 MB L2

    def tail():                                  # a4-a6 and a9 on the reconstructed volume
        cb.tf_decompose(d_f, d_alpha)
        cb.tf_shrink(d_alpha, MU)
        cb.tf_reconstruct(d_alpha, d_tmp)
        cb.mg_restrict(d_tmp, d_coarse)
        cb.mg_prolong(d_coarse, d_tmp)

    def step_device():
        rec.run(d_g, d_f, [1], N_CGLS, MU, True)
        tail()

    def step_host():
        rec.run_host(h_g, h_f, [1], N_CGLS, MU, True)   # H2D g, A2 iteration, D2H f, stream sync
        d_f.copy_(h_f, non_blocking=True)                 # the tail works on the volume the host now owns
        tail()

    def timed(fn, n):
        """n steps, each bracketed by its own CUDA events on the launching stream; L2 flushed between."""
        evs = []
        for _ in range(n):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    # ---- device-resident arm -------------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        step_device()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    launches0 = cb.launch_count()
    cb.profile_begin()
    t_wall0 = time.perf_counter()
    ms = timed(step_device, args.steps)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    prof = cb.profile_end()
    launches = cb.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    step_ms = replicas.max_over_ranks(float(np.sum(ms)), "cuda")
    value = world * samples_per_step * args.steps / (step_ms * 1e-3) / 1e9
    rec_ok, rec_bits = rec.status()

    # ---- end-to-end arm (host buffers through the C ABI) -----------------------------------------
    for _ in range(2):
        step_host()
    barrier()
    ms_e2e = timed(step_host, args.steps)
    barrier()
    e2e_ms = replicas.max_over_ranks(float(np.sum(ms_e2e)), "cuda")
    e2e_value = world * samples_per_step * args.steps / (e2e_ms * 1e-3) / 1e9

    if rank != 0:
        replicas.shutdown()
        return
    if world > 1:                                            # context numbers belong to the 1-GPU line; keep the scaling runs short
        args.no_variants = args.no_full_recon = True

    errors = []

    def guarded(what, fn, default=None):
        """context numbers must never cost the bench line: a failure is recorded, not raised"""
        try:
            return fn()
        except Exception as exc:  # noqa: BLE001
            errors.append(f"{what}: {type(exc).__name__}: {exc}")
            return default

    # ---- standalone kernels (the headline's components) -------------------------------------------------
    d_vol = torch.from_numpy(f0).cuda()
    d_proj = torch.empty(geom.proj_shape, dtype=torch.float32, device="cuda")

    def med(fn, n=5):
        fn()
        return float(np.median(timed(fn, n)))

    ms_p = med(lambda: geom.forward(d_vol, d_proj))
    ms_pt = med(lambda: geom.backproject(d_g, d_tmp))
    ms_tf = med(lambda: cb.tf_apply_fused(d_vol, d_tmp, MU, True))
    geom_ok, geom_bits = geom.status()

    # ---- roofline denominators, measured in this process -------------------------------------
    peaks = guarded("cbct_microbench", measure_peaks, {})
    hbm = load_peaks()
    f_clk_mhz = (clocks or {}).get("sm_mhz") or hbm["sm_max_mhz"]
    f_clk = f_clk_mhz * 1e6

    def rate(name, nominal):
        v = (peaks.get(name) or {}).get("value")
        return (float(v), "measured (cbct_microbench, this process)") if v else (nominal, "nominal (micro-benchmark unavailable)")

    (ms_f, n_f), (ms_b, n_b) = prof["forward"], prof["backproject"]
    per_call = dict(forward=ms_f / max(n_f, 1), backproject=ms_b / max(n_b, 1))
    dom = "backproject" if per_call["backproject"] >= per_call["forward"] else "forward"
    wave_name = "atoms_add_s32" if dom == "backproject" else "lds32"
    r_wave, src_wave = rate(wave_name, 1.0)               # conflict-free warp instructions (= wavefronts) per clock per SM
    r_issue, src_issue = rate("ffma", float(SMSP_PER_SM))  # warp instructions issued per clock per SM

    def ceilings(r_w, r_i):
        return dict(lsu_wavefront=N_SM * r_w * f_clk * 32.0 / ACCESSES_PER_SAMPLE / 1e9,
                    thread_instr=N_SM * r_i * f_clk * 32.0 / INSTR_PER_SAMPLE / 1e9)

    ceil = ceilings(r_wave, r_issue)
    binding = min(ceil, key=ceil.get)
    dom_ms = per_call[dom]
    achieved = geom.n_samples / (dom_ms * 1e-3) / 1e9
    roofline = dict(
        bound="alu", kernel=f"cbct_{dom}", kernels=geom.describe(), achieved=achieved, peak=ceil[binding], unit="Gsamples/s",
        frac=achieved / ceil[binding], binding=binding, traffic=None,
        traffic_note="null: no ncu capture of the kernels timed here exists (GPU use was closed to this repository while they "
                     "were written); algorithmic HBM bytes are 105e6 per launch = 16 us, the projectors are not HBM bound",
        launch_ms=dom_ms, samples_per_launch=geom.n_samples,
        ceilings_gsamples_s=ceil,
        frac_lsu_wavefront=achieved / ceil["lsu_wavefront"], frac_thread_instr=achieved / ceil["thread_instr"],
        formula="lsu_wavefront = 148 SM x wavefronts/clk/SM x f_clk x 32 lanes / 8 accesses per sample; "
                "thread_instr = 148 SM x warp-instr/clk/SM x f_clk x 32 lanes / 40 instructions per sample; peak = the lower",
        rates=dict(wavefronts_per_clk_per_sm=r_wave, wavefront_kind=wave_name, wavefront_source=src_wave,
                   warp_instr_per_clk_per_sm=r_issue, issue_source=src_issue, sm_clock_mhz=f_clk_mhz,
                   sm_clock_source="median nvidia-smi clocks.sm during the timed region" if (clocks or {}).get("sm_mhz") else "max SM clock"),
        other_projector=dict(kernel="cbct_forward" if dom == "backproject" else "cbct_backproject",
                             launch_ms=per_call["forward" if dom == "backproject" else "backproject"]),
        share_of_step=dict(forward=ms_f / step_ms, backproject=ms_b / step_ms))
    for k in ("forward", "backproject"):                  # both §8(d) fractions for both projectors
        a = geom.n_samples / (per_call[k] * 1e-3) / 1e9
        rw, _ = rate("atoms_add_s32" if k == "backproject" else "lds32", 1.0)
        c = ceilings(rw, r_issue)
        roofline[f"{k}_gsamples_s"] = a
        roofline[f"{k}_frac"] = dict(lsu_wavefront=a / c["lsu_wavefront"], thread_instr=a / c["thread_instr"], binding=min(c, key=c.get))

    # ---- A/B timings of the other kernel variants (context; each variant is a handle created under its selection variable) ----
    variants = {}
    if not args.no_variants:
        sel = ("CBCT_FORWARD_IMPL", "CBCT_BACKPROJECT_IMPL", "CBCT_FW_PACKED", "CBCT_BT_PACKED", "CBCT_BT_LANES")

        def variant(env, fn_name, src, dst):
            saved = {k: os.environ.pop(k, None) for k in sel}
            os.environ.update(env)
            try:
                h = cb.Geometry(G)
            finally:
                for k in sel:
                    os.environ.pop(k, None)
                    if saved[k] is not None:
                        os.environ[k] = saved[k]
            t = med(lambda: getattr(h, fn_name)(src, dst), 3)
            ok, bits = h.status()
            d = h.describe()
            h.close()
            return dict(ms=t, kernel=d.split("; ")[0 if fn_name == "forward" else 1], device_status=bits)

        for name, env in (("p_tma_scalar", {"CBCT_FORWARD_IMPL": "tma", "CBCT_FW_PACKED": "0"}),
                          ("p_tma_packed", {"CBCT_FORWARD_IMPL": "tma", "CBCT_FW_PACKED": "1"}),
                          ("p_tiled", {"CBCT_FORWARD_IMPL": "tiled"})):
            variants[name] = guarded(name, lambda env=env: variant(env, "forward", d_vol, d_proj))
        for name, env in (("pt_scatter_lm1_scalar", {"CBCT_BACKPROJECT_IMPL": "scatter", "CBCT_BT_LANES": "1", "CBCT_BT_PACKED": "0"}),
                          ("pt_scatter_lm1_packed", {"CBCT_BACKPROJECT_IMPL": "scatter", "CBCT_BT_LANES": "1", "CBCT_BT_PACKED": "1"}),
                          ("pt_scatter_lm0_scalar", {"CBCT_BACKPROJECT_IMPL": "scatter", "CBCT_BT_LANES": "0", "CBCT_BT_PACKED": "0"}),
                          ("pt_scatter_lm0_packed", {"CBCT_BACKPROJECT_IMPL": "scatter", "CBCT_BT_LANES": "0", "CBCT_BT_PACKED": "1"}),
                          ("pt_cell", {"CBCT_BACKPROJECT_IMPL": "cell"})):
            variants[name] = guarded(name, lambda env=env: variant(env, "backproject", d_g, d_tmp))
    # the paper's own pair (Siddon), Eq. 3 and the HBM-bound kernels: context numbers
    ctx = {}
    ctx["siddon_p_ms"] = guarded("siddon_forward", lambda: med(lambda: geom.siddon_forward(d_vol, d_proj), 3))
    ctx["siddon_pt_ms"] = guarded("siddon_backproject", lambda: med(lambda: geom.siddon_backproject(d_g, d_tmp), 3))
    ctx["eq3_ms"] = guarded("backproject_eq3", lambda: med(lambda: geom.backproject_eq3(d_g, d_tmp), 3))
    ctx["tf_fused_tile_ms"] = guarded("tf_apply_fused_tile", lambda: med(lambda: cb.tf_apply_fused(d_vol, d_tmp, MU, True, impl="tile"), 3))
    ctx["tf_fused_march_ms"] = guarded("tf_apply_fused_march", lambda: med(lambda: cb.tf_apply_fused(d_vol, d_tmp, MU, True, impl="march"), 3))
    ctx["tf_decompose_ms"] = guarded("tf_decompose", lambda: med(lambda: cb.tf_decompose(d_vol, d_alpha), 3))
    ctx["tf_shrink_ms"] = guarded("tf_shrink", lambda: med(lambda: cb.tf_shrink(d_alpha, MU), 3))
    ctx["tf_reconstruct_ms"] = guarded("tf_reconstruct", lambda: med(lambda: cb.tf_reconstruct(d_alpha, d_tmp), 3))
    ctx["tf_reconstruct_direct_ms"] = guarded("tf_reconstruct_direct", lambda: med(lambda: cb.tf_reconstruct_direct(d_alpha, d_tmp), 2))
    ctx["mg_prolong_ms"] = guarded("mg_prolong", lambda: med(lambda: cb.mg_prolong(d_coarse, d_tmp), 3))
    ctx["mg_restrict_ms"] = guarded("mg_restrict", lambda: med(lambda: cb.mg_restrict(d_tmp, d_coarse), 3))

    # ---- the paper's full reconstruction, end to end (context number; 3 levels, 5/10/15) ----
    full_recon_s, rrms = None, None
    n_outer_full = [int(v) for v in args.full_recon_outer.split(",")]
    if len(n_outer_full) != 3 or min(n_outer_full) < 0:
        raise SystemExit("--full-recon-outer takes three non-negative counts, coarse to fine")
    if not args.no_full_recon:
        def full():
            rec3 = cb.Recon(G, 3)
            rec3.run(d_g, d_f, [1, 1, 1], N_CGLS, MU, True)       # warm-up
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rec3.run(d_g, d_f, n_outer_full, N_CGLS, MU, True)
            b.record()
            torch.cuda.synchronize()
            ok3, bits3 = rec3.status()
            r = float(torch.linalg.vector_norm(d_f - d_vol) / torch.linalg.vector_norm(d_vol))
            rec3.close()
            if not ok3:
                errors.append(f"full reconstruction: device error word {bits3}")
            return a.elapsed_time(b) * 1e-3, r
        del d_alpha                                            # 2 GB of three-call coefficients no longer needed
        full_recon_s, rrms = guarded("full reconstruction", full, (None, None))

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:              # the oracle is timed beside the 1-GPU number only
        r = time_oracle_sample(G, f0, g, [G.n_views // 3])
        cpu_baseline = dict(value=r["samples"] / r["seconds"] / 1e9, unit=UNIT, cores=omp_threads(), kind="oracle",
                            sample=f"oracle P + P^T (fp64, scatter form) on 1 of {G.n_views} views of the same workload: "
                                   f"{r['samples']:.3g} samples in {r['seconds']:.1f} s",
                            p_gsamples_s=0.5 * r["samples"] / r["t_forward"] / 1e9,
                            pt_gsamples_s=0.5 * r["samples"] / r["t_back"] / 1e9)

    if not (rec_ok and geom_ok):
        errors.append(f"device error word raised: recon {rec_bits}, geometry {geom_bits} -- the numbers of this line are INVALID")
    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
        ms_per_step=step_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
        data="synthetic",
        # BASELINE.json's metric, spelled out: P and P^T throughput, roofline fraction, seconds per CGLS iteration
        s_per_cgls_iter=(per_call["forward"] + per_call["backproject"]) * 1e-3 + 0.0,
        p_gsamples_s=geom.n_samples / ms_p / 1e6, pt_gsamples_s=geom.n_samples / ms_pt / 1e6,
        kernels=geom.describe(),
        config=dict(workload=f"cfg{args.workload}:{w.name} {G.nx}x{G.ny}x{G.nz} vol ({G.dx}x{G.dy}x{G.dz} mm), "
                             f"{G.n_views}x{G.nv}x{G.nu} proj, SAD {G.sad:.0f}/SDD {G.sdd:.0f} mm",
                    step_mm=geom.step_mm, K=geom.K, samples_per_projector_call=geom.n_samples,
                    step="1 A2 outer iteration (CGLS init + 3 steps = 4 P + 4 P^T, fused TF+H) + tf_decompose/shrink/"
                         "reconstruct + mg_restrict/prolong", n_cgls=N_CGLS, mu=MU,
                    l2="256 MiB buffer written between timed steps (L2 flush); step working set ~3.5 GB >> 126 MB L2",
                    replicas=world, parallelism="replicas only (path does not shard)"),
        clocks=clocks, gpu_launches=int(launches),
        e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=int(h_g.numel() * 4 + h_f.numel() * 4),
                 d2h_bytes_per_step=int(h_f.numel() * 4), ms_per_step=e2e_ms / args.steps,
                 api="cbct_recon_run_host (HOST g in, HOST f out) + TF/MG tail on the returned volume"),
        roofline=roofline, cpu_baseline=cpu_baseline,
        extra=dict(p_ms=ms_p, pt_ms=ms_pt, tf_fused_ms=ms_tf,
                   s_per_cgls_iter_standalone=(ms_p + ms_pt) * 1e-3,
                   s_per_cgls_iter_note="top-level s_per_cgls_iter = mean P + mean P^T launch time inside the timed steps "
                                        "(vector kernels add < 2 %); standalone = the two kernels timed alone after an L2 flush",
                   variants=variants, context_ms=ctx, microbench=peaks,
                   full_recon_s=full_recon_s,
                   full_recon=f"3-level multigrid, {'/'.join(map(str, n_outer_full))} A2 outer iterations, n_cgls=3, mu=5e-4, device-resident "
                              "(PAPER.md:288 recipe; paper: ~5 min on Tesla C1060)",
                   full_recon_rrms_vs_phantom=rrms,
                   tf_fused_kernel=guarded("tf_apply_fused_describe", cb.tf_apply_fused_describe),
                   tf_fused_gbs=2 * geom.n_vox * 4 / ms_tf / 1e6, hbm_peak_gbs=hbm["hbm_gbs"], hbm_peak_source=hbm["source"],
                   wall_s_timed_region=t_wall, errors=errors,
                   paper_context="paper: ~2.7-3.5 s per P+P^T pair, ~5 min full recon on Tesla C1060 (PAPER.md:23, :402)"))
    print(json.dumps(line), flush=True)
    replicas.shutdown()


if __name__ == "__main__":
    main()
