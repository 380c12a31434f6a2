#!/usr/bin/env python
"""bench.py -- whole-hot-path benchmark of the B200 CBCT library (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 4]
    python bench.py --kernels-only      # P, P^T, fused TF, Siddon pair a few times (the command ncu wraps)
    python bench.py --peaks             # cbct_microbench: the per-SM rates that bound P / P^T on this device

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
N_SM, LANES_PER_CLK_PER_SM = 148, 128


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

    if args.peaks:
        # per-SM rates that bound P / P^T; rates per clock are converted with the max SM clock for context
        res = cb.microbench()
        clk = load_peaks()["sm_max_mhz"] * 1e6
        line = dict(peaks=True, n_sm=N_SM, sm_max_mhz=clk / 1e6)
        for name, (rate, unit) in res.items():
            line[name] = dict(value=rate, unit=unit)
        line["derived"] = dict(
            ffma_tinstr_s=res["ffma"][0] * 32 * N_SM * clk / 1e12, ffma2_tinstr_s=res["ffma2"][0] * 64 * N_SM * clk / 1e12,
            lds_wavefronts_per_clk_sm=res["lds32"][0], atoms_wavefronts_per_clk_sm=res["atoms_add_s32"][0])
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
        e = evs[-1]
        print(json.dumps(dict(kernels_only=True, workload=args.workload, p_ms=e[0].elapsed_time(e[1]),
                              pt_ms=e[1].elapsed_time(e[2]), tf_fused_ms=e[2].elapsed_time(e[3]),
                              siddon_p_ms=s[0].elapsed_time(s[1]), siddon_pt_ms=s[1].elapsed_time(s[2]),
                              samples=geom.n_samples)), flush=True)
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

    # ---- end-to-end arm (host buffers through the C ABI) -----------------------------------------
    for _ in range(2):
        step_host()
    barrier()
    ms_e2e = timed(step_host, args.steps)
    barrier()
    e2e_ms = replicas.max_over_ranks(float(np.sum(ms_e2e)), "cuda")
    e2e_value = world * samples_per_step * args.steps / (e2e_ms * 1e-3) / 1e9

    # ---- standalone kernels (context numbers) -----------------------------------------------------
    d_vol = torch.from_numpy(f0).cuda()
    d_proj = torch.empty(geom.proj_shape, dtype=torch.float32, device="cuda")
    for _ in range(3):
        geom.forward(d_vol, d_proj); geom.backproject(d_g, d_tmp)
    ms_p = float(np.median(timed(lambda: geom.forward(d_vol, d_proj), 5)))
    ms_pt = float(np.median(timed(lambda: geom.backproject(d_g, d_tmp), 5)))
    ms_tf = float(np.median(timed(lambda: cb.tf_apply_fused(d_vol, d_tmp, MU, True), 5)))
    # the paper's own pair (Siddon) and the scalar instruction stream of P: context numbers
    geom.siddon_forward(d_vol, d_proj); geom.siddon_backproject(d_g, d_tmp)
    ms_sp = float(np.median(timed(lambda: geom.siddon_forward(d_vol, d_proj), 3)))
    ms_spt = float(np.median(timed(lambda: geom.siddon_backproject(d_g, d_tmp), 3)))
    os.environ["CBCT_FW_PACKED"] = "0"
    geom.forward(d_vol, d_proj)
    ms_p_scalar = float(np.median(timed(lambda: geom.forward(d_vol, d_proj), 5)))
    del os.environ["CBCT_FW_PACKED"]

    # ---- the paper's full reconstruction, end to end (context number; 3 levels, 5/10/15) ----
    full_recon_s = None
    if rank == 0 and not args.no_full_recon:
        del d_alpha                                            # 2 GB of three-call coefficients no longer needed
        rec3 = cb.Recon(G, 3)
        rec3.run(d_g, d_f, [1, 1, 1], N_CGLS, MU, True)       # warm-up
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        rec3.run(d_g, d_f, [5, 10, 15], N_CGLS, MU, True)
        b.record()
        torch.cuda.synchronize()
        full_recon_s = a.elapsed_time(b) * 1e-3
        rrms = float(torch.linalg.vector_norm(d_f - d_vol) / torch.linalg.vector_norm(d_vol))
        rec3.close()

    if rank != 0:
        replicas.shutdown()
        return

    peaks = load_peaks()
    # dominant kernel = the projector with the larger share of the step
    (ms_f, n_f), (ms_b, n_b) = prof["forward"], prof["backproject"]
    dom = "backproject" if ms_b >= ms_f else "forward"
    dom_ms = (ms_b / max(n_b, 1)) if dom == "backproject" else (ms_f / max(n_f, 1))
    f_clk = peaks["sm_max_mhz"] * 1e6
    peak_tinstr = N_SM * LANES_PER_CLK_PER_SM * f_clk / 1e12
    achieved_tinstr = geom.n_samples * INSTR_PER_SAMPLE / (dom_ms * 1e-3) / 1e12
    # DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` captures (profiles/README.md),
    # cfg 4 only: P = forward_tma_kernel (r1_kernels_full.csv), P^T = scatter kernel, both view groups (r1_scatter_full.csv)
    ncu_traffic = {("forward", 4): 1.851507e9 + 35.917e6, ("backproject", 4): (439.53e6 + 84.42e6) + (2.635912e9 + 0.169432e9)}
    roofline = dict(bound="alu", kernel=f"cbct_{dom}", achieved=achieved_tinstr, peak=peak_tinstr, unit="Tinstr/s",
                    frac=achieved_tinstr / peak_tinstr, traffic=ncu_traffic.get((dom, args.workload)),
                    traffic_unit="DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum); algorithmic HBM bytes "
                                 "are 105e6 per launch, the kernel is not HBM bound; taken from the committed r1 captures (scalar streams, "
                                 "16x2 scatter layout) -- the packed default kernels move the same data and are to be re-captured",
                    algorithmic=f"{geom.n_samples} samples x {INSTR_PER_SAMPLE:.0f} thread-instr/sample per launch",
                    launch_ms=dom_ms, gsamples_s=geom.n_samples / (dom_ms * 1e-3) / 1e9,
                    peak_source=f"148 SM x 128 lanes/clk x {peaks['sm_max_mhz']:.0f} MHz ({peaks['source']} max SM clock)",
                    share_of_step=dict(forward=ms_f / step_ms, backproject=ms_b / step_ms))

    cpu_baseline = None
    if not args.no_cpu_baseline:
        r = time_oracle_sample(G, f0, g, [0, G.n_views // 3])
        cpu_baseline = dict(value=r["samples"] / r["seconds"] / 1e9, unit=UNIT, cores=omp_threads(), kind="oracle",
                            sample=f"oracle P + P^T (fp64, scatter form) on 2 of {G.n_views} views of the same workload: "
                                   f"{r['samples']:.3g} samples in {r['seconds']:.1f} s",
                            p_gsamples_s=0.5 * r["samples"] / r["t_forward"] / 1e9,
                            pt_gsamples_s=0.5 * r["samples"] / r["t_back"] / 1e9)

    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
        ms_per_step=step_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
        data="synthetic",
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
        extra=dict(p_ms=ms_p, pt_ms=ms_pt, tf_fused_ms=ms_tf, p_scalar_stream_ms=ms_p_scalar,
                   siddon_p_ms=ms_sp, siddon_pt_ms=ms_spt,
                   p_gsamples_s=geom.n_samples / ms_p / 1e6, pt_gsamples_s=geom.n_samples / ms_pt / 1e6,
                   s_per_cgls_iter=(ms_p + ms_pt) * 1e-3 + 0.0,
                   s_per_cgls_iter_in_step=(ms_f / max(n_f, 1) + ms_b / max(n_b, 1)) * 1e-3,
                   full_recon_s=full_recon_s,
                   full_recon="3-level multigrid, 5/10/15 A2 outer iterations, n_cgls=3, mu=5e-4, device-resident "
                              "(PAPER.md:288 recipe; paper: ~5 min on Tesla C1060)",
                   full_recon_rrms_vs_phantom=(rrms if full_recon_s is not None else None),
                   tf_fused_gbs=2 * geom.n_vox * 4 / ms_tf / 1e6, hbm_peak_gbs=peaks["hbm_gbs"],
                   wall_s_timed_region=t_wall,
                   paper_context="paper: ~2.7-3.5 s per P+P^T pair, ~5 min full recon on Tesla C1060 (PAPER.md:23, :402)"))
    print(json.dumps(line), flush=True)
    replicas.shutdown()


if __name__ == "__main__":
    main()
